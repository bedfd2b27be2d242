// sweep.cuh -- the PPM stencil of S2 as a register window that slides
// along a pencil, one new zone value per step.  A thread that marches along direction d feeds
// q[p] for p = -3, -2, ..., L+2 (L = zones of the pencil inside the tile); the window then holds
// exactly what CW84 (1.6)-(1.10) needs, so every slope, edge value and parabola of the pencil is
// computed ONCE and nothing is exchanged between threads.
//
// Feeding order and what exists afterwards (all indices relative to the pencil):
//   start(q[-3]); warm1(q[-2]); warm2(q[-1]) -> limited slope of zone -2
//   warm3(q[0])                              -> slope of zone -1, edge between zones -2 and -1
//   push(q[p]), p >= 1                       -> slope of zone p-1, edge between zones p-2 and p-1,
//                                               monotonised parabola of zone p-2: qm (minus edge),
//                                               qp (plus edge); qpL = plus edge of zone p-3
//   p >= 2 : the face between zones p-3 and p-2 has both states: left = qpL, right = qm.
#pragma once
#include "hydro.cuh"

struct PpmWindow {
    double q1, q2;     // q[p-1], q[p-2]
    double dq1;        // q[p-1] - q[p-2]
    double s2;         // twice the limited slope of zone p-2
    double e;          // edge value between zones p-3 and p-2
    double qpL;        // plus edge of the parabola of zone p-3   (left state of the next face)
    double qm, qp;     // parabola edges of zone p-2 after the last push

    __device__ __forceinline__ void start(double qn) { q1 = qn; qp = qn; }
    __device__ __forceinline__ void warm1(double qn) { dq1 = qn - q1; q2 = q1; q1 = qn; }
    __device__ __forceinline__ void warm2(double qn)
    {
        const double dqn = qn - q1;
        s2 = slope2(dq1, dqn);
        q2 = q1; q1 = qn; dq1 = dqn;
    }
    __device__ __forceinline__ void warm3(double qn)
    {
        const double dqn = qn - q1;
        const double s1 = slope2(dq1, dqn);
        e = edge_value(q2, dq1, s2, s1);
        q2 = q1; q1 = qn; dq1 = dqn; s2 = s1;
    }
    __device__ __forceinline__ void push(double qn)
    {
        qpL = qp;
        const double dqn = qn - q1;
        const double s1 = slope2(dq1, dqn);             // zone p-1
        const double en = edge_value(q2, dq1, s2, s1);  // between zones p-2 and p-1
        double a = e, b = en;
        monotonize(q2, a, b);                           // zone p-2
        qm = a; qp = b;
        q2 = q1; q1 = qn; dq1 = dqn; s2 = s1; e = en;
    }
    // push with CW84 shock flattening (flatten.cu, reading F4): the parabola of zone p-2 that this step completes is
    // blended with the zone average, q+- <- chi q+- + (1 - chi) q, chi = the coefficient of zone p-2 (chi = 1: unchanged)
    __device__ __forceinline__ void push_flat(double qn, double chi)
    {
        qpL = qp;
        const double dqn = qn - q1;
        const double s1 = slope2(dq1, dqn);
        const double en = edge_value(q2, dq1, s2, s1);
        double a = e, b = en;
        monotonize(q2, a, b);
        const double rest = (1.0 - chi) * q2;
        qm = fma(chi, a, rest); qp = fma(chi, b, rest);
        q2 = q1; q1 = qn; dq1 = dqn; s2 = s1; e = en;
    }
};
