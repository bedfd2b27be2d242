// advect.cu -- S1-S4 (+ fused S5): <A(U)> on every interior zone (include/cst.h cst_advance_A,
// cst_advance_A_update).  FIRST CORRECT VERSION: one thread per zone, each thread rebuilds the
// 7-zone stencil of every direction from global memory (this is the paper's own GPU strategy,
// PAPER.md L52, "each CUDA thread handles the update of a single zone").  It exists to establish
// parity; the tiled kernel that replaces it is described in DESIGN.md section 6.
#include "hydro.cuh"

// parabolas of the three zones at stencil positions 2,3,4 of q[0..6]  (zone i-1, i, i+1)
__device__ __forceinline__ void ppm3(const double q[7], double qm[3], double qp[3])
{
    double dq[6], s[5], e[4];
#pragma unroll
    for (int n = 0; n < 6; ++n) dq[n] = q[n + 1] - q[n];
#pragma unroll
    for (int n = 0; n < 5; ++n) s[n] = slope2(dq[n], dq[n + 1]);          // zone n+1
#pragma unroll
    for (int n = 0; n < 4; ++n) e[n] = edge_value(q[n + 1], dq[n + 1], s[n], s[n + 1]); // face n+3/2
#pragma unroll
    for (int n = 0; n < 3; ++n) {
        double a = e[n], b = e[n + 1];
        monotonize(q[n + 2], a, b);
        qm[n] = a; qp[n] = b;
    }
}

struct UpdArgs {
    bool fused;
    double* U_next;
    double dt_m;
    const double* A_old;     // nullptr = "the value just computed"
    int nquad;
    const double* Aq[CST_MAX_QUAD];   // nullptr = "the value just computed"
    double w[CST_MAX_QUAD];
};

template <int D>
__device__ __forceinline__ void direction_pass(const Geom& g, const double* __restrict__ Ub,
                                               long long zc, long long stride, double rdx,
                                               double A5[5], double Fm[2], bool left[2], double r7[7])
{
    double W7[5][7];
#pragma unroll
    for (int n = 0; n < 7; ++n) {
        const long long z = zc + (long long)(n - 3) * stride;
        double W[5];
        r7[n] = cons_to_prim(g, Ub[z], Ub[g.comp_g + z], Ub[2 * g.comp_g + z], Ub[3 * g.comp_g + z],
                             Ub[4 * g.comp_g + z], W);
#pragma unroll
        for (int c = 0; c < 5; ++c) W7[c][n] = W[c];
    }
    double qm[5][3], qp[5][3];
#pragma unroll
    for (int c = 0; c < 5; ++c) ppm3(W7[c], qm[c], qp[c]);
    double F[2][5];
#pragma unroll
    for (int f = 0; f < 2; ++f) {            // f = 0: low face (zones i-1 | i), f = 1: high face
        double WL[5], WR[5];
#pragma unroll
        for (int c = 0; c < 5; ++c) { WL[c] = qp[c][f]; WR[c] = qm[c][f + 1]; }
        WL[0] = fmax(WL[0], g.small_dens); WR[0] = fmax(WR[0], g.small_dens);
        WL[4] = fmax(WL[4], g.small_pres); WR[4] = fmax(WR[4], g.small_pres);
        left[f] = hllc<D>(g, WL, WR, F[f]);
        Fm[f] = F[f][0];
    }
#pragma unroll
    for (int c = 0; c < 5; ++c) A5[c] = fma(-(F[1][c] - F[0][c]), rdx, A5[c]);
}

__device__ __forceinline__ double species_pass(const double* __restrict__ Us, long long zc,
                                               long long stride, const double r7[7],
                                               const double Fm[2], const bool left[2])
{
    double q[7], qm[3], qp[3];
#pragma unroll
    for (int n = 0; n < 7; ++n) q[n] = Us[zc + (long long)(n - 3) * stride] * r7[n];
    ppm3(q, qm, qp);
    const double flo = Fm[0] * (left[0] ? qp[0] : qm[1]);
    const double fhi = Fm[1] * (left[1] ? qp[1] : qm[2]);
    return fhi - flo;
}

__global__ void __launch_bounds__(128)
k_advance_naive(Geom g, const double* __restrict__ U, double* __restrict__ A, UpdArgs up)
{
    const int ng = CST_NG;
    const long long nzb = g.comp_a;
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nzb * g.nbox) return;
    const int b = (int)(t / nzb);
    const long long zl = t - (long long)b * nzb;
    const int k = (int)(zl / ((long long)g.nx * g.ny));
    const int rem = (int)(zl - (long long)k * g.nx * g.ny);
    const int j = rem / g.nx, i = rem - j * g.nx;
    const double* Ub = U + (long long)b * g.box_g;
    const long long zc = ((long long)(k + ng) * g.ey + (j + ng)) * g.ex + (i + ng);
    const long long za = (long long)b * g.box_a + zl;

    double A5[5] = { 0, 0, 0, 0, 0 };
    double Fm[3][2], r7[3][7];
    bool left[3][2];
    direction_pass<0>(g, Ub, zc, 1, g.rdx, A5, Fm[0], left[0], r7[0]);
    direction_pass<1>(g, Ub, zc, g.ex, g.rdy, A5, Fm[1], left[1], r7[1]);
    direction_pass<2>(g, Ub, zc, g.plane_g, g.rdz, A5, Fm[2], left[2], r7[2]);
    // S4 source: constant gravity, from the zone-centre state
    const double rho = Ub[zc], mx = Ub[g.comp_g + zc], my = Ub[2 * g.comp_g + zc], mz = Ub[3 * g.comp_g + zc];
    A5[1] = fma(rho, g.grav[0], A5[1]);
    A5[2] = fma(rho, g.grav[1], A5[2]);
    A5[3] = fma(rho, g.grav[2], A5[3]);
    A5[4] += fma(mz, g.grav[2], fma(my, g.grav[1], mx * g.grav[0]));

    for (int c = 0; c < g.nvar; ++c) {
        double a;
        if (c < 5) {
            a = A5[c];
        } else {
            const double* Us = Ub + (long long)c * g.comp_g;
            const double ax = species_pass(Us, zc, 1, r7[0], Fm[0], left[0]);
            const double ay = species_pass(Us, zc, g.ex, r7[1], Fm[1], left[1]);
            const double az = species_pass(Us, zc, g.plane_g, r7[2], Fm[2], left[2]);
            a = -fma(az, g.rdz, fma(ay, g.rdy, ax * g.rdx));
        }
        const long long ia = za + (long long)c * g.comp_a;
        if (up.fused) {
            const double aold = up.A_old ? up.A_old[ia] : a;
            double acc = 0.0;
            for (int q = 0; q < up.nquad; ++q) acc = fma(up.w[q], up.Aq[q] ? up.Aq[q][ia] : a, acc);
            const long long iu = (long long)b * g.box_g + (long long)c * g.comp_g + zc;
            up.U_next[iu] = fma(up.dt_m, a - aold, U[iu]) + acc;
        }
        A[ia] = a;
    }
}

int launch_advance_A(cst_ctx* ctx, const double* U, double* A, double* U_next, double dt_m,
                     const double* A_old_m, const QuadArgs& q, bool fused, cudaStream_t st)
{
    const Geom& g = ctx->g;
    UpdArgs up{};
    up.fused = fused;
    up.U_next = U_next;
    up.dt_m = dt_m;
    up.A_old = (A_old_m == A) ? nullptr : A_old_m;
    up.nquad = fused ? q.nquad : 0;
    for (int n = 0; n < up.nquad; ++n) { up.Aq[n] = (q.A[n] == A) ? nullptr : q.A[n]; up.w[n] = q.w[n]; }
    const long long nt = g.comp_a * g.nbox;
    const long long nb = (nt + 127) / 128;
    k_advance_naive<<<(unsigned)nb, 128, 0, st>>>(g, U, A, up);
    ctx->launches++;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}
