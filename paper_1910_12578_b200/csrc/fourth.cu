// fourth.cu -- the fourth-order finite-volume <A(U)> ("a fourth-order method in space and time (using a
// Simpsons rule for the integral and the spatial reconstruction of [12])", L60; include/cst.h
// cst_set_order; readings G1-G9).  Selected with cst_set_order(ctx, 4); the graded path is order 2.
//
// Steps (all on cell AVERAGES <U>; second differences are undivided, so h^2/24 is 1/24):
//   k4_qavg        G1-G3  U^c = <U> - Lap<U>/24,  q^c = prim(U^c),  <q> = q^c + Lap(prim<U>)/24       zones -3 .. n+2
//   k4_states<D>   G4-G5  (7/12, -1/12) face averages, Colella-Sekora face limiting, the extremum-preserving limiter
//                         of [12] (without its third-difference test): W_L, W_R on every face of every line whose
//                         transverse zones lie in -1 .. n; one thread per ZONE (its two face values are recomputed by
//                         the neighbours -- cheaper than a serial march, and coalesced for every direction)
//   k4_fa<D>       G7     F^a = HLLC(W_L, W_R) on those faces
//   k4_favg<D>     G6-G7  face-centred states W - Lap_t(W)/24, F^c = HLLC, <F> = F^c + Lap_t(F^a)/24   interior lines
//   k4_div<D>      G8     A accumulates the three directions in the order ((x + y) + z), sign and gravity source last
// Everything up to the Riemann solves is written with explicitly rounded operations in the order of the readings:
// the limiter is full of comparisons, and they are then taken on the same numbers whatever the compiler contracts.
// Face arrays of direction d have extents (nx+2, ny+2, nz+2) with n_d+1 along d: index (f | t+1) per direction, x
// fastest.  This is a straightforward multi-pass implementation (five arrays of N doubles per zone in the workspace);
// the tiled, fused treatment the second-order path got is future work.
#include "hydro.cuh"
#include "common.cuh"

#define R24 (1.0 / 24.0)

struct Face4 {                       // geometry of the face arrays of one direction
    int fe[3];                       // extents
    long long per_comp, per_box;     // fe[0]*fe[1]*fe[2], nvar * that
};
__host__ __device__ inline Face4 face4(const Geom& g, int d)
{
    Face4 f;
    f.fe[0] = g.nx + 2; f.fe[1] = g.ny + 2; f.fe[2] = g.nz + 2;
    f.fe[d] = (d == 0 ? g.nx : d == 1 ? g.ny : g.nz) + 1;
    f.per_comp = (long long)f.fe[0] * f.fe[1] * f.fe[2];
    f.per_box = f.per_comp * g.nvar;
    return f;
}
long long fourth_face_doubles(const Geom& g)
{
    long long m = 0;
    for (int d = 0; d < 3; ++d) { const long long s = face4(g, d).per_box; if (s > m) m = s; }
    return m * g.nbox;
}
// workspace (doubles): [qavg: nbox*box_g][WL][WR][Fa][Favg: 4 x fourth_face_doubles]
long long fourth_workspace_doubles(const Geom& g) { return (long long)g.nbox * g.box_g + 4 * fourth_face_doubles(g); }

__device__ __forceinline__ double sub_rn(double a, double b) { return __dadd_rn(a, -b); }
// (a - 2 c) + b, the undivided second difference in the order of the readings
__device__ __forceinline__ double d2_rn(double a, double c, double b) { return __dadd_rn(sub_rn(a, __dmul_rn(2.0, c)), b); }

// S1 with explicitly rounded operations (the order of the readings): r = 1/rho, v = m r, p floored
__device__ __forceinline__ void prim4(const Geom& g, const double U5[5], double W5[5], double& r)
{
    r = __ddiv_rn(1.0, U5[0]);
    const double u = __dmul_rn(U5[1], r), v = __dmul_rn(U5[2], r), w = __dmul_rn(U5[3], r);
    const double v2 = __dadd_rn(__dadd_rn(__dmul_rn(u, u), __dmul_rn(v, v)), __dmul_rn(w, w));
    const double p = __dmul_rn(g.gm1, sub_rn(U5[4], __dmul_rn(__dmul_rn(0.5, U5[0]), v2)));
    W5[0] = U5[0]; W5[1] = u; W5[2] = v; W5[3] = w; W5[4] = p < g.small_pres ? g.small_pres : p;
}

// ---------------------------------------------------------------------------------------- G1-G3 ----
__global__ void __launch_bounds__(128)
k4_qavg(Geom g, const double* __restrict__ U, double* __restrict__ qavg)
{
    const int mx = g.ex - 2, my = g.ey - 2, mz = g.ez - 2;
    const long long per_box = (long long)mx * my * mz, total = per_box * g.nbox;
    const long long st[3] = { 1, g.ex, g.plane_g };
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int b = (int)(t / per_box);
        long long r = t - (long long)b * per_box;
        const int i = (int)(r % mx) + 1; r /= mx;
        const int j = (int)(r % my) + 1;
        const int k = (int)(r / my) + 1;
        const double* __restrict__ Ub = U + (long long)b * g.box_g;
        double* __restrict__ qb = qavg + (long long)b * g.box_g;
        const long long z = ((long long)k * g.ey + j) * g.ex + i;
        // qbar = prim(<U>) at the zone and its six neighbours (n = 0: centre; 1 + 2 d: minus d; 2 + 2 d: plus d)
        double W[7][5], rr[7], Uc5[5];
#pragma unroll
        for (int n = 0; n < 7; ++n) {
            const long long zn = z + (n == 0 ? 0 : ((n & 1) ? -st[(n - 1) >> 1] : st[(n - 1) >> 1]));
            double U5[5];
#pragma unroll
            for (int c = 0; c < 5; ++c) U5[c] = Ub[zn + c * g.comp_g];
            prim4(g, U5, W[n], rr[n]);
            if (n == 0) {
#pragma unroll
                for (int c = 0; c < 5; ++c) Uc5[c] = U5[c];
            }
        }
        // G1: U^c of the five hydro components (the neighbours' conserved values are read again: L1 hits)
#pragma unroll
        for (int c = 0; c < 5; ++c) {
            const double* u = Ub + c * g.comp_g + z;
            const double lap = __dadd_rn(__dadd_rn(d2_rn(u[st[0]], u[0], u[-st[0]]), d2_rn(u[st[1]], u[0], u[-st[1]])),
                                         d2_rn(u[st[2]], u[0], u[-st[2]]));
            Uc5[c] = sub_rn(u[0], __dmul_rn(R24, lap));
        }
        double qc[5], rc;
        prim4(g, Uc5, qc, rc);                                                     // G2: q^c
#pragma unroll
        for (int c = 0; c < 5; ++c) {
            const double lap = __dadd_rn(__dadd_rn(d2_rn(W[2][c], W[0][c], W[1][c]), d2_rn(W[4][c], W[0][c], W[3][c])),
                                         d2_rn(W[6][c], W[0][c], W[5][c]));
            qb[z + c * g.comp_g] = __dadd_rn(qc[c], __dmul_rn(R24, lap));          // G3
        }
        for (int s = 5; s < g.nvar; ++s) {
            const double* u = Ub + s * g.comp_g + z;
            const double lapU = __dadd_rn(__dadd_rn(d2_rn(u[st[0]], u[0], u[-st[0]]), d2_rn(u[st[1]], u[0], u[-st[1]])),
                                          d2_rn(u[st[2]], u[0], u[-st[2]]));
            const double Xc = __dmul_rn(sub_rn(u[0], __dmul_rn(R24, lapU)), rc);   // species of q^c
            const double X0 = __dmul_rn(u[0], rr[0]);
            const double lapX = __dadd_rn(__dadd_rn(d2_rn(__dmul_rn(u[st[0]], rr[2]), X0, __dmul_rn(u[-st[0]], rr[1])),
                                                    d2_rn(__dmul_rn(u[st[1]], rr[4]), X0, __dmul_rn(u[-st[1]], rr[3]))),
                                          d2_rn(__dmul_rn(u[st[2]], rr[6]), X0, __dmul_rn(u[-st[2]], rr[5])));
            qb[z + s * g.comp_g] = __dadd_rn(Xc, __dmul_rn(R24, lapX));
        }
    }
}

// ---------------------------------------------------------------------------------------- G4-G5 ----
// face value between zones (b, c) of the line a b | c d: G4 and G4b
__device__ __forceinline__ double face4_value(double a, double b, double c, double d)
{
    const double C = 1.25;
    double qf = sub_rn(__dmul_rn(7.0 / 12.0, __dadd_rn(b, c)), __dmul_rn(1.0 / 12.0, __dadd_rn(a, d)));
    if (__dmul_rn(sub_rn(qf, b), sub_rn(c, qf)) < 0.0) {
        const double D2 = __dmul_rn(3.0, d2_rn(b, qf, c));
        const double D2L = d2_rn(a, b, c), D2R = d2_rn(b, c, d);
        double lim = 0.0;
        if (D2 > 0.0 && D2L > 0.0 && D2R > 0.0) {
            lim = __dmul_rn(C, D2L);
            if (__dmul_rn(C, D2R) < lim) lim = __dmul_rn(C, D2R);
            if (D2 < lim) lim = D2;
        } else if (D2 < 0.0 && D2L < 0.0 && D2R < 0.0) {
            lim = __dmul_rn(C, D2L);
            if (__dmul_rn(C, D2R) > lim) lim = __dmul_rn(C, D2R);
            if (D2 > lim) lim = D2;
        }
        qf = sub_rn(__dmul_rn(0.5, __dadd_rn(b, c)), __dmul_rn(1.0 / 6.0, lim));
    }
    return qf;
}

// limited parabola edges of the middle zone of q[0..4] (G5)
__device__ __forceinline__ void limit4(const double q[5], double& qm, double& qp)
{
    const double C = 1.25;
    const double fl = face4_value(q[0], q[1], q[2], q[3]), fr = face4_value(q[1], q[2], q[3], q[4]);
    double dm = sub_rn(q[2], fl), dp = sub_rn(fr, q[2]);
    const bool extremum = (__dmul_rn(dm, dp) <= 0.0) || (__dmul_rn(sub_rn(q[2], q[0]), sub_rn(q[4], q[2])) <= 0.0);
    if (extremum) {
        const double D2f = __dmul_rn(6.0, d2_rn(fl, q[2], fr));
        const double D2l = d2_rn(q[0], q[1], q[2]), D2c = d2_rn(q[1], q[2], q[3]), D2r = d2_rn(q[2], q[3], q[4]);
        double lim = 0.0;
        if (D2f > 0.0 && D2l > 0.0 && D2c > 0.0 && D2r > 0.0) {
            lim = __dmul_rn(C, D2l);
            if (__dmul_rn(C, D2c) < lim) lim = __dmul_rn(C, D2c);
            if (__dmul_rn(C, D2r) < lim) lim = __dmul_rn(C, D2r);
            if (D2f < lim) lim = D2f;
        } else if (D2f < 0.0 && D2l < 0.0 && D2c < 0.0 && D2r < 0.0) {
            lim = __dmul_rn(C, D2l);
            if (__dmul_rn(C, D2c) > lim) lim = __dmul_rn(C, D2c);
            if (__dmul_rn(C, D2r) > lim) lim = __dmul_rn(C, D2r);
            if (D2f > lim) lim = D2f;
        }
        double qmax = fabs(q[0]);
#pragma unroll
        for (int n = 1; n < 5; ++n) qmax = fabs(q[n]) > qmax ? fabs(q[n]) : qmax;
        const double rho = (fabs(D2f) <= __dmul_rn(1e-12, qmax)) ? 0.0 : __ddiv_rn(lim, D2f);
        if (rho < 1.0 - 1e-12) {
            if (__dmul_rn(dm, dp) < 0.0) { dm = __dmul_rn(rho, dm); dp = __dmul_rn(rho, dp); }
            else if (fabs(dm) >= __dmul_rn(2.0, fabs(dp)))
                dm = __dadd_rn(__dmul_rn(__dmul_rn(2.0, sub_rn(1.0, rho)), dp), __dmul_rn(rho, dm));
            else if (fabs(dp) >= __dmul_rn(2.0, fabs(dm)))
                dp = __dadd_rn(__dmul_rn(__dmul_rn(2.0, sub_rn(1.0, rho)), dm), __dmul_rn(rho, dp));
        }
    } else {
        if (fabs(dm) >= __dmul_rn(2.0, fabs(dp))) dm = __dmul_rn(2.0, dp);
        else if (fabs(dp) >= __dmul_rn(2.0, fabs(dm))) dp = __dmul_rn(2.0, dm);
    }
    qm = sub_rn(q[2], dm);
    qp = __dadd_rn(q[2], dp);
}

// zone coordinates (i, j, k) in -1 .. n  ->  index in the face array of direction D at face f along D
__device__ __forceinline__ long long fidx(const Face4& fa, int D, int i, int j, int k, int f)
{
    const int c0 = D == 0 ? f : i + 1, c1 = D == 1 ? f : j + 1, c2 = D == 2 ? f : k + 1;
    return ((long long)c2 * fa.fe[1] + c1) * fa.fe[0] + c0;
}

template <int D>
__global__ void __launch_bounds__(128)
k4_states(Geom g, Face4 fa, const double* __restrict__ qavg, double* __restrict__ WL, double* __restrict__ WR)
{
    const int ng = CST_NG;
    const int mx = g.nx + 2, my = g.ny + 2, mz = g.nz + 2;               // zones -1 .. n
    const long long per_box = (long long)mx * my * mz, total = per_box * g.nbox;
    const long long st = D == 0 ? 1 : D == 1 ? (long long)g.ex : g.plane_g;
    const int nd = D == 0 ? g.nx : D == 1 ? g.ny : g.nz;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int b = (int)(t / per_box);
        long long r = t - (long long)b * per_box;
        const int i = (int)(r % mx) - 1; r /= mx;
        const int j = (int)(r % my) - 1;
        const int k = (int)(r / my) - 1;
        const int id = D == 0 ? i : D == 1 ? j : k;                      // coordinate along the line
        const long long z = ((long long)(k + ng) * g.ey + (j + ng)) * g.ex + (i + ng);
        const double* __restrict__ qb = qavg + (long long)b * g.box_g + z;
        double* __restrict__ wl = WL + (long long)b * fa.per_box;
        double* __restrict__ wr = WR + (long long)b * fa.per_box;
        for (int c = 0; c < g.nvar; ++c) {
            const double* q0 = qb + c * g.comp_g;
            const double q[5] = { q0[-2 * st], q0[-st], q0[0], q0[st], q0[2 * st] };
            double qm, qp;
            limit4(q, qm, qp);
            if (id >= 0) wr[c * fa.per_comp + fidx(fa, D, i, j, k, id)] = qm;            // right state of face id
            if (id < nd) wl[c * fa.per_comp + fidx(fa, D, i, j, k, id + 1)] = qp;        // left state of face id + 1
        }
    }
}

// ---------------------------------------------------------------------------------------- G6-G7 ----
__device__ __forceinline__ void floor4(const Geom& g, double W[5])
{
    W[0] = dmax(W[0], g.small_dens);
    W[4] = dmax(W[4], g.small_pres);
}

// F^a = HLLC(W_L, W_R) on every face of every line with transverse zones -1 .. n
template <int D>
__global__ void __launch_bounds__(128)
k4_fa(Geom g, Face4 fa, const double* __restrict__ WL, const double* __restrict__ WR, double* __restrict__ Fa)
{
    const long long total = fa.per_comp * g.nbox;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int b = (int)(t / fa.per_comp);
        const long long w = t - (long long)b * fa.per_comp + (long long)b * fa.per_box;
        double wl[5], wr[5], F[5];
#pragma unroll
        for (int c = 0; c < 5; ++c) { wl[c] = WL[w + c * fa.per_comp]; wr[c] = WR[w + c * fa.per_comp]; }
        floor4(g, wl); floor4(g, wr);
        const bool left = hllc_ieee<D>(g, wl, wr, F);
#pragma unroll
        for (int c = 0; c < 5; ++c) Fa[w + c * fa.per_comp] = F[c];
        for (int s = 5; s < g.nvar; ++s)               // Q8: mass flux x upwind X
            Fa[w + s * fa.per_comp] = F[0] * (left ? WL[w + s * fa.per_comp] : WR[w + s * fa.per_comp]);
    }
}

__device__ __forceinline__ double lap_t(const double* __restrict__ a, long long sa, long long sb)
{   // (a+ - 2 a + a-) along the first transverse direction + the same along the second
    return __dadd_rn(d2_rn(a[sa], a[0], a[-sa]), d2_rn(a[sb], a[0], a[-sb]));
}

// face-centred states, F^c and the face-average flux on the faces of interior lines
template <int D>
__global__ void __launch_bounds__(128)
k4_favg(Geom g, Face4 fa, const double* __restrict__ WL, const double* __restrict__ WR, const double* __restrict__ Fa,
        double* __restrict__ Fv)
{
    const int nf = fa.fe[D];
    const int na = D == 0 ? g.ny : g.nx, nb = D == 2 ? g.ny : g.nz;      // interior extents of the transverse directions a < b
    const long long per_box = (long long)nf * na * nb, total = per_box * g.nbox;
    const int A_ = D == 0 ? 1 : 0, B_ = D == 2 ? 1 : 2;
    const long long s3[3] = { 1, fa.fe[0], (long long)fa.fe[0] * fa.fe[1] };
    const long long sa = s3[A_], sb = s3[B_];
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int b = (int)(t / per_box);
        long long r = t - (long long)b * per_box;
        // x-fastest enumeration of (f, a, b) in array order
        int c3[3];
        const int e0 = D == 0 ? nf : g.nx, e1 = D == 1 ? nf : g.ny;
        c3[0] = (int)(r % e0); r /= e0;
        c3[1] = (int)(r % e1);
        c3[2] = (int)(r / e1);
        const int i = D == 0 ? 0 : c3[0], j = D == 1 ? 0 : c3[1], k = D == 2 ? 0 : c3[2];
        const long long w = (long long)b * fa.per_box + fidx(fa, D, i, j, k, c3[D]);
        double wl[5], wr[5], Fc[5];
#pragma unroll
        for (int c = 0; c < 5; ++c) {
            const double* l = WL + w + c * fa.per_comp;
            const double* rgt = WR + w + c * fa.per_comp;
            wl[c] = sub_rn(l[0], __dmul_rn(R24, lap_t(l, sa, sb)));                      // G6
            wr[c] = sub_rn(rgt[0], __dmul_rn(R24, lap_t(rgt, sa, sb)));
        }
        floor4(g, wl); floor4(g, wr);
        const bool left = hllc_ieee<D>(g, wl, wr, Fc);
#pragma unroll
        for (int c = 0; c < 5; ++c)
            Fv[w + c * fa.per_comp] = Fc[c] + R24 * lap_t(Fa + w + c * fa.per_comp, sa, sb);           // G7
        for (int s = 5; s < g.nvar; ++s) {
            const double* l = WL + w + s * fa.per_comp;
            const double* rgt = WR + w + s * fa.per_comp;
            const double xl = sub_rn(l[0], __dmul_rn(R24, lap_t(l, sa, sb)));
            const double xr = sub_rn(rgt[0], __dmul_rn(R24, lap_t(rgt, sa, sb)));
            const double fc = Fc[0] * (left ? xl : xr);
            Fv[w + s * fa.per_comp] = fc + R24 * lap_t(Fa + w + s * fa.per_comp, sa, sb);
        }
    }
}

// G8: A accumulates direction D (x, then y, then z: ((x + y) + z)); the z pass applies the sign and the source
template <int D>
__global__ void __launch_bounds__(128)
k4_div(Geom g, Face4 fa, const double* __restrict__ Fv, const double* __restrict__ U, double* __restrict__ A)
{
    const int ng = CST_NG;
    const long long total = (long long)g.nbox * g.comp_a;
    const double h = D == 0 ? g.dx : D == 1 ? g.dy : g.dz;
    const long long s3[3] = { 1, fa.fe[0], (long long)fa.fe[0] * fa.fe[1] };
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(t % g.nx);
        const long long r1 = t / g.nx;
        const int j = (int)(r1 % g.ny);
        const long long r2 = r1 / g.ny;
        const int k = (int)(r2 % g.nz);
        const int b = (int)(r2 / g.nz);
        const int id = D == 0 ? i : D == 1 ? j : k;
        const long long w = (long long)b * fa.per_box + fidx(fa, D, i, j, k, id);
        const long long ia = (long long)b * g.box_a + ((long long)k * g.ny + j) * g.nx + i;
        const long long zu = (long long)b * g.box_g + ((long long)(k + ng) * g.ey + (j + ng)) * g.ex + (i + ng);
        for (int c = 0; c < g.nvar; ++c) {
            const double* f = Fv + w + c * fa.per_comp;
            const double dF = __ddiv_rn(sub_rn(f[s3[D]], f[0]), h);
            double* a = A + ia + c * g.comp_a;
            if (D == 0) *a = dF;
            else if (D == 1) *a = __dadd_rn(*a, dF);
            else {
                double S = 0.0;
                if (c >= 1 && c <= 3) S = __dmul_rn(U[zu], g.grav[c - 1]);
                else if (c == 4)
                    S = __dadd_rn(__dadd_rn(__dmul_rn(U[zu + g.comp_g], g.grav[0]), __dmul_rn(U[zu + 2 * g.comp_g], g.grav[1])),
                                  __dmul_rn(U[zu + 3 * g.comp_g], g.grav[2]));
                *a = __dadd_rn(-__dadd_rn(*a, dF), S);
            }
        }
    }
}

static unsigned grid4(const cst_ctx* ctx, long long total)
{
    long long nb = (total + 127) / 128;
    const long long cap = (long long)ctx->sm_count * 32;
    return (unsigned)(nb > cap ? cap : (nb < 1 ? 1 : nb));
}

template <int D>
static void launch_dir(cst_ctx* ctx, const double* U, double* A, double* qavg, double* WL, double* WR, double* Fa,
                       double* Fv, cudaStream_t st)
{
    const Geom& g = ctx->g;
    const Face4 fa = face4(g, D);
    const long long zones = (long long)(g.nx + 2) * (g.ny + 2) * (g.nz + 2) * g.nbox;
    const int nf = fa.fe[D], na = D == 0 ? g.ny : g.nx, nb = D == 2 ? g.ny : g.nz;
    k4_states<D><<<grid4(ctx, zones), 128, 0, st>>>(g, fa, qavg, WL, WR);
    k4_fa<D><<<grid4(ctx, fa.per_comp * g.nbox), 128, 0, st>>>(g, fa, WL, WR, Fa);
    k4_favg<D><<<grid4(ctx, (long long)nf * na * nb * g.nbox), 128, 0, st>>>(g, fa, WL, WR, Fa, Fv);
    k4_div<D><<<grid4(ctx, (long long)g.nbox * g.comp_a), 128, 0, st>>>(g, fa, Fv, U, A);
    ctx->launches += 4;
}

int launch_advance_A4(cst_ctx* ctx, const double* U, double* A, cudaStream_t st)
{
    const Geom& g = ctx->g;
    double* qavg = ctx->ws;
    const long long fd = fourth_face_doubles(g);
    double* WL = qavg + (long long)g.nbox * g.box_g;
    double *WR = WL + fd, *Fa = WR + fd, *Fv = Fa + fd;
    k4_qavg<<<grid4(ctx, (long long)(g.ex - 2) * (g.ey - 2) * (g.ez - 2) * g.nbox), 128, 0, st>>>(g, U, qavg);
    ctx->launches++;
    launch_dir<0>(ctx, U, A, qavg, WL, WR, Fa, Fv, st);
    launch_dir<1>(ctx, U, A, qavg, WL, WR, Fa, Fv, st);
    launch_dir<2>(ctx, U, A, qavg, WL, WR, Fa, Fv, st);
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}
