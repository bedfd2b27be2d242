// ctu.cu -- the unsplit CTU PPM advective operator ("the main unsplit PPM hydrodynamics scheme [15, 16]",
// the solver of the paper's Strang path; include/cst.h cst_advance_ctu; readings C1-C9):
//   A_ctu(U, dt) = -div F^{n+1/2} + S,   U^{n+1} = U^n + dt A_ctu.
// Passes (one thread per zone or per face, x fastest in every array: coalesced for every direction):
//   kctu_trace<D>      C1-C4  primitives of the five zones of the stencil, CW84 parabolas (hydro.cuh), characteristic
//                             tracing over dt/2 -> the states every zone -1 .. n sends to its two D faces  (Sm, Sp)
//   kctu_flux<D, 0>    C5     F^D = HLLC(Sp[z - e_D], Sm[z]) at the low D face of zone z
//   kctu_flux<D, 1>    C6     both states corrected by dt/(3 h_T) x the T-flux difference of their own zone (conserved
//                             variables, back through S1), then HLLC -> F^{D|T}
//   kctu_flux<D, 2>    C7     both states corrected by dt/(2 h) x the two doubly-transverse flux differences -> F^{D,fin}
//   kctu_div           C8     divergence in the order ((x + y) + z) + gravity source
// The tracing switches on the signs of u - c, u, u + c; the primitives and the sound speed they are taken on are formed
// with individually rounded operations in the order of the readings (as in flatten.cu), so both sides decide alike.
// Eighteen scratch arrays of the size of U (caller-owned: cst_ctu_workspace_bytes): a straightforward multi-pass
// implementation of a NEXT row, parity-tested, not tuned.
#include "hydro.cuh"
#include "common.cuh"

struct CtuArr { double* a[18]; };          // Sm[d] = d, Sp[d] = 3 + d, F1[d] = 6 + d, Ft[d][t] = 9 + 2 d + (rank of t), Ff[d] = 15 + d
__host__ __device__ inline int ctu_ft(int d, int t) { return 9 + 2 * d + ((t > d) ? t - 1 : t); }

long long ctu_workspace_doubles(const Geom& g) { return 18LL * g.nbox * g.box_g; }

__device__ __forceinline__ double csub(double a, double b) { return __dadd_rn(a, -b); }

// S1 with individually rounded operations in the oracle's order: r = 1/rho, v = m r, p floored; returns r
__device__ __forceinline__ double ctu_prim(const Geom& g, const double* __restrict__ Ub, long long z, double W[5])
{
    const double rho = Ub[z];
    const double r = __ddiv_rn(1.0, rho);
    const double u = __dmul_rn(Ub[z + g.comp_g], r), v = __dmul_rn(Ub[z + 2 * g.comp_g], r), w = __dmul_rn(Ub[z + 3 * g.comp_g], r);
    const double v2 = __dadd_rn(__dadd_rn(__dmul_rn(u, u), __dmul_rn(v, v)), __dmul_rn(w, w));
    const double p = __dmul_rn(g.gm1, csub(Ub[z + 4 * g.comp_g], __dmul_rn(__dmul_rn(0.5, rho), v2)));
    W[0] = rho; W[1] = u; W[2] = v; W[3] = w; W[4] = p < g.small_pres ? g.small_pres : p;
    return r;
}

// CW84 parabola of the middle zone of q[0..4] (S2 steps 1-3, the forms of hydro.cuh)
__device__ __forceinline__ void ctu_parabola(const double q[5], double& qm, double& qp)
{
    const double d1 = q[1] - q[0], d2 = q[2] - q[1], d3 = q[3] - q[2], d4 = q[4] - q[3];
    const double s1 = slope2(d1, d2), s2 = slope2(d2, d3), s3 = slope2(d3, d4);
    double a = edge_value(q[1], d2, s1, s2), b = edge_value(q[2], d3, s2, s3);
    monotonize(q[2], a, b);
    qm = a; qp = b;
}

__device__ __forceinline__ double ctu_Ip(double qm, double qp, double q, double sigma)
{
    const double Dq = qp - qm, q6 = 6.0 * (q - 0.5 * (qm + qp));
    return qp - 0.5 * sigma * (Dq - (1.0 - (2.0 / 3.0) * sigma) * q6);
}
__device__ __forceinline__ double ctu_Im(double qm, double qp, double q, double sigma)
{
    const double Dq = qp - qm, q6 = 6.0 * (q - 0.5 * (qm + qp));
    return qm + 0.5 * sigma * (Dq + (1.0 - (2.0 / 3.0) * sigma) * q6);
}

// ---------------------------------------------------------------------------------------- C1-C4 ----
template <int D>
__global__ void __launch_bounds__(128)
kctu_trace(Geom g, CtuArr arr, const double* __restrict__ U, double dtdx, double hdt)
{
    const int ng = CST_NG;
    const int mx = g.nx + 2, my = g.ny + 2, mz = g.nz + 2;               // zones -1 .. n
    const long long per_box = (long long)mx * my * mz, total = per_box * g.nbox;
    const long long st = D == 0 ? 1 : D == 1 ? (long long)g.ex : g.plane_g;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int b = (int)(t / per_box);
        long long r = t - (long long)b * per_box;
        const int i = (int)(r % mx) - 1; r /= mx;
        const int j = (int)(r % my) - 1;
        const int k = (int)(r / my) - 1;
        const long long z = ((long long)(k + ng) * g.ey + (j + ng)) * g.ex + (i + ng);
        const double* __restrict__ Ub = U + (long long)b * g.box_g;
        double* __restrict__ Sm = arr.a[D] + (long long)b * g.box_g + z;
        double* __restrict__ Sp = arr.a[3 + D] + (long long)b * g.box_g + z;
        double W[5][5], rr[5];                                               // [zone of the stencil][variable]
#pragma unroll
        for (int n = 0; n < 5; ++n) rr[n] = ctu_prim(g, Ub, z + (n - 2) * st, W[n]);
        const double rho = W[2][0], u = W[2][1 + D], p = W[2][4];
        const double c = __dsqrt_rn(__ddiv_rn(__dmul_rn(g.gamma, p), rho));
        const double lam[3] = { csub(u, c), u, __dadd_rn(u, c) };
        double sig[3];
#pragma unroll
        for (int w = 0; w < 3; ++w) sig[w] = fabs(lam[w]) * dtdx;
        double qm[5], qp[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            const double q[5] = { W[0][v], W[1][v], W[2][v], W[3][v], W[4][v] };
            ctu_parabola(q, qm[v], qp[v]);
        }
        const int iv[3] = { 0, 1 + D, 4 };
#pragma unroll
        for (int side = 0; side < 2; ++side) {                               // 0: minus face, 1: plus face
            bool tw[3];
#pragma unroll
            for (int w = 0; w < 3; ++w) tw[w] = side ? (lam[w] > 0.0) : (lam[w] < 0.0);
            double I[3][3];
#pragma unroll
            for (int w = 0; w < 3; ++w)
#pragma unroll
                for (int v = 0; v < 3; ++v)
                    I[w][v] = side ? ctu_Ip(qm[iv[v]], qp[iv[v]], W[2][iv[v]], sig[w]) : ctu_Im(qm[iv[v]], qp[iv[v]], W[2][iv[v]], sig[w]);
            const int kref = side ? 2 : 0;
            double ref[3];
#pragma unroll
            for (int v = 0; v < 3; ++v) ref[v] = tw[kref] ? I[kref][v] : W[2][iv[v]];
            double ap = 0.0, am = 0.0, a0 = 0.0;
            if (tw[2]) { const double du = ref[1] - I[2][1], dp = ref[2] - I[2][2]; ap = 0.5 * (dp / (rho * c) + du) * rho / c; }
            if (tw[0]) { const double du = ref[1] - I[0][1], dp = ref[2] - I[0][2]; am = 0.5 * (dp / (rho * c) - du) * rho / c; }
            if (tw[1]) { const double dr = ref[0] - I[1][0], dp = ref[2] - I[1][2]; a0 = dr - dp / (c * c); }
            double out[5];
            out[0] = ref[0] - ((ap + am) + a0);
            out[1 + D] = ref[1] - (ap - am) * c / rho;
            out[4] = ref[2] - (ap + am) * (c * c);
#pragma unroll
            for (int v = 1; v <= 3; ++v) {
                if (v == 1 + D) continue;
                out[v] = tw[1] ? (side ? ctu_Ip(qm[v], qp[v], W[2][v], sig[1]) : ctu_Im(qm[v], qp[v], W[2][v], sig[1])) : W[2][v];
            }
#pragma unroll
            for (int e = 0; e < 3; ++e) out[1 + e] += hdt * g.grav[e];       // C4
            double* __restrict__ S = side ? Sp : Sm;
#pragma unroll
            for (int v = 0; v < 5; ++v) S[v * g.comp_g] = out[v];
        }
        for (int s = 5; s < g.nvar; ++s) {                                   // species: passive on the u wave
            const double* us = Ub + s * g.comp_g + z;
            const double q[5] = { __dmul_rn(us[-2 * st], rr[0]), __dmul_rn(us[-st], rr[1]), __dmul_rn(us[0], rr[2]),
                                  __dmul_rn(us[st], rr[3]), __dmul_rn(us[2 * st], rr[4]) };
            double xm, xp;
            ctu_parabola(q, xm, xp);
            Sm[s * g.comp_g] = (lam[1] < 0.0) ? ctu_Im(xm, xp, q[2], sig[1]) : q[2];
            Sp[s * g.comp_g] = (lam[1] > 0.0) ? ctu_Ip(xm, xp, q[2], sig[1]) : q[2];
        }
    }
}

// ---------------------------------------------------------------------------------------- C5-C7 ----
struct CtuRange { int lo[3], ext[3]; };      // zone coordinates lo .. lo + ext - 1 per direction

// state of zone zz (side: 0 = Sm, 1 = Sp of direction D) -> conserved, minus the transverse flux differences of the zone
// (MODE 1: one direction T1 with dt / (3 h); MODE 2: T1 < T2 with dt / (2 h) each), back to primitives (S1, floors);
// hydro part here, the species are done one by one by the caller with the r_new and rho_old this returns
template <int MODE>
__device__ __forceinline__ void ctu_corrected(const Geom& g, const CtuArr& arr, int sidx, long long zz, int T1, int T2,
                                              double c1, double c2, long long st1, long long st2, int f1, int f2,
                                              double W[5], double& rho_old, double& r_new)
{
    const double* __restrict__ S = arr.a[sidx] + zz;
#pragma unroll
    for (int v = 0; v < 5; ++v) W[v] = S[v * g.comp_g];
    rho_old = W[0];
    r_new = 0.0;
    if (MODE > 0) {
        double Uc[5];
        Uc[0] = W[0]; Uc[1] = W[0] * W[1]; Uc[2] = W[0] * W[2]; Uc[3] = W[0] * W[3];
        Uc[4] = W[4] * g.rgm1 + 0.5 * W[0] * ((W[1] * W[1] + W[2] * W[2]) + W[3] * W[3]);
        const double* __restrict__ F1 = arr.a[f1] + zz;
#pragma unroll
        for (int v = 0; v < 5; ++v) Uc[v] = Uc[v] - c1 * (F1[v * g.comp_g + st1] - F1[v * g.comp_g]);
        if (MODE == 2) {
            const double* __restrict__ F2 = arr.a[f2] + zz;
#pragma unroll
            for (int v = 0; v < 5; ++v) Uc[v] = Uc[v] - c2 * (F2[v * g.comp_g + st2] - F2[v * g.comp_g]);
        }
        r_new = 1.0 / Uc[0];
        const double u = Uc[1] * r_new, v = Uc[2] * r_new, w = Uc[3] * r_new;
        const double p = g.gm1 * (Uc[4] - 0.5 * Uc[0] * ((u * u + v * v) + w * w));
        W[0] = Uc[0]; W[1] = u; W[2] = v; W[3] = w; W[4] = dmax(p, g.small_pres);
    }
    (void)T1; (void)T2;
    W[0] = dmax(W[0], g.small_dens);                    // interface floors (S2 step 4)
    W[4] = dmax(W[4], g.small_pres);
}

// species value of a state after the same correction:  X_new = (rho_old X - c1 dF1 - c2 dF2) / rho_new
template <int MODE>
__device__ __forceinline__ double ctu_corrected_x(const Geom& g, const CtuArr& arr, int sidx, long long zz, int s,
                                                  double c1, double c2, long long st1, long long st2, int f1, int f2,
                                                  double rho_old, double r_new)
{
    const double X = arr.a[sidx][zz + s * g.comp_g];
    if (MODE == 0) return X;
    const double* __restrict__ F1 = arr.a[f1] + zz + s * g.comp_g;
    double Us = rho_old * X;
    Us = Us - c1 * (F1[st1] - F1[0]);
    if (MODE == 2) {
        const double* __restrict__ F2 = arr.a[f2] + zz + s * g.comp_g;
        Us = Us - c2 * (F2[st2] - F2[0]);
    }
    return Us * r_new;
}

// flux at the low D face of every zone of the range: MODE 0 from the traced states, 1 / 2 from corrected states
template <int D, int MODE>
__global__ void __launch_bounds__(128)
kctu_flux(Geom g, CtuArr arr, CtuRange rg, int T1, int T2, double c1, double c2, int f1, int f2, int fout)
{
    const int ng = CST_NG;
    const long long per_box = (long long)rg.ext[0] * rg.ext[1] * rg.ext[2], total = per_box * g.nbox;
    const long long s3[3] = { 1, g.ex, g.plane_g };
    const long long stD = s3[D], st1 = s3[T1], st2 = s3[T2];
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int b = (int)(t / per_box);
        long long r = t - (long long)b * per_box;
        const int i = (int)(r % rg.ext[0]) + rg.lo[0]; r /= rg.ext[0];
        const int j = (int)(r % rg.ext[1]) + rg.lo[1];
        const int k = (int)(r / rg.ext[1]) + rg.lo[2];
        const long long z = (long long)b * g.box_g + ((long long)(k + ng) * g.ey + (j + ng)) * g.ex + (i + ng);
        double wl[5], wr[5], F[5], rol, rnl, ror, rnr;
        ctu_corrected<MODE>(g, arr, 3 + D, z - stD, T1, T2, c1, c2, st1, st2, f1, f2, wl, rol, rnl);     // plus state of the low neighbour
        ctu_corrected<MODE>(g, arr, D, z, T1, T2, c1, c2, st1, st2, f1, f2, wr, ror, rnr);               // minus state of this zone
        const bool left = hllc_ieee<D>(g, wl, wr, F);
        double* __restrict__ Fo = arr.a[fout] + z;
#pragma unroll
        for (int v = 0; v < 5; ++v) Fo[v * g.comp_g] = F[v];
        for (int s = 5; s < g.nvar; ++s) {
            const double X = left
                ? ctu_corrected_x<MODE>(g, arr, 3 + D, z - stD, s, c1, c2, st1, st2, f1, f2, rol, rnl)
                : ctu_corrected_x<MODE>(g, arr, D, z, s, c1, c2, st1, st2, f1, f2, ror, rnr);
            Fo[s * g.comp_g] = F[0] * X;
        }
    }
}

// ---------------------------------------------------------------------------------------- C8 ----
__global__ void __launch_bounds__(128)
kctu_div(Geom g, CtuArr arr, const double* __restrict__ U, double* __restrict__ A)
{
    const int ng = CST_NG;
    const long long total = (long long)g.nbox * g.comp_a;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(t % g.nx);
        const long long r1 = t / g.nx;
        const int j = (int)(r1 % g.ny);
        const long long r2 = r1 / g.ny;
        const int k = (int)(r2 % g.nz);
        const int b = (int)(r2 / g.nz);
        const long long z = (long long)b * g.box_g + ((long long)(k + ng) * g.ey + (j + ng)) * g.ex + (i + ng);
        const long long ia = (long long)b * g.box_a + ((long long)k * g.ny + j) * g.nx + i;
        for (int c = 0; c < g.nvar; ++c) {
            const double* fx = arr.a[15] + z + c * g.comp_g;
            const double* fy = arr.a[16] + z + c * g.comp_g;
            const double* fz = arr.a[17] + z + c * g.comp_g;
            double S = 0.0;
            if (c >= 1 && c <= 3) S = U[z] * g.grav[c - 1];
            else if (c == 4) S = (U[z + g.comp_g] * g.grav[0] + U[z + 2 * g.comp_g] * g.grav[1]) + U[z + 3 * g.comp_g] * g.grav[2];
            A[ia + c * g.comp_a] = -(((fx[1] - fx[0]) / g.dx + (fy[g.ex] - fy[0]) / g.dy) + (fz[g.plane_g] - fz[0]) / g.dz) + S;
        }
    }
}

static unsigned ctu_grid(const cst_ctx* ctx, long long total)
{
    long long nb = (total + 127) / 128;
    const long long cap = (long long)ctx->sm_count * 32;
    return (unsigned)(nb > cap ? cap : (nb < 1 ? 1 : nb));
}

template <int D>
static void ctu_dir_flux(cst_ctx* ctx, const CtuArr& arr, int mode, int T1, int T2, double c1, double c2, int f1, int f2,
                         int fout, cudaStream_t st)
{
    const Geom& g = ctx->g;
    const int n[3] = { g.nx, g.ny, g.nz };
    CtuRange rg;
    for (int t = 0; t < 3; ++t) { rg.lo[t] = -1; rg.ext[t] = n[t] + 2; }                  // -1 .. n
    rg.lo[D] = 0; rg.ext[D] = n[D] + 1;                                                    // faces 0 .. n along D
    if (mode >= 1) { rg.lo[T1] = 0; rg.ext[T1] = n[T1]; }                                  // corrected along T1: interior
    if (mode == 2) { rg.lo[T2] = 0; rg.ext[T2] = n[T2]; }
    const long long total = (long long)rg.ext[0] * rg.ext[1] * rg.ext[2] * g.nbox;
    if (mode == 0) kctu_flux<D, 0><<<ctu_grid(ctx, total), 128, 0, st>>>(g, arr, rg, T1, T2, c1, c2, f1, f2, fout);
    else if (mode == 1) kctu_flux<D, 1><<<ctu_grid(ctx, total), 128, 0, st>>>(g, arr, rg, T1, T2, c1, c2, f1, f2, fout);
    else kctu_flux<D, 2><<<ctu_grid(ctx, total), 128, 0, st>>>(g, arr, rg, T1, T2, c1, c2, f1, f2, fout);
    ctx->launches++;
}

static void ctu_flux(cst_ctx* ctx, const CtuArr& arr, int d, int mode, int T1, int T2, double c1, double c2, int f1, int f2,
                     int fout, cudaStream_t st)
{
    if (d == 0) ctu_dir_flux<0>(ctx, arr, mode, T1, T2, c1, c2, f1, f2, fout, st);
    else if (d == 1) ctu_dir_flux<1>(ctx, arr, mode, T1, T2, c1, c2, f1, f2, fout, st);
    else ctu_dir_flux<2>(ctx, arr, mode, T1, T2, c1, c2, f1, f2, fout, st);
}

int launch_advance_ctu(cst_ctx* ctx, const double* U, double dt, double* A, double* ws, cudaStream_t st)
{
    const Geom& g = ctx->g;
    CtuArr arr;
    for (int a = 0; a < 18; ++a) arr.a[a] = ws + (long long)a * g.nbox * g.box_g;
    const double h[3] = { g.dx, g.dy, g.dz };
    const long long zones = (long long)(g.nx + 2) * (g.ny + 2) * (g.nz + 2) * g.nbox;
    kctu_trace<0><<<ctu_grid(ctx, zones), 128, 0, st>>>(g, arr, U, dt / h[0], 0.5 * dt);
    kctu_trace<1><<<ctu_grid(ctx, zones), 128, 0, st>>>(g, arr, U, dt / h[1], 0.5 * dt);
    kctu_trace<2><<<ctu_grid(ctx, zones), 128, 0, st>>>(g, arr, U, dt / h[2], 0.5 * dt);
    ctx->launches += 3;
    for (int d = 0; d < 3; ++d) ctu_flux(ctx, arr, d, 0, (d + 1) % 3, (d + 2) % 3, 0.0, 0.0, 0, 0, 6 + d, st);              // C5
    for (int d = 0; d < 3; ++d)                                                                                             // C6
        for (int t = 0; t < 3; ++t)
            if (t != d) ctu_flux(ctx, arr, d, 1, t, 3 - d - t, dt / (3.0 * h[t]), 0.0, 6 + t, 0, ctu_ft(d, t), st);
    for (int d = 0; d < 3; ++d) {                                                                                           // C7
        const int t1 = d == 0 ? 1 : 0, t2 = d == 2 ? 1 : 2;
        ctu_flux(ctx, arr, d, 2, t1, t2, dt / (2.0 * h[t1]), dt / (2.0 * h[t2]), ctu_ft(t1, t2), ctu_ft(t2, t1), 15 + d, st);
    }
    kctu_div<<<ctu_grid(ctx, (long long)g.nbox * g.comp_a), 128, 0, st>>>(g, arr, U, A);                                    // C8
    ctx->launches++;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}
