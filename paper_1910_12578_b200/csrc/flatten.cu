// flatten.cu -- the coefficient of CW84's shock flattening (CW84 appendix; "[15, 16]"; SURVEY 8(f)
// NEXT-2 (i); include/cst.h cst_set_flattening; readings F1-F4), an OPTION that is off on the graded path.
//   F1  along direction d (u = velocity component along d):  dp = p_{i+1} - p_{i-1},  dp2 = p_{i+2} - p_{i-2},
//       z = |dp| / max(|dp2|, small_pres),  chi~_i = clamp(1 - (z - 0.75) / (0.85 - 0.75), 0, 1) if
//       u_{i-1} - u_{i+1} >= 0 and |dp| / min(p_{i+1}, p_{i-1}) > 1/3, else 1;
//   F2  chi^d_i = min(chi~_i, chi~_{i+s}), s = -1 if dp > 0 else +1;      F3  chi_i = min_d chi^d_i;
//   F4  (in the sweeps, sweep.cuh push_flat)  q+- <- chi q+- + (1 - chi) q.
// k_flatten writes chi of the zones -1 .. n (every direction) of every box into the workspace, one thread per zone.
// The shock test is a hard switch, so the primitives it looks at are formed with explicitly rounded operations in
// the order the readings state (1/rho by division, no FMA contraction): the decision is then taken on the same
// numbers whatever the compiler does.  Reads the whole 4-deep shell (edges and corners included).
#include "common.cuh"
#include "tile.cuh"

__device__ __forceinline__ void flat_prim(const Geom& g, const double* __restrict__ Ub, long long z, int d, double& p, double& ud)
{
    const double rho = Ub[z];
    const double r = __ddiv_rn(1.0, rho);
    const double u = __dmul_rn(Ub[z + g.comp_g], r), v = __dmul_rn(Ub[z + 2 * g.comp_g], r), w = __dmul_rn(Ub[z + 3 * g.comp_g], r);
    const double v2 = __dadd_rn(__dadd_rn(__dmul_rn(u, u), __dmul_rn(v, v)), __dmul_rn(w, w));
    const double pr = __dmul_rn(g.gm1, __dadd_rn(Ub[z + 4 * g.comp_g], -__dmul_rn(__dmul_rn(0.5, rho), v2)));
    p = pr < g.small_pres ? g.small_pres : pr;
    ud = d == 0 ? u : d == 1 ? v : w;
}

__device__ __forceinline__ double flat_tilde(const Geom& g, double pm2, double pm1, double pp1, double pp2, double um1, double up1)
{
    const double dp = __dadd_rn(pp1, -pm1), dp2 = __dadd_rn(pp2, -pm2);
    const double den = fabs(dp2) > g.small_pres ? fabs(dp2) : g.small_pres;
    const double z = __ddiv_rn(fabs(dp), den);
    double zeta = __dadd_rn(1.0, -__ddiv_rn(__dadd_rn(z, -0.75), __dadd_rn(0.85, -0.75)));
    zeta = zeta < 0.0 ? 0.0 : zeta;
    zeta = zeta > 1.0 ? 1.0 : zeta;
    const double pmin = pp1 < pm1 ? pp1 : pm1;
    const bool shock = (__dadd_rn(um1, -up1) >= 0.0) && (__ddiv_rn(fabs(dp), pmin) > 1.0 / 3.0);
    return shock ? zeta : 1.0;
}

__global__ void __launch_bounds__(128)
k_flatten(Geom g, const double* __restrict__ U, double* __restrict__ chi)
{
    const int ng = CST_NG;
    const int mx = g.nx + 2, my = g.ny + 2, mz = g.nz + 2;                 // zones -1 .. n
    const long long per_box = (long long)mx * my * mz, total = per_box * g.nbox;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total; t += (long long)gridDim.x * blockDim.x) {
        const int b = (int)(t / per_box);
        long long r = t - (long long)b * per_box;
        const int i = (int)(r % mx); r /= mx;
        const int j = (int)(r % my);
        const int k = (int)(r / my);
        const double* __restrict__ Ub = U + (long long)b * g.box_g;
        const long long zc = ((long long)(k + ng - 1) * g.ey + (j + ng - 1)) * g.ex + (i + ng - 1);
        double c = 1.0;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const long long st = d == 0 ? 1 : d == 1 ? (long long)g.ex : g.plane_g;
            double p[7], u[7];
#pragma unroll
            for (int n = 0; n < 7; ++n) flat_prim(g, Ub, zc + (n - 3) * st, d, p[n], u[n]);
            const double tm = flat_tilde(g, p[0], p[1], p[3], p[4], u[1], u[3]);      // zone i-1
            const double t0 = flat_tilde(g, p[1], p[2], p[4], p[5], u[2], u[4]);      // zone i
            const double tp = flat_tilde(g, p[2], p[3], p[5], p[6], u[3], u[5]);      // zone i+1
            const double nb = (__dadd_rn(p[4], -p[2]) > 0.0) ? tm : tp;
            const double cd = t0 < nb ? t0 : nb;
            c = cd < c ? cd : c;
        }
        chi[(long long)b * g.comp_g + zc] = c;
    }
}

int launch_flatten(cst_ctx* ctx, const double* U, cudaStream_t st)
{
    const Geom& g = ctx->g;
    double* chi = ctx->ws + ws_rinv_doubles(g) + ws_fm_doubles(g);
    const long long total = (long long)(g.nx + 2) * (g.ny + 2) * (g.nz + 2) * g.nbox;
    long long nb = (total + 127) / 128;
    const long long cap = (long long)ctx->sm_count * 32;
    if (nb > cap) nb = cap;
    k_flatten<<<(unsigned)nb, 128, 0, st>>>(g, U, chi);
    ctx->launches++;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}
