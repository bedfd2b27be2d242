// diffuse.cu -- explicit thermal diffusion as an extra term of <A(U)> ("thermal diffusion", L62
// "explicit diffusion"; include/cst.h cst_set_diffusion; readings D1-D3):
//   A[rho E] += k_th lap T,   T = p / ((gamma - 1) rho c_v),   second-order centred differences on the +-1 star,
// and, behind the fused call, U_next[rho E] += ca * (k_th lap T) so that the node update sees the complete A.
//
// 2.5-D streaming: a CTA of 32 x 8 threads owns a 32 x 8 patch of (i, j) and marches along k over a chunk of the
// box.  Every thread keeps T of its own zone on planes k-1, k, k+1 in registers (the z differences never touch
// shared memory); plane k, with its one-zone halo ring, sits in shared memory for the x and y differences.  Each
// zone's five conserved values are read once per patch (plus the ring).  T and the Laplacian are evaluated with
// explicitly rounded operations in the order of the readings, so that the term is reproducible bit for bit.
#include "common.cuh"

#define DF_BX 32
#define DF_BY 8
#define DF_CHUNK 32          // planes per CTA along k

__device__ __forceinline__ double diff_temperature(const Geom& g, double cv, const double* __restrict__ Ub, long long z)
{
    const double rho = Ub[z], mx = Ub[z + g.comp_g], my = Ub[z + 2 * g.comp_g], mz = Ub[z + 3 * g.comp_g];
    const double E = Ub[z + 4 * g.comp_g];
    const double u = __ddiv_rn(mx, rho), v = __ddiv_rn(my, rho), w = __ddiv_rn(mz, rho);
    const double v2 = __dadd_rn(__dadd_rn(__dmul_rn(u, u), __dmul_rn(v, v)), __dmul_rn(w, w));
    double p = __dmul_rn(g.gm1, __dadd_rn(E, -__dmul_rn(__dmul_rn(0.5, rho), v2)));
    p = p < g.small_pres ? g.small_pres : p;
    return __ddiv_rn(p, __dmul_rn(__dmul_rn(g.gm1, rho), cv));
}

__global__ void __launch_bounds__(DF_BX * DF_BY)
k_diffuse_add(Geom g, double kth, double cv, const double* __restrict__ U, double* __restrict__ A,
              double* __restrict__ U_next, double ca, int ntx, int nty, int nchunk)
{
    __shared__ double Ts[DF_BY + 2][DF_BX + 2];
    const int ng = CST_NG;
    const int tx = threadIdx.x, ty = threadIdx.y, tid = ty * DF_BX + tx;
    int blk = blockIdx.x;
    const int cz = blk % nchunk; blk /= nchunk;
    const int px = blk % ntx; blk /= ntx;
    const int py = blk % nty;
    const int b = blk / nty;
    const int i = px * DF_BX + tx, j = py * DF_BY + ty;
    const int k0 = cz * DF_CHUNK, k1 = min(g.nz, k0 + DF_CHUNK);
    const bool in = (i < g.nx) && (j < g.ny);
    const bool have = (i <= g.nx) && (j <= g.ny);   // a ragged patch also needs T of the first ghost layer inside it
    const double* __restrict__ Ub = U + (long long)b * g.box_g;
    // ring zone of this thread (threads 0 .. 2*(BX+BY)-1): left / right columns, then bottom / top rows
    int ri = 0, rj = 0;
    bool ring = false;
    if (tid < 2 * DF_BY) { rj = tid >> 1; ri = (tid & 1) ? DF_BX : -1; ring = true; }
    else if (tid < 2 * DF_BY + 2 * DF_BX) { const int t = tid - 2 * DF_BY; ri = t >> 1; rj = (t & 1) ? DF_BY : -1; ring = true; }
    const int gi = px * DF_BX + ri, gj = py * DF_BY + rj;              // interior coordinates of the ring zone (-1 .. n)
    ring = ring && gi <= g.nx && gj <= g.ny;
    const double dx2 = __dmul_rn(g.dx, g.dx), dy2 = __dmul_rn(g.dy, g.dy), dz2 = __dmul_rn(g.dz, g.dz);
    const long long zcol = ((long long)(j + ng)) * g.ex + (i + ng);    // + (k + ng) * plane
    const long long zring = ((long long)(gj + ng)) * g.ex + (gi + ng);
    double Tm = 0.0, Tc = 0.0, Tp = 0.0;
    if (have) {
        Tm = diff_temperature(g, cv, Ub, zcol + (long long)(k0 - 1 + ng) * g.plane_g);
        Tc = diff_temperature(g, cv, Ub, zcol + (long long)(k0 + ng) * g.plane_g);
    }
    for (int k = k0; k < k1; ++k) {
        if (have) {
            Tp = diff_temperature(g, cv, Ub, zcol + (long long)(k + 1 + ng) * g.plane_g);
            Ts[ty + 1][tx + 1] = Tc;
        }
        if (ring) Ts[rj + 1][ri + 1] = diff_temperature(g, cv, Ub, zring + (long long)(k + ng) * g.plane_g);
        __syncthreads();
        if (in) {
            const double lx = __ddiv_rn(__dadd_rn(__dadd_rn(Ts[ty + 1][tx + 2], -__dmul_rn(2.0, Tc)), Ts[ty + 1][tx]), dx2);
            const double ly = __ddiv_rn(__dadd_rn(__dadd_rn(Ts[ty + 2][tx + 1], -__dmul_rn(2.0, Tc)), Ts[ty][tx + 1]), dy2);
            const double lz = __ddiv_rn(__dadd_rn(__dadd_rn(Tp, -__dmul_rn(2.0, Tc)), Tm), dz2);
            const double D = __dmul_rn(kth, __dadd_rn(__dadd_rn(lx, ly), lz));
            const long long ia = (long long)b * g.box_a + 4 * g.comp_a + ((long long)k * g.ny + j) * g.nx + i;
            A[ia] = __dadd_rn(A[ia], D);
            if (U_next) {
                const long long iu = (long long)b * g.box_g + 4 * g.comp_g + zcol + (long long)(k + ng) * g.plane_g;
                U_next[iu] = fma(ca, D, U_next[iu]);
            }
        }
        Tm = Tc; Tc = Tp;
        __syncthreads();
    }
}

int launch_diffuse_add(cst_ctx* ctx, const double* U, double* A, double* U_next, double ca, cudaStream_t st)
{
    const Geom& g = ctx->g;
    const int ntx = (g.nx + DF_BX - 1) / DF_BX, nty = (g.ny + DF_BY - 1) / DF_BY, nchunk = (g.nz + DF_CHUNK - 1) / DF_CHUNK;
    const long long nb = (long long)g.nbox * ntx * nty * nchunk;
    if (nb > 0x7fffffffLL) return CST_EINVAL;
    k_diffuse_add<<<(unsigned)nb, dim3(DF_BX, DF_BY, 1), 0, st>>>(g, ctx->diff_kth, ctx->diff_cv, U, A, U_next, ca, ntx, nty, nchunk);
    ctx->launches++;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}
