// ghost_fill.cu -- S0: fill the 4-deep ghost shell of every box (include/cst.h; Q16).
// One thread per ghost zone (all components); ghost zones are enumerated region by region
// (z slabs, then y slabs, then x slabs) so that no thread is spent on interior zones.
// Sources are always interior zones, so the in-place fill has no ordering hazard.
// When the context's boxes are a brick of a larger lattice (cst_set_sublattice, exchange.cu) the zone map is the
// GLOBAL one; ghost zones whose source box lives on another rank are left for cst_exchange_unpack.
#include "common.cuh"

__device__ __forceinline__ int map_dir(int g, int D, int bc_lo, int bc_hi, bool& flip)
{   // global index g (may lie outside [0,D)) -> in-domain source index
    flip = false;
    if (g < 0) {
        if (bc_lo == CST_BC_PERIODIC) return g + D * ((-g + D - 1) / D);
        if (bc_lo == CST_BC_OUTFLOW) return 0;
        flip = true;
        return -1 - g;
    }
    if (g >= D) {
        if (bc_hi == CST_BC_PERIODIC) return g % D;
        if (bc_hi == CST_BC_OUTFLOW) return D - 1;
        flip = true;
        return 2 * D - 1 - g;
    }
    return g;
}

__global__ void __launch_bounds__(256)
k_fill_ghosts(Geom g, double* __restrict__ U, long long n0, long long n1, long long n2, unsigned blocks_per_box)
{
    const int ng = CST_NG;
    const int b = blockIdx.x / blocks_per_box;          // 1-D grid: no limit on the number of boxes
    const int bi = b % g.nbx, bj = (b / g.nbx) % g.nby, bk = b / (g.nbx * g.nby);
    const long long ntot = n0 + n1 + n2;
    const long long t = (long long)(blockIdx.x - (unsigned)b * blocks_per_box) * blockDim.x + threadIdx.x;
    if (t >= ntot) return;
    int i, j, k;
    if (t < n0) {                       // z slabs: all j, all i
        const int kk = (int)(t / g.plane_g);
        const int r = (int)(t - (long long)kk * g.plane_g);
        k = kk < ng ? kk : kk + g.nz;
        j = r / g.ex; i = r - j * g.ex;
    } else if (t < n0 + n1) {           // y slabs: interior k, all i
        const long long s = t - n0;
        const int row = (int)(s / g.ex);
        i = (int)(s - (long long)row * g.ex);
        const int kk = row / (2 * ng), jj = row - kk * 2 * ng;
        k = kk + ng;
        j = jj < ng ? jj : jj + g.ny;
    } else {                            // x slabs: interior k and j
        const long long s = t - n0 - n1;
        const int row = (int)(s / (2 * ng));
        const int ii = (int)(s - (long long)row * 2 * ng);
        const int kk = row / g.ny, jj = row - kk * g.ny;
        k = kk + ng; j = jj + ng;
        i = ii < ng ? ii : ii + g.nx;
    }
    bool fx, fy, fz;
    const int sx = map_dir((bi + g.obx) * g.nx + i - ng, g.gnbx * g.nx, g.bc_lo[0], g.bc_hi[0], fx);
    const int sy = map_dir((bj + g.oby) * g.ny + j - ng, g.gnby * g.ny, g.bc_lo[1], g.bc_hi[1], fy);
    const int sz = map_dir((bk + g.obz) * g.nz + k - ng, g.gnbz * g.nz, g.bc_lo[2], g.bc_hi[2], fz);
    const int gbi = sx / g.nx, gbj = sy / g.ny, gbk = sz / g.nz;          // source box in the global lattice
    const int sbi = gbi - g.obx, sbj = gbj - g.oby, sbk = gbk - g.obz;    // ... in this rank's brick
    if (sbi < 0 || sbi >= g.nbx || sbj < 0 || sbj >= g.nby || sbk < 0 || sbk >= g.nbz) return;   // remote source
    const int sb = sbi + g.nbx * (sbj + g.nby * sbk);
    // the zone map is the same for every component: one thread moves all NVAR values of its ghost zone
    const double* __restrict__ src = U + uidx(g, sb, 0, sz - gbk * g.nz + ng, sy - gbj * g.ny + ng, sx - gbi * g.nx + ng);
    double* __restrict__ dst = U + uidx(g, b, 0, k, j, i);
    const double s1 = fx ? -1.0 : 1.0, s2 = fy ? -1.0 : 1.0, s3 = fz ? -1.0 : 1.0;
    int c = 0;
    for (; c + 4 <= g.nvar; c += 4) {
        double v[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) v[e] = src[(c + e) * g.comp_g];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int cc = c + e;
            const double sg = (cc == 1) ? s1 : (cc == 2) ? s2 : (cc == 3) ? s3 : 1.0;
            dst[cc * g.comp_g] = (cc >= 1 && cc <= 3) ? v[e] * sg : v[e];
        }
    }
    for (; c < g.nvar; ++c) {
        const double v = src[c * g.comp_g];
        const double sg = (c == 1) ? s1 : (c == 2) ? s2 : (c == 3) ? s3 : 1.0;
        dst[c * g.comp_g] = (c >= 1 && c <= 3) ? v * sg : v;
    }
}

int launch_fill_ghosts(cst_ctx* ctx, double* U, cudaStream_t st)
{
    const Geom& g = ctx->g;
    const int ng = CST_NG;
    const long long n0 = 2LL * ng * g.plane_g;
    const long long n1 = 2LL * ng * g.nz * g.ex;
    const long long n2 = 2LL * ng * (long long)g.nz * g.ny;
    const long long ntot = n0 + n1 + n2;
    const long long nb = (ntot + 255) / 256;
    if (nb * g.nbox > 0x7fffffffLL) return CST_EINVAL;  // more ghost zones than any device memory holds
    k_fill_ghosts<<<(unsigned)(nb * g.nbox), 256, 0, st>>>(g, U, n0, n1, n2, (unsigned)nb);
    ctx->launches++;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}
