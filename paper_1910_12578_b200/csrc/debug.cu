// debug.cu -- test aids behind the C ABI (include/cst.h "test aids"): nothing here is on the hot path.
//   cst_debug_rcp_sqrt : evaluates the kernels' own reciprocal / square-root sequences (hydro.cuh rcp_fast,
//                        sqrt_fast) on an array, so that tests can measure their error in ulps over the range of
//                        arguments the method produces (densities, pressures, wave-speed differences).
//   cst_debug_tile_map : every CTA of the advance kernels' grid writes the tile it would work on, so that tests
//                        can check that blockIdx -> tile (tile.cuh tile_coord, brick walk included) is a bijection.
#include "hydro.cuh"
#include "tile.cuh"

__global__ void k_debug_rcp_sqrt(const double* __restrict__ x, double* __restrict__ r, double* __restrict__ s, long long n)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        r[i] = rcp_fast(x[i]);
        s[i] = sqrt_fast(x[i]);
    }
}

__global__ void k_debug_tile_map(Geom g, TileGeom tg, int* __restrict__ out)
{
    const TileCoord tc = tile_coord(g, tg, blockIdx.x);
    if (threadIdx.x == 0) {
        int* o = out + 8LL * blockIdx.x;
        o[0] = tc.b; o[1] = tc.i0; o[2] = tc.j0; o[3] = tc.k0; o[4] = tc.tx; o[5] = tc.ty; o[6] = tc.tz;
        o[7] = (int)tc.tile;
    }
}

int launch_debug_rcp_sqrt(const double* x, double* r, double* s, long long n, cudaStream_t st)
{
    k_debug_rcp_sqrt<<<256, 256, 0, st>>>(x, r, s, n);
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}

long long debug_tile_count(const Geom& g) { return make_tile_geom(g).ntiles; }

int launch_debug_tile_map(cst_ctx* ctx, int* out, cudaStream_t st)
{
    const TileGeom tg = make_tile_geom(ctx->g);
    k_debug_tile_map<<<(unsigned)tg.ntiles, 32, 0, st>>>(ctx->g, tg, out);
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}
