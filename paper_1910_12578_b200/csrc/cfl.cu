// cfl.cu -- S6: CFL time step (BASELINE.json north_star; sum form, Q20):
//   dt = cfl / max_zones [ (|u|+c)/dx + (|v|+c)/dy + (|w|+c)/dz ],  c = sqrt(gamma p / rho).
// Per-thread running max -> warp shuffles -> one atomicMax per block on the bit pattern of the
// (non-negative) double, whose integer order equals its floating-point order.
#include "common.cuh"

__global__ void k_cfl_reset(double* scratch)
{
    reinterpret_cast<unsigned long long*>(scratch)[0] = 0ull;
}

// signal rate of one zone: (|u|+c)/dx + (|v|+c)/dy + (|w|+c)/dz
__device__ __forceinline__ double cfl_rate(const Geom& g, double rho, double mx, double my, double mz, double E)
{
    const double r = 1.0 / rho;
    const double u = mx * r, v = my * r, w = mz * r;
    double p = g.gm1 * (E - 0.5 * rho * (u * u + v * v + w * w));
    p = fmax(p, g.small_pres);
    const double c = sqrt(g.gamma * p * r);
    return (fabs(u) + c) * g.rdx + (fabs(v) + c) * g.rdy + (fabs(w) + c) * g.rdz;
}

// V = 2: one thread per pair of zones along x (16-byte loads; nx even, U 16-byte aligned); V = 1: one zone
template <int V>
__global__ void __launch_bounds__(256)
k_cfl_max(Geom g, const double* __restrict__ U, double* scratch)
{
    const int ng = CST_NG;
    const int nxv = g.nx / V;
    const long long total = (long long)g.nbox * g.nz * g.ny * nxv;
    double smax = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total;
         t += (long long)gridDim.x * blockDim.x) {
        const int iv = (int)(t % nxv);
        const long long r1 = t / nxv;
        const int j = (int)(r1 % g.ny);
        const long long r2 = r1 / g.ny;
        const int k = (int)(r2 % g.nz);
        const long long b = r2 / g.nz;
        const long long z = b * g.box_g + ((long long)(k + ng) * g.ey + (j + ng)) * g.ex + (iv * V + ng);
        if (V == 2) {
            double2 q[5];
#pragma unroll
            for (int c = 0; c < 5; ++c) q[c] = *reinterpret_cast<const double2*>(U + z + c * g.comp_g);
            smax = fmax(smax, cfl_rate(g, q[0].x, q[1].x, q[2].x, q[3].x, q[4].x));
            smax = fmax(smax, cfl_rate(g, q[0].y, q[1].y, q[2].y, q[3].y, q[4].y));
        } else {
            smax = fmax(smax, cfl_rate(g, U[z], U[z + g.comp_g], U[z + 2 * g.comp_g], U[z + 3 * g.comp_g],
                                       U[z + 4 * g.comp_g]));
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, o));
    __shared__ double wmax[8];
    if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = smax;
    __syncthreads();
    if (threadIdx.x < 32) {
        double m = threadIdx.x < (blockDim.x >> 5) ? wmax[threadIdx.x] : 0.0;
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (threadIdx.x == 0)
            atomicMax(reinterpret_cast<unsigned long long*>(scratch), (unsigned long long)__double_as_longlong(m));
    }
}

// cst_validate: number of interior zones whose state is not usable (a non-finite component, rho <= 0 or p <= 0)
__global__ void __launch_bounds__(256)
k_validate(Geom g, const double* __restrict__ U, unsigned long long* count)
{
    const int ng = CST_NG;
    const long long total = (long long)g.nbox * g.comp_a;
    unsigned long long bad = 0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total;
         t += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(t % g.nx);
        const long long r1 = t / g.nx;
        const int j = (int)(r1 % g.ny);
        const long long r2 = r1 / g.ny;
        const int k = (int)(r2 % g.nz);
        const long long b = r2 / g.nz;
        const long long z = b * g.box_g + ((long long)(k + ng) * g.ey + (j + ng)) * g.ex + (i + ng);
        bool ok = true;
        for (int c = 0; c < g.nvar; ++c) ok = ok && isfinite(U[z + c * g.comp_g]);
        const double rho = U[z], mx = U[z + g.comp_g], my = U[z + 2 * g.comp_g], mz = U[z + 3 * g.comp_g];
        const double p = g.gm1 * (U[z + 4 * g.comp_g] - 0.5 * (mx * mx + my * my + mz * mz) / rho);
        ok = ok && (rho > 0.0) && (p > 0.0);
        bad += ok ? 0 : 1;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) bad += __shfl_xor_sync(0xffffffffu, bad, o);
    if ((threadIdx.x & 31) == 0 && bad) atomicAdd(count, bad);
}

int launch_validate(cst_ctx* ctx, const double* U, cudaStream_t st)
{
    const Geom& g = ctx->g;
    const long long total = (long long)g.nbox * g.comp_a;
    long long nb = (total + 255) / 256;
    const long long cap = (long long)ctx->sm_count * 16;
    if (nb > cap) nb = cap;
    k_cfl_reset<<<1, 1, 0, st>>>(ctx->d_scratch + 2);
    k_validate<<<(unsigned)nb, 256, 0, st>>>(g, U, reinterpret_cast<unsigned long long*>(ctx->d_scratch + 2));
    ctx->launches += 2;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}

__global__ void k_cfl_final(const double* scratch, double cfl, double* dt_out)
{
    *dt_out = cfl / scratch[0];
}

// the two ends of the reduction on their own, for the advance call that folds the max into its z sweep (advect.cu)
int launch_cfl_reset(cst_ctx* ctx, cudaStream_t st)
{
    k_cfl_reset<<<1, 1, 0, st>>>(ctx->d_scratch);
    ctx->launches++;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}
int launch_cfl_final(cst_ctx* ctx, double cfl, double* dt_out_dev, cudaStream_t st)
{
    k_cfl_final<<<1, 1, 0, st>>>(ctx->d_scratch, cfl, dt_out_dev);
    ctx->launches++;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}

int launch_cfl(cst_ctx* ctx, const double* U, double cfl, double* dt_out_dev, cudaStream_t st)
{
    const Geom& g = ctx->g;
    const long long total = (long long)g.nbox * g.comp_a;
    const bool vec = (g.nx % 2 == 0) && (((uintptr_t)U & 15) == 0);
    long long nb = (total / (vec ? 2 : 1) + 255) / 256;
    const long long cap = (long long)ctx->sm_count * 32;
    if (nb > cap) nb = cap;
    if (nb < 1) nb = 1;
    k_cfl_reset<<<1, 1, 0, st>>>(ctx->d_scratch);
    if (vec) k_cfl_max<2><<<(unsigned)nb, 256, 0, st>>>(g, U, ctx->d_scratch);
    else     k_cfl_max<1><<<(unsigned)nb, 256, 0, st>>>(g, U, ctx->d_scratch);
    k_cfl_final<<<1, 1, 0, st>>>(ctx->d_scratch, cfl, dt_out_dev);
    ctx->launches += 3;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}
