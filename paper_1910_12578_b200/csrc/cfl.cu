// cfl.cu -- S6: CFL time step (BASELINE.json north_star; sum form, Q20):
//   dt = cfl / max_zones [ (|u|+c)/dx + (|v|+c)/dy + (|w|+c)/dz ],  c = sqrt(gamma p / rho).
// Per-thread running max -> warp shuffles -> one atomicMax per block on the bit pattern of the
// (non-negative) double, whose integer order equals its floating-point order.
#include "common.cuh"

__global__ void k_cfl_reset(double* scratch)
{
    reinterpret_cast<unsigned long long*>(scratch)[0] = 0ull;
}

__global__ void __launch_bounds__(256)
k_cfl_max(Geom g, const double* __restrict__ U, double* scratch)
{
    const int ng = CST_NG;
    const long long total = (long long)g.nbox * g.comp_a;
    double smax = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total;
         t += (long long)gridDim.x * blockDim.x) {
        const int i = (int)(t % g.nx);
        const long long r1 = t / g.nx;
        const int j = (int)(r1 % g.ny);
        const long long r2 = r1 / g.ny;
        const int k = (int)(r2 % g.nz);
        const long long b = r2 / g.nz;
        const long long z = b * g.box_g + ((long long)(k + ng) * g.ey + (j + ng)) * g.ex + (i + ng);
        const double rho = U[z];
        const double r = 1.0 / rho;
        const double u = U[z + g.comp_g] * r, v = U[z + 2 * g.comp_g] * r, w = U[z + 3 * g.comp_g] * r;
        double p = g.gm1 * (U[z + 4 * g.comp_g] - 0.5 * rho * (u * u + v * v + w * w));
        p = fmax(p, g.small_pres);
        const double c = sqrt(g.gamma * p * r);
        const double s = (fabs(u) + c) * g.rdx + (fabs(v) + c) * g.rdy + (fabs(w) + c) * g.rdz;
        smax = fmax(smax, s);
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

__global__ void k_cfl_final(const double* scratch, double cfl, double* dt_out)
{
    *dt_out = cfl / scratch[0];
}

int launch_cfl(cst_ctx* ctx, const double* U, double cfl, double* dt_out_dev, cudaStream_t st)
{
    const Geom& g = ctx->g;
    const long long total = (long long)g.nbox * g.comp_a;
    long long nb = (total + 255) / 256;
    const long long cap = (long long)ctx->sm_count * 8;
    if (nb > cap) nb = cap;
    k_cfl_reset<<<1, 1, 0, st>>>(ctx->d_scratch);
    k_cfl_max<<<(unsigned)nb, 256, 0, st>>>(g, U, ctx->d_scratch);
    k_cfl_final<<<1, 1, 0, st>>>(ctx->d_scratch, cfl, dt_out_dev);
    ctx->launches += 3;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}
