// sdc_update.cu -- S5: the SDC node update, Eq. (2) of the paper with R = 0:
//   U_next = U_m + dt_m (A_new_m - A_old_m) + sum_q w_q A_q      on interior zones.
// Pure bandwidth: one thread per pair of zones along x (16-byte accesses when nx is even).
#include "common.cuh"

template <int V>
__global__ void __launch_bounds__(256)
k_sdc_update(Geom g, double* U_next, const double* U_m, double dt_m,
             const double* __restrict__ A_new, const double* __restrict__ A_old, QuadArgs q)
{
    const int ng = CST_NG;
    const int nxv = g.nx / V;
    const long long rows = (long long)g.nbox * g.nvar * g.nz * g.ny;
    const long long total = rows * nxv;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < total;
         t += (long long)gridDim.x * blockDim.x) {
        const long long row = t / nxv;
        const int iv = (int)(t - row * nxv);
        const int j = (int)(row % g.ny);
        const long long r2 = row / g.ny;
        const int k = (int)(r2 % g.nz);
        const long long bc = r2 / g.nz;                       // b*nvar + c
        const long long ia = row * g.nx + (long long)iv * V;
        const long long iu = bc * g.comp_g + ((long long)(k + ng) * g.ey + (j + ng)) * g.ex + ng + iv * V;
        if (V == 2) {
            const double2 um = *reinterpret_cast<const double2*>(U_m + iu);
            const double2 an = *reinterpret_cast<const double2*>(A_new + ia);
            const double2 ao = *reinterpret_cast<const double2*>(A_old + ia);
            double2 acc = make_double2(0.0, 0.0);
            for (int n = 0; n < q.nquad; ++n) {
                const double2 aq = *reinterpret_cast<const double2*>(q.A[n] + ia);
                acc.x = fma(q.w[n], aq.x, acc.x);
                acc.y = fma(q.w[n], aq.y, acc.y);
            }
            double2 out;
            out.x = fma(dt_m, an.x - ao.x, um.x) + acc.x;
            out.y = fma(dt_m, an.y - ao.y, um.y) + acc.y;
            *reinterpret_cast<double2*>(U_next + iu) = out;
        } else {
            double acc = 0.0;
            for (int n = 0; n < q.nquad; ++n) acc = fma(q.w[n], q.A[n][ia], acc);
            U_next[iu] = fma(dt_m, A_new[ia] - A_old[ia], U_m[iu]) + acc;
        }
    }
}

int launch_sdc_update(cst_ctx* ctx, double* U_next, const double* U_m, double dt_m,
                      const double* A_new_m, const double* A_old_m, const QuadArgs& q, cudaStream_t st)
{
    const Geom& g = ctx->g;
    bool vec = (g.nx % 2 == 0);
    const uintptr_t bits = (uintptr_t)U_next | (uintptr_t)U_m | (uintptr_t)A_new_m | (uintptr_t)A_old_m;
    if (bits & 15) vec = false;
    for (int n = 0; n < q.nquad; ++n) if ((uintptr_t)q.A[n] & 15) vec = false;
    const long long total = (long long)g.nbox * g.nvar * g.comp_a / (vec ? 2 : 1);
    long long nb = (total + 255) / 256;
    const long long cap = (long long)ctx->sm_count * 16;
    if (nb > cap) nb = cap;
    if (nb < 1) nb = 1;
    if (vec) k_sdc_update<2><<<(unsigned)nb, 256, 0, st>>>(g, U_next, U_m, dt_m, A_new_m, A_old_m, q);
    else     k_sdc_update<1><<<(unsigned)nb, 256, 0, st>>>(g, U_next, U_m, dt_m, A_new_m, A_old_m, q);
    ctx->launches++;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}
