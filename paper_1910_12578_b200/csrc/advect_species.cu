// advect_species.cu -- S1-S4 (+ fused S5) for the passively advected components rho X_s of <A(U)>
// (BASELINE north_star "plus passively advected rho*X_k"; Q2, Q8).
//
// F(rho X_s) = F(rho) * X_s(upwind side), so the species need only the face mass fluxes of the hydro
// kernel (workspace Fm) and 1/rho (workspace rinv).  One CTA = one 16^3 tile, same pencil <-> thread
// map as the hydro kernel (tile.cuh).  Per species: the tile core of rho X_s is staged in shared
// memory (read once from HBM, used by all three sweeps and by the fused update), each thread
// marches along its x, then y, then z pencil with the PPM window (sweep.cuh) on X = rho X / rho,
// multiplies the upwind edge value with the face mass flux, and differences consecutive faces.
// The three halo zones at either pencil end come straight from global memory.
#include "sweep.cuh"
#include "tile.cuh"

#define SP_PITCH 17
#define SP_TILE (TILE * TILE * SP_PITCH)

template <int D>
__device__ __forceinline__ void species_sweep(const Geom& g, const TileCoord& tc, const double* __restrict__ Us,
                                              const double* __restrict__ rinv_b,
                                              const double* __restrict__ Xs, const double* __restrict__ Rs,
                                              double* __restrict__ Ps, const double* __restrict__ fm_tile,
                                              double* __restrict__ A, int c, const UpdArgs& up)
{
    const int ng = CST_NG;
    const int tid = threadIdx.x, a = tid & (TILE - 1), b = tid >> 4;
    int L, ea, eb;
    if (D == 0) { L = tc.tx; ea = tc.ty; eb = tc.tz; }
    else if (D == 1) { L = tc.ty; ea = tc.tx; eb = tc.tz; }
    else { L = tc.tz; ea = tc.tx; eb = tc.ty; }
    if (a >= ea || b >= eb) return;

    long long z0, stride;
    int s0, sstride;                                    // shared-memory index of p = 0 and stride
    if (D == 0) {
        z0 = ((long long)(tc.k0 + b + ng) * g.ey + (tc.j0 + a + ng)) * g.ex + (tc.i0 + ng);
        stride = 1; s0 = (b * TILE + a) * SP_PITCH; sstride = 1;
    } else if (D == 1) {
        z0 = ((long long)(tc.k0 + b + ng) * g.ey + (tc.j0 + ng)) * g.ex + (tc.i0 + a + ng);
        stride = g.ex; s0 = (b * TILE) * SP_PITCH + a; sstride = SP_PITCH;
    } else {
        z0 = ((long long)(tc.k0 + ng) * g.ey + (tc.j0 + b + ng)) * g.ex + (tc.i0 + a + ng);
        stride = g.plane_g; s0 = b * SP_PITCH + a; sstride = TILE * SP_PITCH;
    }
    const double rd = (D == 0) ? g.rdx : (D == 1) ? g.rdy : g.rdz;
    const double* fm = fm_tile + (D * (TILE + 1)) * NTHR + tid;

    // halo zones p = -3..-1 and L..L+2 from global memory
    double hlo[3], hhi[3];
#pragma unroll
    for (int n = 0; n < 3; ++n) {
        const long long zl = z0 + (long long)(n - 3) * stride, zh = z0 + (long long)(L + n) * stride;
        hlo[n] = Us[zl] * rinv_b[zl];
        hhi[n] = Us[zh] * rinv_b[zh];
    }
    PpmWindow w;
    w.start(hlo[0]); w.warm1(hlo[1]); w.warm2(hlo[2]);
    w.warm3(Xs[s0] * Rs[s0]);
    double Fprev = 0.0;
    double fmn = fm[0];
    for (int p = 1; p <= L + 2; ++p) {
        double qn;
        if (p < L) { const int s = s0 + p * sstride; qn = Xs[s] * Rs[s]; }
        else qn = (p == L) ? hhi[0] : (p == L + 1) ? hhi[1] : hhi[2];
        w.push(qn);
        if (p >= 2) {
            const double fmc = fmn;                     // mass flux of face f = p-2
            if (p < L + 2) fmn = fm[(p - 1) * NTHR];
            const double F = fmc * (fmc >= 0.0 ? w.qpL : w.qm);
            if (p >= 3) {
                const int q = p - 3;
                const int s = s0 + q * sstride;
                const double dF = F - Fprev;
                if (D == 0) Ps[s] = -dF * rd;
                else if (D == 1) Ps[s] = fma(-dF, rd, Ps[s]);
                else {
                    const double av = fma(-dF, rd, Ps[s]);
                    const long long ia = (long long)tc.b * g.box_a + (long long)c * g.comp_a +
                        ((long long)(tc.k0 + q) * g.ny + (tc.j0 + b)) * g.nx + (tc.i0 + a);
                    if (up.fused)
                        up.U_next[(long long)tc.b * g.box_g + (long long)c * g.comp_g + z0 + (long long)q * stride] =
                            node_update(up, Xs[s], av, ia);
                    A[ia] = av;
                }
            }
            Fprev = F;
        }
    }
}

__global__ void __launch_bounds__(NTHR, 2)
k_advect_species(Geom g, TileGeom tg, const double* __restrict__ U, double* __restrict__ A,
                 const double* __restrict__ rinv, const double* __restrict__ Fm, UpdArgs up)
{
    extern __shared__ double sm[];
    double* Xs = sm;                    // rho X_s of the tile core
    double* Rs = sm + SP_TILE;          // 1/rho of the tile core
    double* Ps = sm + 2 * SP_TILE;      // x (+ y) contribution to A
    const int ng = CST_NG;
    const TileCoord tc = tile_coord(g, tg, blockIdx.x);
    const double* Ub = U + (long long)tc.b * g.box_g;
    const double* rinv_b = rinv + (long long)tc.b * g.comp_g;
    const double* fm_tile = Fm + tc.tile * 3LL * (TILE + 1) * NTHR;
    const int tid = threadIdx.x, ti = tid & (TILE - 1), tr = tid >> 4;   // tr = row group 0..15

    // stage a core array: rows (k, j), 16 zones along x each; thread (ti, tr) takes x = ti of rows tr, tr+16, ..
    auto stage = [&](const double* __restrict__ src, double* __restrict__ dst) {
        for (int row = tr; row < TILE * TILE; row += NTHR / TILE) {
            const int k = row >> 4, j = row & (TILE - 1);
            if (k < tc.tz && j < tc.ty && ti < tc.tx)
                dst[row * SP_PITCH + ti] =
                    src[((long long)(tc.k0 + k + ng) * g.ey + (tc.j0 + j + ng)) * g.ex + (tc.i0 + ti + ng)];
        }
    };
    stage(rinv_b, Rs);
    for (int s = 0; s < g.nspec; ++s) {
        const int c = 5 + s;
        const double* Us = Ub + (long long)c * g.comp_g;
        __syncthreads();                                // previous species done with Xs / Ps
        stage(Us, Xs);
        __syncthreads();
        species_sweep<0>(g, tc, Us, rinv_b, Xs, Rs, Ps, fm_tile, A, c, up);
        __syncthreads();
        species_sweep<1>(g, tc, Us, rinv_b, Xs, Rs, Ps, fm_tile, A, c, up);
        __syncthreads();
        species_sweep<2>(g, tc, Us, rinv_b, Xs, Rs, Ps, fm_tile, A, c, up);
    }
}

int launch_advect_species(cst_ctx* ctx, const double* U, double* A, const UpdArgs& up, cudaStream_t st)
{
    const Geom& g = ctx->g;
    if (g.nspec == 0) return CST_OK;
    const TileGeom tg = make_tile_geom(g);
    const size_t smem = 3ull * SP_TILE * sizeof(double);
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(k_advect_species, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return CST_ECUDA;
        attr_set = true;
    }
    const double* rinv = ctx->ws;
    const double* Fm = ctx->ws + ws_rinv_doubles(g);
    k_advect_species<<<(unsigned)tg.ntiles, NTHR, smem, st>>>(g, tg, U, A, rinv, Fm, up);
    ctx->launches++;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}
