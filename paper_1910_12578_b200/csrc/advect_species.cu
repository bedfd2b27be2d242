// advect_species.cu -- S1-S4 (+ fused S5) for the passively advected components rho X_s of <A(U)>
// (BASELINE north_star "plus passively advected rho*X_k"; Q2, Q8).
//
// F(rho X_s) = F(rho) * X_s(upwind side), so the species need only the face mass fluxes of the hydro
// kernel (workspace Fm) and 1/rho (workspace rinv).  One CTA = one 16^3 tile, same pencil <-> thread
// map as the hydro kernel (tile.cuh).  Per species: X = rho X_s / rho of the tile core is staged in
// shared memory (rho X_s read once from HBM, used by all three sweeps), each thread marches along
// its x, then y, then z pencil with the PPM window (sweep.cuh), multiplies the upwind edge value
// with the face mass flux, and differences consecutive faces.  The three halo zones at either
// pencil end come straight from global memory into the window.  The contributions to A accumulate
// in a second shared array.
//
// Two kernels, same arithmetic:
//   k_advect_species_tma (species_tma.cuh) -- boxes made of full 16^3 tiles (every BASELINE config): TMA tile loads
//                          double-buffered on mbarriers, L2 prefetches of every other operand stream, three CTAs
//                          per tile (each a contiguous share of the species), two CTAs per SM;
//   k_advect_species (below) -- any box shape (ragged tiles), unaligned arrays, or no TMA driver entry point.
#include "sweep.cuh"
#include "tile.cuh"
#include "species_tma.cuh"

#ifndef SPT_SPLIT
#define SPT_SPLIT 3     // consecutive CTAs that share one tile (each takes a contiguous share of the species)
#endif

#define SP_PITCH 17
#define SP_TILE (TILE * TILE * SP_PITCH)

// --------------------------------------------------------------------------- any tile extent ----
template <int D, int NR, bool FLAT>
__device__ __forceinline__ void species_sweep(const Geom& g, const TileCoord& tc, const double* __restrict__ Us,
                                              const double* __restrict__ rinv_b,
                                              const double* __restrict__ Xs, double* __restrict__ Ps,
                                              const double* __restrict__ fm_tile,
                                              double* __restrict__ A, int c, const UpdArgs& up,
                                              const double* __restrict__ chi_b)
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
    const double nrd = -((D == 0) ? g.rdx : (D == 1) ? g.rdy : g.rdz);
    const double* fm = fm_tile + (D * (TILE + 1)) * NTHR + tid;

    double hlo[3], hhi[3];
#pragma unroll
    for (int n = 0; n < 3; ++n) {
        const long long zl = z0 + (long long)(n - 3) * stride, zh = z0 + (long long)(L + n) * stride;
        hlo[n] = Us[zl] * rinv_b[zl];
        hhi[n] = Us[zh] * rinv_b[zh];
    }
    PpmWindow w;
    w.start(hlo[0]); w.warm1(hlo[1]); w.warm2(hlo[2]);
    w.warm3(Xs[s0]);
    double Fprev = 0.0;
    double fmn = fm[0];
    for (int p = 1; p <= L + 2; ++p) {
        double qn;
        if (p < L) qn = Xs[s0 + p * sstride];
        else qn = (p == L) ? hhi[0] : (p == L + 1) ? hhi[1] : hhi[2];
        if (FLAT) w.push_flat(qn, chi_b[z0 + (long long)(p - 2) * stride]);   // optional CW84 flattening of zone p-2
        else w.push(qn);
        if (p >= 2) {
            const double fmc = fmn;                     // mass flux of face f = p-2
            if (p < L + 2) fmn = fm[(p - 1) * NTHR];
            const double F = fmc * (sign_bit(fmc) ? w.qm : w.qpL);
            if (p >= 3) {
                const int q = p - 3;
                const int s = s0 + q * sstride;
                const double dF = F - Fprev;
                if (D == 0) Ps[s] = dF * nrd;
                else if (D == 1) Ps[s] = fma(dF, nrd, Ps[s]);
                else {
                    const double av = fma(dF, nrd, Ps[s]);
                    const long long ia = (long long)tc.b * g.box_a + (long long)c * g.comp_a +
                        ((long long)(tc.k0 + q) * g.ny + (tc.j0 + b)) * g.nx + (tc.i0 + a);
                    if (NR >= 0) {
                        const long long iu = (long long)tc.b * g.box_g + (long long)c * g.comp_g + z0 + (long long)q * stride;
                        up.U_next[iu] = node_update<NR>(up, up.U_m[iu], av, ia);
                    }
                    A[ia] = av;
                }
            }
            Fprev = F;
        }
    }
}

template <int NR, bool FLAT>
__global__ void __launch_bounds__(NTHR, 2)
k_advect_species(Geom g, TileGeom tg, const double* __restrict__ U, double* __restrict__ A,
                 const double* __restrict__ rinv, const double* __restrict__ Fm, UpdArgs up, const double* __restrict__ chi)
{
    extern __shared__ double sm[];
    double* Xs = sm;                    // X_s = rho X_s / rho of the tile core
    double* Ps = sm + SP_TILE;          // x (+ y) contribution to A
    const int ng = CST_NG;
    const TileCoord tc = tile_coord(g, tg, blockIdx.x);
    const double* Ub = U + (long long)tc.b * g.box_g;
    const double* rinv_b = rinv + (long long)tc.b * g.comp_g;
    const double* fm_tile = Fm + tc.tile * 3LL * (TILE + 1) * NTHR;
    const double* chi_b = FLAT ? chi + (long long)tc.b * g.comp_g : nullptr;
    const int tid = threadIdx.x, ti = tid & (TILE - 1), tr = tid >> 4;   // tr = row group 0..15
    // ghosted index of the tile zone (i = ti, j = tr, k = 0); row n of this thread is k = n
    const long long zt = ((long long)(tc.k0 + ng) * g.ey + (tc.j0 + tr + ng)) * g.ex + (tc.i0 + ti + ng);
    for (int s = 0; s < g.nspec; ++s) {
        const int c = 5 + s;
        const double* Us = Ub + (long long)c * g.comp_g;
        __syncthreads();                                // previous species done with Xs / Ps
        for (int k = 0; k < tc.tz; ++k)
            if (tr < tc.ty && ti < tc.tx) {
                const long long z = zt + k * g.plane_g;
                Xs[(k * TILE + tr) * SP_PITCH + ti] = Us[z] * rinv_b[z];
            }
        __syncthreads();
        species_sweep<0, NR, FLAT>(g, tc, Us, rinv_b, Xs, Ps, fm_tile, A, c, up, chi_b);
        __syncthreads();
        species_sweep<1, NR, FLAT>(g, tc, Us, rinv_b, Xs, Ps, fm_tile, A, c, up, chi_b);
        __syncthreads();
        species_sweep<2, NR, FLAT>(g, tc, Us, rinv_b, Xs, Ps, fm_tile, A, c, up, chi_b);
    }
}

// every tile of every box is a full 16^3 (species_tma.cuh).  `split` consecutive CTAs share one tile, each taking a
// contiguous share of the species: the tiles that are in flight at one time (and with them the Fm / 1/rho working
// set that L2 has to keep) are split x fewer.
template <int NR>
__global__ void __launch_bounds__(NTHR, 2)
k_advect_species_tma(const Geom g, const TileGeom tg, const __grid_constant__ SptMaps maps, const double* __restrict__ U,
                     double* __restrict__ A, const double* __restrict__ rinv, const double* __restrict__ Fm,
                     const UpdArgs up, const int split)
{
    extern __shared__ __align__(128) double sm[];
    const int part = blockIdx.x % split;
    const TileCoord tc = tile_coord(g, tg, blockIdx.x / split);
    const int s_begin = (int)((long long)g.nspec * part / split), s_end = (int)((long long)g.nspec * (part + 1) / split);
    spt_tile<NR>(g, tc, maps, U + (long long)tc.b * g.box_g, rinv + (long long)tc.b * g.comp_g,
                 Fm + tc.tile * 3LL * (TILE + 1) * NTHR, A, up, sm, s_begin, s_end);
}

// the variant kernels (species_tma.cuh spt_tile_v; cst_set_variant / cst_tune_advance): same arithmetic, fewer phases
template <int NR, int V>
__global__ void __launch_bounds__(NTHR, 2)
k_advect_species_tma_v(const Geom g, const TileGeom tg, const __grid_constant__ SptMaps maps, const double* __restrict__ U,
                       double* __restrict__ A, const double* __restrict__ rinv, const double* __restrict__ Fm,
                       const UpdArgs up, const int split)
{
    extern __shared__ __align__(128) double sm[];
    const int part = blockIdx.x % split;
    const TileCoord tc = tile_coord(g, tg, blockIdx.x / split);
    const int s_begin = (int)((long long)g.nspec * part / split), s_end = (int)((long long)g.nspec * (part + 1) / split);
    spt_tile_v<NR, V>(g, tc, maps, U + (long long)tc.b * g.box_g, rinv + (long long)tc.b * g.comp_g,
                      Fm + tc.tile * 3LL * (TILE + 1) * NTHR, A, up, sm, s_begin, s_end);
}

template <int NR>
static int launch_species_nr(cst_ctx* ctx, const double* U, double* A, const UpdArgs& up, cudaStream_t st)
{
    const Geom& g = ctx->g;
    const TileGeom tg = make_tile_geom(g);
    const double* rinv = ctx->ws;
    const double* Fm = ctx->ws + ws_rinv_doubles(g);
    // 16-byte vector accesses and the tensor maps of the fast path need even rows (true for multiples of 16) and aligned bases
    const bool vec_ok = ((((uintptr_t)U | (uintptr_t)A | (uintptr_t)up.U_next | (uintptr_t)up.P[0] |
                           (uintptr_t)up.P[1] | (uintptr_t)up.P[2] | (uintptr_t)rinv) & 15) == 0);
    const bool all_full = vec_ok && (g.nx % TILE == 0) && (g.ny % TILE == 0) && (g.nz % TILE == 0);
    bool tma = all_full && !ctx->flatten;              // flattening runs on the general kernel
    SptMaps maps;
    if (tma) {
        const unsigned long long nbv = (unsigned long long)g.nbox * g.nvar;
        tma = tma_encode_3d_f64(&maps.u, U, g.ex, g.ey, nbv * g.ez, SPT_XW, TILE, TILE) &&
              tma_encode_3d_f64(&maps.r, rinv, g.ex, g.ey, (unsigned long long)g.nbox * g.ez, 24, 22, 22);
        for (int r = 0; r < UPD_MAX_EXT; ++r)
            maps.p[r] = maps.u;                               // unused slots: any valid map
        for (int r = 0; tma && r < NR; ++r)
            tma = tma_encode_3d_f64(&maps.p[r], up.P[r], g.nx, g.ny, nbv * g.nz, TILE, TILE, TILE);
    }
    if (tma) {
        if (cudaFuncSetAttribute(k_advect_species_tma<NR>, cudaFuncAttributeMaxDynamicSharedMemorySize, SPT_SMEM) != cudaSuccess)
            return CST_ECUDA;
        const int want = ctx->species_split > 0 ? ctx->species_split : SPT_SPLIT;
        const int split = g.nspec < want ? g.nspec : want;
        const unsigned grid = (unsigned)(tg.ntiles * split);
        if (ctx->species_variant == 1) {
            if (cudaFuncSetAttribute(k_advect_species_tma_v<NR, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, SPT_SMEM) != cudaSuccess)
                return CST_ECUDA;
            k_advect_species_tma_v<NR, 1><<<grid, NTHR, SPT_SMEM, st>>>(g, tg, maps, U, A, rinv, Fm, up, split);
        } else if (ctx->species_variant == 2) {
            if (cudaFuncSetAttribute(k_advect_species_tma_v<NR, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, SPT_SMEM) != cudaSuccess)
                return CST_ECUDA;
            k_advect_species_tma_v<NR, 2><<<grid, NTHR, SPT_SMEM, st>>>(g, tg, maps, U, A, rinv, Fm, up, split);
        } else if (ctx->species_variant == 3) {
            if (cudaFuncSetAttribute(k_advect_species_tma_v<NR, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, SPT_SMEM) != cudaSuccess)
                return CST_ECUDA;
            k_advect_species_tma_v<NR, 3><<<grid, NTHR, SPT_SMEM, st>>>(g, tg, maps, U, A, rinv, Fm, up, split);
        } else {
            k_advect_species_tma<NR><<<grid, NTHR, SPT_SMEM, st>>>(g, tg, maps, U, A, rinv, Fm, up, split);
        }
    } else {
        const size_t smem = 2ull * SP_TILE * sizeof(double);
        if (ctx->flatten) {
            if (cudaFuncSetAttribute(k_advect_species<NR, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
                return CST_ECUDA;
            k_advect_species<NR, true><<<(unsigned)tg.ntiles, NTHR, smem, st>>>(g, tg, U, A, rinv, Fm, up, Fm + ws_fm_doubles(g));
        } else {
            if (cudaFuncSetAttribute(k_advect_species<NR, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
                return CST_ECUDA;
            k_advect_species<NR, false><<<(unsigned)tg.ntiles, NTHR, smem, st>>>(g, tg, U, A, rinv, Fm, up, nullptr);
        }
    }
    ctx->launches++;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}

int launch_advect_species(cst_ctx* ctx, const double* U, double* A, const UpdArgs& up, cudaStream_t st)
{
    if (ctx->g.nspec == 0) return CST_OK;
    switch (up.nr) {
    case -1: return launch_species_nr<-1>(ctx, U, A, up, st);
    case 0: return launch_species_nr<0>(ctx, U, A, up, st);
    case 1: return launch_species_nr<1>(ctx, U, A, up, st);
    case 2: return launch_species_nr<2>(ctx, U, A, up, st);
    case 3: return launch_species_nr<3>(ctx, U, A, up, st);
    }
    return CST_EINVAL;
}
