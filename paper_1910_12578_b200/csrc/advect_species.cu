// advect_species.cu -- S1-S4 (+ fused S5) for the passively advected components rho X_s of <A(U)>
// (BASELINE north_star "plus passively advected rho*X_k"; Q2, Q8).
//
// F(rho X_s) = F(rho) * X_s(upwind side), so the species need only the face mass fluxes of the hydro
// kernel (workspace Fm) and 1/rho (workspace rinv).  One CTA = one 16^3 tile, same pencil <-> thread
// map as the hydro kernel (tile.cuh).  Per species: X = rho X_s / rho of the tile core is staged in
// shared memory (rho X_s read once from HBM, used by all three sweeps), each thread marches along
// its x, then y, then z pencil with the PPM window (sweep.cuh), multiplies the upwind edge value
// with the face mass flux, and differences consecutive faces.  The three halo zones at either
// pencil end come straight from global memory into the window.  The x and y contributions to A
// wait in a second shared array; the z sweep adds its own and writes A (and, fused, U_next).
//
// Two bodies of the same arithmetic:
//   species_sweep_full  -- the tile is a full 16^3: the march is unrolled at compile time (the
//                          window slides by register renaming, shared-memory offsets are immediates);
//   species_sweep       -- any tile extent (ragged edges of boxes whose sides are not multiples of 16).
// Shared memory: 2 x 16*16*17 + 18*256 doubles = 106.5 KB per CTA, so two CTAs (16 warps) share an SM.
#include "sweep.cuh"
#include "tile.cuh"
#include "species_group.cuh"

#ifndef SPG_G
#define SPG_G 1        // species per pass of the full-tile fast path
#endif
#ifndef SPG_PP
#define SPG_PP 1       // pencils per thread of the full-tile fast path (CTA = 256 / SPG_PP threads)
#endif
#define SPG_NT (NTHR / SPG_PP)
#ifndef SPG_CTAS
#define SPG_CTAS 2     // resident CTAs per SM the fast path is sized for (128 registers per thread)
#endif

#define SP_PITCH 17
#define SP_TILE (TILE * TILE * SP_PITCH)

// ------------------------------------------------------------------------ full 16^3 tiles ----
// Shared memory of the fast path: Xs (core of X), Ps (A under construction), Hs (halo X values,
// [direction][n = 0..5][tid]: n < 3 are pencil positions -3..-1, n >= 3 are 16..18, stored under the
// thread id of the pencil that reads them).  All global->shared traffic of a species happens in
// one streaming phase with many independent loads in flight; the sweeps touch global memory only
// for the face mass fluxes, which are loaded one sweep ahead into registers.
#define SP_HALO (3 * 6 * NTHR)

// L2 residency hints (PTX createpolicy / .L2::cache_hint): the face mass fluxes and 1/rho of a tile are
// read again for each of the nspec species, so they should outlive the once-only streams (A_old
// arrays in, A and U_next out) that pass through the same L2.
__device__ __forceinline__ unsigned long long l2_policy_keep()
{
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ unsigned long long l2_policy_stream()
{
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ double ldg_hint(const double* a, unsigned long long pol)
{
    double v;
    asm volatile("ld.global.nc.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(a), "l"(pol));
    return v;
}
__device__ __forceinline__ double2 ldg2_hint(const double* a, unsigned long long pol)
{
    double2 v;
    asm volatile("ld.global.nc.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(a), "l"(pol));
    return v;
}
__device__ __forceinline__ void stg2_hint(double* a, double2 v, unsigned long long pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1,%2}, %3;" :: "l"(a), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}
__device__ __forceinline__ double2 ldg2(const double* a) { return __ldg(reinterpret_cast<const double2*>(a)); }

__device__ __forceinline__ void load_fm(const double* __restrict__ fm_tile, int D, double fmv[TILE + 1])
{
    const unsigned long long pol = l2_policy_keep();
    const double* __restrict__ fm = fm_tile + (D * (TILE + 1)) * NTHR + threadIdx.x;
#pragma unroll
    for (int f = 0; f <= TILE; ++f) fmv[f] = ldg_hint(fm + f * NTHR, pol);
}

template <int D>
__device__ __forceinline__ void species_sweep_full(const Geom& g, const double* __restrict__ Xs,
                                                   double* __restrict__ Ps, const double* __restrict__ Hs,
                                                   const double fmv[TILE + 1])
{
    const int tid = threadIdx.x, a = tid & (TILE - 1), b = tid >> 4;
    constexpr int L = TILE;
    constexpr int SST = (D == 0) ? 1 : (D == 1) ? SP_PITCH : TILE * SP_PITCH;   // smem stride along the pencil
    const int s0 = (D == 0) ? (b * TILE + a) * SP_PITCH : (D == 1) ? (b * TILE) * SP_PITCH + a : b * SP_PITCH + a;
    const double nrd = -((D == 0) ? g.rdx : (D == 1) ? g.rdy : g.rdz);
    const double* __restrict__ xs = Xs + s0;
    double* __restrict__ ps = Ps + s0;
    const double* __restrict__ hs = Hs + D * 6 * NTHR + tid;

    PpmWindow w;
    w.start(hs[0]); w.warm1(hs[NTHR]); w.warm2(hs[2 * NTHR]);
    w.warm3(xs[0]);
    double Fprev = 0.0;
#pragma unroll
    for (int p = 1; p <= L + 2; ++p) {
        const double qn = (p < L) ? xs[p * SST] : hs[(3 + p - L) * NTHR];
        w.push(qn);
        if (p >= 2) {
            const double fmc = fmv[p - 2];              // mass flux of face f = p-2
            const double F = fmc * (sign_bit(fmc) ? w.qm : w.qpL);
            if (p >= 3) {
                const int q = p - 3;
                const double dF = F - Fprev;
                if (D == 0) ps[q * SST] = dF * nrd;
                else ps[q * SST] = fma(dF, nrd, ps[q * SST]);
            }
            Fprev = F;
        }
    }
}

// streaming phase: write out species c_out (A and, fused, U_next) from Ps, stage species c_in into
// Xs / Hs.  Rows of the tile are handled as 8 x 16-byte pieces: thread t takes piece cp = t % 8 of rows
// t / 8 + 32 n (row = 16 k + j), so every global access is a full 16-byte vector.
template <int NR>
__device__ __forceinline__ void species_stream_full(const Geom& g, const TileCoord& tc,
                                                    const double* __restrict__ Ub, const double* __restrict__ rinv_b,
                                                    double* __restrict__ Xs, const double* __restrict__ Ps,
                                                    double* __restrict__ Hs, double* __restrict__ A,
                                                    const UpdArgs& up, const int c_out, const int c_in)
{
    const int ng = CST_NG;
    const int tid = threadIdx.x, cp = tid & 7, r0 = tid >> 3;
    const unsigned long long keep = l2_policy_keep(), strm = l2_policy_stream();
    // ghosted index (within a component) of tile zone (0, 0, 0)
    const long long zt = ((long long)(tc.k0 + ng) * g.ey + (tc.j0 + ng)) * g.ex + (tc.i0 + ng);
    if (c_in >= 0) {
        const double* __restrict__ Us = Ub + (long long)c_in * g.comp_g;
        // core
#pragma unroll
        for (int n = 0; n < 8; ++n) {
            const int row = r0 + 32 * n, k = row >> 4, j = row & 15;
            const long long z = zt + k * g.plane_g + (long long)j * g.ex + 2 * cp;
            const double2 u = ldg2(Us + z), ri = ldg2_hint(rinv_b + z, keep);
            double* x = Xs + row * SP_PITCH + 2 * cp;
            x[0] = u.x * ri.x; x[1] = u.y * ri.y;
        }
        // y halos (consumer thread = 16 k + i) and z halos (consumer thread = 16 j + i): 768 pieces each
#pragma unroll
        for (int m = 0; m < 3; ++m) {
            const int idx = tid + NTHR * m, hp = idx & 7, q = (idx >> 3) & 15, n = idx >> 7;
            const int off = n < 3 ? n - 3 : TILE - 3 + n;
            const long long zy = zt + q * g.plane_g + (long long)off * g.ex + 2 * hp;
            const long long zz = zt + off * g.plane_g + (long long)q * g.ex + 2 * hp;
            const double2 uy = ldg2(Us + zy), ry = ldg2_hint(rinv_b + zy, keep);
            const double2 uz = ldg2(Us + zz), rz = ldg2_hint(rinv_b + zz, keep);
            *reinterpret_cast<double2*>(Hs + (6 + n) * NTHR + q * TILE + 2 * hp) = make_double2(uy.x * ry.x, uy.y * ry.y);
            *reinterpret_cast<double2*>(Hs + (12 + n) * NTHR + q * TILE + 2 * hp) = make_double2(uz.x * rz.x, uz.y * rz.y);
        }
        // x halos of this thread's own x pencil (j = tid % 16, k = tid / 16): positions -3 | -2 -1 and 16 17 | 18
        {
            const long long zx = zt + (tid >> 4) * g.plane_g + (long long)(tid & 15) * g.ex;
            const double ul = Us[zx - 3], rl = ldg_hint(rinv_b + zx - 3, keep);
            const double2 ul2 = ldg2(Us + zx - 2), rl2 = ldg2_hint(rinv_b + zx - 2, keep);
            const double2 uh2 = ldg2(Us + zx + TILE), rh2 = ldg2_hint(rinv_b + zx + TILE, keep);
            const double uh = Us[zx + TILE + 2], rh = ldg_hint(rinv_b + zx + TILE + 2, keep);
            Hs[0 * NTHR + tid] = ul * rl; Hs[1 * NTHR + tid] = ul2.x * rl2.x; Hs[2 * NTHR + tid] = ul2.y * rl2.y;
            Hs[3 * NTHR + tid] = uh2.x * rh2.x; Hs[4 * NTHR + tid] = uh2.y * rh2.y; Hs[5 * NTHR + tid] = uh * rh;
        }
    }
    if (c_out >= 0) {
        const long long ia0 = (long long)tc.b * g.box_a + (long long)c_out * g.comp_a +
            ((long long)tc.k0 * g.ny + tc.j0) * g.nx + tc.i0 + 2 * cp;
        const long long iu0 = (long long)tc.b * g.box_g + (long long)c_out * g.comp_g + zt + 2 * cp;
        // batches of four rows: every load of a batch is issued before its first store (the
        // compiler may not move loads over stores that could alias them)
#pragma unroll
        for (int n0 = 0; n0 < 8; n0 += 4) {
            double2 av[4], um[4], pv[4][UPD_MAX_EXT];
            long long ia[4], iu[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int row = r0 + 32 * (n0 + e), k = row >> 4, j = row & 15;
                ia[e] = ia0 + ((long long)k * g.ny + j) * g.nx;
                iu[e] = iu0 + k * g.plane_g + (long long)j * g.ex;
                const double* x = Ps + row * SP_PITCH + 2 * cp;
                av[e] = make_double2(x[0], x[1]);
                if (NR >= 0) {
                    um[e] = ldg2(up.U_m + iu[e]);
#pragma unroll
                    for (int r = 0; r < NR; ++r) pv[e][r] = ldg2_hint(up.P[r] + ia[e], strm);
                }
            }
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                if (NR >= 0) {
                    double2 acc = make_double2(fma(up.ca, av[e].x, um[e].x), fma(up.ca, av[e].y, um[e].y));
#pragma unroll
                    for (int r = 0; r < NR; ++r) {
                        acc.x = fma(up.c[r], pv[e][r].x, acc.x); acc.y = fma(up.c[r], pv[e][r].y, acc.y);
                    }
                    stg2_hint(up.U_next + iu[e], acc, strm);
                }
                stg2_hint(A + ia[e], av[e], strm);
            }
        }
    }
}

template <int NR>
__device__ __forceinline__ void species_tile_full(const Geom& g, const TileCoord& tc, const double* __restrict__ Ub,
                                                  const double* __restrict__ rinv_b,
                                                  const double* __restrict__ fm_tile, double* __restrict__ A,
                                                  const UpdArgs& up, double* __restrict__ sm)
{
    double* Xs = sm;
    double* Ps = sm + SP_TILE;
    double* Hs = sm + 2 * SP_TILE;
    double fmc[TILE + 1], fmn[TILE + 1];
    load_fm(fm_tile, 0, fmc);
    for (int s = 0; s <= g.nspec; ++s) {
        __syncthreads();                                // z sweep of species s-1 done; Xs, Hs free
        species_stream_full<NR>(g, tc, Ub, rinv_b, Xs, Ps, Hs, A, up,
                                s > 0 ? 5 + s - 1 : -1, s < g.nspec ? 5 + s : -1);
        if (s == g.nspec) break;
        __syncthreads();
        load_fm(fm_tile, 1, fmn);
        species_sweep_full<0>(g, Xs, Ps, Hs, fmc);
        __syncthreads();
        load_fm(fm_tile, 2, fmc);
        species_sweep_full<1>(g, Xs, Ps, Hs, fmn);
        __syncthreads();
        load_fm(fm_tile, 0, fmn);
        species_sweep_full<2>(g, Xs, Ps, Hs, fmc);
#pragma unroll
        for (int f = 0; f <= TILE; ++f) fmc[f] = fmn[f];
    }
}

// --------------------------------------------------------------------------- any tile extent ----
template <int D, int NR>
__device__ __forceinline__ void species_sweep(const Geom& g, const TileCoord& tc, const double* __restrict__ Us,
                                              const double* __restrict__ rinv_b,
                                              const double* __restrict__ Xs, double* __restrict__ Ps,
                                              const double* __restrict__ fm_tile,
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
        w.push(qn);
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

template <int NR>
__global__ void __launch_bounds__(NTHR, 2)
k_advect_species(Geom g, TileGeom tg, const double* __restrict__ U, double* __restrict__ A,
                 const double* __restrict__ rinv, const double* __restrict__ Fm, UpdArgs up)
{
    extern __shared__ double sm[];
    double* Xs = sm;                    // X_s = rho X_s / rho of the tile core
    double* Ps = sm + SP_TILE;          // x (+ y) contribution to A
    const int ng = CST_NG;
    const TileCoord tc = tile_coord(g, tg, blockIdx.x);
    const double* Ub = U + (long long)tc.b * g.box_g;
    const double* rinv_b = rinv + (long long)tc.b * g.comp_g;
    const double* fm_tile = Fm + tc.tile * 3LL * (TILE + 1) * NTHR;
    const int tid = threadIdx.x, ti = tid & (TILE - 1), tr = tid >> 4;   // tr = row group 0..15
    if ((tc.tx == TILE) && (tc.ty == TILE) && (tc.tz == TILE)) {
        species_tile_full<NR>(g, tc, Ub, rinv_b, fm_tile, A, up, sm);
        return;
    }
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
        species_sweep<0, NR>(g, tc, Us, rinv_b, Xs, Ps, fm_tile, A, c, up);
        __syncthreads();
        species_sweep<1, NR>(g, tc, Us, rinv_b, Xs, Ps, fm_tile, A, c, up);
        __syncthreads();
        species_sweep<2, NR>(g, tc, Us, rinv_b, Xs, Ps, fm_tile, A, c, up);
    }
}

// every tile of every box is a full 16^3: CTAs of SPG_NT threads, SPG_PP pencils per thread (species_group.cuh)
template <int NR>
__global__ void __launch_bounds__(SPG_NT, SPG_CTAS)
k_advect_species_full(Geom g, TileGeom tg, const double* __restrict__ U, double* __restrict__ A,
                      const double* __restrict__ rinv, const double* __restrict__ Fm, UpdArgs up)
{
    extern __shared__ double sm[];
    const TileCoord tc = tile_coord(g, tg, blockIdx.x);
    spg_tile<SPG_G, SPG_PP, NR>(g, tc, U + (long long)tc.b * g.box_g, rinv + (long long)tc.b * g.comp_g,
                                Fm + tc.tile * 3LL * (TILE + 1) * NTHR, A, up, sm);
}

template <int NR>
static int launch_species_nr(cst_ctx* ctx, const double* U, double* A, const UpdArgs& up, cudaStream_t st)
{
    const Geom& g = ctx->g;
    const TileGeom tg = make_tile_geom(g);
    const double* rinv = ctx->ws;
    const double* Fm = ctx->ws + ws_rinv_doubles(g);
    static bool attr_set = false;
    const size_t smem_full = 2ull * SPG_G * SPG_TILE * sizeof(double);
    const size_t smem = (2ull * SP_TILE + SP_HALO) * sizeof(double);
    if (!attr_set) {
        if (cudaFuncSetAttribute(k_advect_species<NR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
            cudaFuncSetAttribute(k_advect_species_full<NR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_full) != cudaSuccess)
            return CST_ECUDA;
        attr_set = true;
    }
    // 16-byte vector accesses of the fast path need even row lengths (true for multiples of 16) and aligned bases
    const bool all_full = (g.nx % TILE == 0) && (g.ny % TILE == 0) && (g.nz % TILE == 0) &&
                          ((((uintptr_t)U | (uintptr_t)A | (uintptr_t)up.U_next | (uintptr_t)up.P[0] |
                             (uintptr_t)up.P[1] | (uintptr_t)up.P[2]) & 15) == 0);
    if (all_full)
        k_advect_species_full<NR><<<(unsigned)tg.ntiles, SPG_NT, smem_full, st>>>(g, tg, U, A, rinv, Fm, up);
    else
        k_advect_species<NR><<<(unsigned)tg.ntiles, NTHR, smem, st>>>(g, tg, U, A, rinv, Fm, up);
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
