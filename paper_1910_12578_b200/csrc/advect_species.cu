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
// Shared memory: 2 x 16*16*17 doubles = 69.6 KB per CTA, so three CTAs (24 warps) share an SM.
#include "sweep.cuh"
#include "tile.cuh"

#define SP_PITCH 17
#define SP_TILE (TILE * TILE * SP_PITCH)

// ------------------------------------------------------------------------ full 16^3 tiles ----
template <int D, int NR>
__device__ __forceinline__ void species_sweep_full(const Geom& g, const TileCoord& tc, const double* __restrict__ Us,
                                                   const double* __restrict__ rinv_b,
                                                   const double* __restrict__ Xs, double* __restrict__ Ps,
                                                   const double* __restrict__ fm_tile,
                                                   double* __restrict__ A, int c, const UpdArgs& up)
{
    const int ng = CST_NG;
    const int tid = threadIdx.x, a = tid & (TILE - 1), b = tid >> 4;
    constexpr int L = TILE;
    constexpr int SST = (D == 0) ? 1 : (D == 1) ? SP_PITCH : TILE * SP_PITCH;   // smem stride along the pencil
    long long z0, stride;
    int s0;
    if (D == 0) {
        z0 = ((long long)(tc.k0 + b + ng) * g.ey + (tc.j0 + a + ng)) * g.ex + (tc.i0 + ng);
        stride = 1; s0 = (b * TILE + a) * SP_PITCH;
    } else if (D == 1) {
        z0 = ((long long)(tc.k0 + b + ng) * g.ey + (tc.j0 + ng)) * g.ex + (tc.i0 + a + ng);
        stride = g.ex; s0 = (b * TILE) * SP_PITCH + a;
    } else {
        z0 = ((long long)(tc.k0 + ng) * g.ey + (tc.j0 + b + ng)) * g.ex + (tc.i0 + a + ng);
        stride = g.plane_g; s0 = b * SP_PITCH + a;
    }
    const double nrd = -((D == 0) ? g.rdx : (D == 1) ? g.rdy : g.rdz);
    const double* __restrict__ fm = fm_tile + (D * (TILE + 1)) * NTHR + tid;
    const double* __restrict__ xs = Xs + s0;
    double* __restrict__ ps = Ps + s0;

    // halo zones p = -3..-1 and L..L+2 from global memory
    double hlo[3], hhi[3];
#pragma unroll
    for (int n = 0; n < 3; ++n) {
        const long long zl = z0 + (long long)(n - 3) * stride, zh = z0 + (long long)(L + n) * stride;
        hlo[n] = Us[zl] * rinv_b[zl];
        hhi[n] = Us[zh] * rinv_b[zh];
    }
    // face mass fluxes of the pencil (thread-private slots, coalesced)
    double fmv[L + 1];
#pragma unroll
    for (int f = 0; f <= L; ++f) fmv[f] = fm[f * NTHR];

    PpmWindow w;
    w.start(hlo[0]); w.warm1(hlo[1]); w.warm2(hlo[2]);
    w.warm3(xs[0]);
    double Fprev = 0.0;
    // output addressing of the z sweep (D == 2): running pointers to zone q of the pencil
    const long long ia0 = (long long)tc.b * g.box_a + (long long)c * g.comp_a +
        ((long long)tc.k0 * g.ny + (tc.j0 + b)) * g.nx + (tc.i0 + a);
    const long long plane_a = (long long)g.ny * g.nx;
    const long long iu0 = (long long)tc.b * g.box_g + (long long)c * g.comp_g + z0;
    double* pA = A + ia0;
    const double* pU = up.U_m + iu0;
    double* pUn = up.U_next + iu0;
    const double* pP[UPD_MAX_EXT];
#pragma unroll
    for (int r = 0; r < UPD_MAX_EXT; ++r) pP[r] = (r < NR) ? up.P[r] + ia0 : nullptr;
#pragma unroll
    for (int p = 1; p <= L + 2; ++p) {
        const double qn = (p < L) ? xs[p * SST] : hhi[p - L];
        w.push(qn);
        if (p >= 2) {
            const double fmc = fmv[p - 2];              // mass flux of face f = p-2
            const double F = fmc * (sign_bit(fmc) ? w.qm : w.qpL);
            if (p >= 3) {
                const int q = p - 3;
                const double dF = F - Fprev;
                if (D == 0) ps[q * SST] = dF * nrd;
                else if (D == 1) ps[q * SST] = fma(dF, nrd, ps[q * SST]);
                else {
                    const double av = fma(dF, nrd, ps[q * SST]);
                    if (NR >= 0) {
                        double acc = fma(up.ca, av, *pU);
#pragma unroll
                        for (int r = 0; r < NR; ++r) { acc = fma(up.c[r], *pP[r], acc); pP[r] += plane_a; }
                        *pUn = acc;
                        pU += stride; pUn += stride;
                    }
                    *pA = av;
                    pA += plane_a;
                }
            }
            Fprev = F;
        }
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
__global__ void __launch_bounds__(NTHR, 3)
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
    const bool full = (tc.tx == TILE) && (tc.ty == TILE) && (tc.tz == TILE);

    // ghosted index of the tile zone (i = ti, j = tr, k = 0); row n of this thread is k = n
    const long long zt = ((long long)(tc.k0 + ng) * g.ey + (tc.j0 + tr + ng)) * g.ex + (tc.i0 + ti + ng);
    for (int s = 0; s < g.nspec; ++s) {
        const int c = 5 + s;
        const double* Us = Ub + (long long)c * g.comp_g;
        __syncthreads();                                // previous species done with Xs / Ps
        if (full) {
#pragma unroll
            for (int k = 0; k < TILE; ++k) {
                const long long z = zt + k * g.plane_g;
                Xs[(k * TILE + tr) * SP_PITCH + ti] = Us[z] * rinv_b[z];
            }
        } else {
            for (int k = 0; k < tc.tz; ++k)
                if (tr < tc.ty && ti < tc.tx) {
                    const long long z = zt + k * g.plane_g;
                    Xs[(k * TILE + tr) * SP_PITCH + ti] = Us[z] * rinv_b[z];
                }
        }
        __syncthreads();
        if (full) {
            species_sweep_full<0, NR>(g, tc, Us, rinv_b, Xs, Ps, fm_tile, A, c, up);
            __syncthreads();
            species_sweep_full<1, NR>(g, tc, Us, rinv_b, Xs, Ps, fm_tile, A, c, up);
            __syncthreads();
            species_sweep_full<2, NR>(g, tc, Us, rinv_b, Xs, Ps, fm_tile, A, c, up);
        } else {
            species_sweep<0, NR>(g, tc, Us, rinv_b, Xs, Ps, fm_tile, A, c, up);
            __syncthreads();
            species_sweep<1, NR>(g, tc, Us, rinv_b, Xs, Ps, fm_tile, A, c, up);
            __syncthreads();
            species_sweep<2, NR>(g, tc, Us, rinv_b, Xs, Ps, fm_tile, A, c, up);
        }
    }
}

template <int NR>
static int launch_species_nr(cst_ctx* ctx, const double* U, double* A, const UpdArgs& up, cudaStream_t st)
{
    const Geom& g = ctx->g;
    const TileGeom tg = make_tile_geom(g);
    const size_t smem = 2ull * SP_TILE * sizeof(double);
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(k_advect_species<NR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return CST_ECUDA;
        attr_set = true;
    }
    const double* rinv = ctx->ws;
    const double* Fm = ctx->ws + ws_rinv_doubles(g);
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
