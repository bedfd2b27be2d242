// advect_hydro.cu -- S1-S4 (+ fused S5) for the five hydrodynamic components (rho, rho u, rho v,
// rho w, rho E) of <A(U)> (include/cst.h cst_advance_A).
//
// One CTA = one 16^3 tile (tile.cuh).  Three sweeps, x then y then z.  In each sweep a thread marches
// along its pencil: it loads the conserved state of the next zone, converts it to primitives
// (S1), slides five PPM windows (S2, sweep.cuh), solves the HLLC problem at the face that has
// just become complete (S3) and differences consecutive face fluxes (S4).  Every face flux and
// every parabola of the tile is therefore computed once.  The x and y contributions to A are
// accumulated in shared memory (5 x 16^3 doubles); the z sweep adds its own, the gravity source and
// writes A (and, fused, the SDC node update S5).
// Side products for the species kernel: 1/rho of every zone the species stencil touches (workspace
// rinv) and the mass flux F(rho) of every face (workspace Fm, thread-private slots, tile.cuh).
//
// Two bodies of the same arithmetic: hydro_sweep_full (full 16^3 tile: march unrolled at compile
// time, the x sweep reads 32-byte groups of four zones so that every fetched sector is used) and
// hydro_sweep (any tile extent).
#include "sweep.cuh"
#include "tile.cuh"

#define PART_PITCH 17                                  // odd pitch: conflict-free for every sweep
#define PART_COMP (TILE * TILE * PART_PITCH)           // doubles per component

// ------------------------------------------------------------------------ full 16^3 tiles ----
// The march is a short loop (x: 6 groups of 4 zones, y/z: 11 pairs of zones) so that its body stays
// in the instruction cache.  Every zone runs the SAME window step (PpmWindow::push) from the first
// halo zone on: a window that starts from zeros holds garbage for three steps, but the first
// quantities that are used (the parabola of zone -1, from p = 1) depend only on real zone values
// (sweep.cuh), so no warm-up variants of the step are needed.
__device__ __forceinline__ void ldg256(const double* p, double v[4])
{   // one 32-byte sector per thread (p is 32-byte aligned)
    asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];"
                 : "=d"(v[0]), "=d"(v[1]), "=d"(v[2]), "=d"(v[3]) : "l"(p));
}

__device__ __forceinline__ double ldg_now(const double* p)
{   // a load the compiler may not sink to its first use: issued here, consumed much later
    double v;
    asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(v) : "l"(p));
    return v;
}

struct HydroMarch {           // per-thread state of one pencil march
    PpmWindow w[5];
    double Fprev[5];
    double* fm_slot;          // Fm slot of the face that completes next
    double* part;             // shared-memory partial of the zone that completes next (component 0)
    double* pA;               // z sweep: A of the zone that completes next (component 0)
    long long zc;             // z sweep: ghosted index (within the box) of that zone
    double cfl;               // CFL = true: running max of the signal rate of the interior zones (S6)
};

template <int D, int NR, bool CFL = false>
__device__ __forceinline__ void hydro_zone(const Geom& g, const TileCoord& tc, HydroMarch& m, const int p,
                                           const double Uc[5], const double* __restrict__ Ub,
                                           double* __restrict__ rinv_b, const UpdArgs& up,
                                           const long long z0, const long long stride, const bool ghost_lo,
                                           const bool ghost_hi)
{
    constexpr int L = TILE;
    constexpr int PST = (D == 0) ? 1 : (D == 1) ? PART_PITCH : TILE * PART_PITCH;
    const double nrd = -((D == 0) ? g.rdx : (D == 1) ? g.rdy : g.rdz);
    // z sweep: operands of the source term and of the fused node update of the zone that completes in
    // this step are requested first, so that their latency hides behind the arithmetic below
    const bool grav = (g.grav[0] != 0.0) || (g.grav[1] != 0.0) || (g.grav[2] != 0.0);
    double Um[5], Pv[5][UPD_MAX_EXT];
    long long ia0 = 0;
    if (D == 2 && p >= 3) {
        ia0 = m.pA - up.A_base;                          // index of component 0 in the A-like arrays
        if (grav || NR >= 0) {
#pragma unroll
            for (int c = 0; c < 5; ++c) Um[c] = ldg_now(Ub + c * g.comp_g + m.zc);
        }
#pragma unroll
        for (int c = 0; c < 5; ++c)
#pragma unroll
            for (int r = 0; r < NR; ++r) Pv[c][r] = ldg_now(up.P[r] + ia0 + c * g.comp_a);
    }
    double W[5];
    const double r = cons_to_prim(g, Uc[0], Uc[1], Uc[2], Uc[3], Uc[4], W);
    if ((D == 2 && p >= 0 && p < L) || (p < 0 && ghost_lo) || (p >= L && ghost_hi))
        rinv_b[z0 + (long long)p * stride] = r;
    if (CFL && D == 2 && p >= 0 && p < L) {             // S6 folded into the z sweep: the primitives of the zone are at hand
        const double cs = sqrt_fast(g.gamma * W[4] * r);
        const double rate = (fabs(W[1]) + cs) * g.rdx + (fabs(W[2]) + cs) * g.rdy + (fabs(W[3]) + cs) * g.rdz;
        m.cfl = dmax(m.cfl, rate);
    }
#pragma unroll
    for (int c = 0; c < 5; ++c) m.w[c].push(W[c]);
    if (p >= 2) {
        // face f = p-2 between zones p-3 and p-2
        double WL[5], WR[5], F[5];
#pragma unroll
        for (int c = 0; c < 5; ++c) { WL[c] = m.w[c].qpL; WR[c] = m.w[c].qm; }
        WL[0] = dmax(WL[0], g.small_dens); WR[0] = dmax(WR[0], g.small_dens);
        WL[4] = dmax(WL[4], g.small_pres); WR[4] = dmax(WR[4], g.small_pres);
        hllc<D>(g, WL, WR, F);
        *m.fm_slot = F[0];
        m.fm_slot += NTHR;
        if (p >= 3) {                                    // zone q = p-3 of the pencil is complete
            if (D == 0) {
#pragma unroll
                for (int c = 0; c < 5; ++c) m.part[c * PART_COMP] = (F[c] - m.Fprev[c]) * nrd;
            } else if (D == 1) {
#pragma unroll
                for (int c = 0; c < 5; ++c)
                    m.part[c * PART_COMP] = fma(F[c] - m.Fprev[c], nrd, m.part[c * PART_COMP]);
            } else {
                double A5[5];
#pragma unroll
                for (int c = 0; c < 5; ++c) A5[c] = fma(F[c] - m.Fprev[c], nrd, m.part[c * PART_COMP]);
                if (grav) {     // S4 source: constant gravity from the zone-centre state
                    A5[1] = fma(Um[0], g.grav[0], A5[1]);
                    A5[2] = fma(Um[0], g.grav[1], A5[2]);
                    A5[3] = fma(Um[0], g.grav[2], A5[3]);
                    A5[4] += fma(Um[3], g.grav[2], fma(Um[2], g.grav[1], Um[1] * g.grav[0]));
                }
#pragma unroll
                for (int c = 0; c < 5; ++c) {
                    if (NR >= 0) {
                        double acc = fma(up.ca, A5[c], Um[c]);
#pragma unroll
                        for (int r = 0; r < NR; ++r) acc = fma(up.c[r], Pv[c][r], acc);
                        up.U_next[(long long)tc.b * g.box_g + c * g.comp_g + m.zc] = acc;
                    }
                    m.pA[c * g.comp_a] = A5[c];
                }
                m.pA += (long long)g.ny * g.nx;
                m.zc += stride;
            }
            m.part += PST;
        }
#pragma unroll
        for (int c = 0; c < 5; ++c) m.Fprev[c] = F[c];
    }
}

template <int D, int NR, bool CFL = false>
__device__ __forceinline__ double hydro_sweep_full(const Geom& g, const TileCoord& tc, const double* __restrict__ Ub,
                                                   double* __restrict__ part, double* __restrict__ fm_tile,
                                                   double* __restrict__ rinv_b, double* __restrict__ A,
                                                   const UpdArgs& up)
{
    const int ng = CST_NG;
    constexpr int L = TILE;
    const int tid = threadIdx.x, a = tid & (TILE - 1), b = tid >> 4;
    long long z0, stride;
    int n_d, o_d, sp0;
    if (D == 0) {
        z0 = ((long long)(tc.k0 + b + ng) * g.ey + (tc.j0 + a + ng)) * g.ex + (tc.i0 + ng);
        stride = 1; n_d = g.nx; o_d = tc.i0; sp0 = (b * TILE + a) * PART_PITCH;
    } else if (D == 1) {
        z0 = ((long long)(tc.k0 + b + ng) * g.ey + (tc.j0 + ng)) * g.ex + (tc.i0 + a + ng);
        stride = g.ex; n_d = g.ny; o_d = tc.j0; sp0 = (b * TILE) * PART_PITCH + a;
    } else {
        z0 = ((long long)(tc.k0 + ng) * g.ey + (tc.j0 + b + ng)) * g.ex + (tc.i0 + a + ng);
        stride = g.plane_g; n_d = g.nz; o_d = tc.k0; sp0 = b * PART_PITCH + a;
    }
    const bool ghost_lo = (o_d == 0), ghost_hi = (o_d + L == n_d);
    HydroMarch m;
#pragma unroll
    for (int c = 0; c < 5; ++c) {
        m.w[c].q1 = m.w[c].q2 = m.w[c].dq1 = m.w[c].s2 = m.w[c].e = m.w[c].qp = 0.0;
        m.Fprev[c] = 0.0;
    }
    m.cfl = 0.0;
    m.fm_slot = fm_tile + (D * (TILE + 1)) * NTHR + tid;
    m.part = part + sp0;
    m.pA = A + (long long)tc.b * g.box_a + ((long long)tc.k0 * g.ny + (tc.j0 + b)) * g.nx + (tc.i0 + a);
    m.zc = z0;

    if (D == 0) {
        // groups of four zones p = 4G .. 4G+3, G = -1 .. 4; zones p = -4 and p = 19 are not used
        double cur[5][4], nxt[5][4];
#pragma unroll
        for (int c = 0; c < 5; ++c) ldg256(Ub + c * g.comp_g + z0 - 4, cur[c]);
#pragma unroll 1
        for (int G = -1; G <= 4; ++G) {
            if (G < 4) {
#pragma unroll
                for (int c = 0; c < 5; ++c) ldg256(Ub + c * g.comp_g + z0 + 4 * (G + 1), nxt[c]);
            }
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                const int p = 4 * G + e;
                if ((e == 0 && G == -1) || (e == 3 && G == 4)) continue;
                const double Uc[5] = { cur[0][e], cur[1][e], cur[2][e], cur[3][e], cur[4][e] };
                hydro_zone<D, NR, CFL>(g, tc, m, p, Uc, Ub, rinv_b, up, z0, stride, ghost_lo, ghost_hi);
            }
#pragma unroll
            for (int c = 0; c < 5; ++c)
#pragma unroll
                for (int e = 0; e < 4; ++e) cur[c][e] = nxt[c][e];
        }
    } else {
        // pairs of zones p = -3 + 2n, -2 + 2n, n = 0 .. 10, loaded one pair ahead
        double cur[5][2], nxt[5][2];
#pragma unroll
        for (int c = 0; c < 5; ++c)
#pragma unroll
            for (int e = 0; e < 2; ++e) cur[c][e] = Ub[c * g.comp_g + z0 + (e - 3) * stride];
#pragma unroll 1
        for (int n = 0; n <= 10; ++n) {
            const int p0 = 2 * n - 3;
            if (n < 10) {
#pragma unroll
                for (int c = 0; c < 5; ++c)
#pragma unroll
                    for (int e = 0; e < 2; ++e) nxt[c][e] = Ub[c * g.comp_g + z0 + (long long)(p0 + 2 + e) * stride];
            }
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const double Uc[5] = { cur[0][e], cur[1][e], cur[2][e], cur[3][e], cur[4][e] };
                hydro_zone<D, NR, CFL>(g, tc, m, p0 + e, Uc, Ub, rinv_b, up, z0, stride, ghost_lo, ghost_hi);
            }
#pragma unroll
            for (int c = 0; c < 5; ++c)
#pragma unroll
                for (int e = 0; e < 2; ++e) cur[c][e] = nxt[c][e];
        }
    }
    return m.cfl;
}

// --------------------------------------------------------------------------- any tile extent ----
template <int D, int NR, bool FLAT>
__device__ __forceinline__ void hydro_sweep(const Geom& g, const TileCoord& tc, const double* __restrict__ Ub,
                                            double* __restrict__ part, double* __restrict__ fm_tile,
                                            double* __restrict__ rinv_b, double* __restrict__ A,
                                            const UpdArgs& up, const double* __restrict__ chi_b)
{
    const int ng = CST_NG;
    const int tid = threadIdx.x, a = tid & (TILE - 1), b = tid >> 4;
    int L, ea, eb;
    if (D == 0) { L = tc.tx; ea = tc.ty; eb = tc.tz; }
    else if (D == 1) { L = tc.ty; ea = tc.tx; eb = tc.tz; }
    else { L = tc.tz; ea = tc.tx; eb = tc.ty; }
    if (a >= ea || b >= eb) return;

    // ghosted linear index of pencil position p = 0 and the stride along the pencil
    long long z0, stride;
    int n_d, o_d;
    if (D == 0) {
        z0 = ((long long)(tc.k0 + b + ng) * g.ey + (tc.j0 + a + ng)) * g.ex + (tc.i0 + ng);
        stride = 1; n_d = g.nx; o_d = tc.i0;
    } else if (D == 1) {
        z0 = ((long long)(tc.k0 + b + ng) * g.ey + (tc.j0 + ng)) * g.ex + (tc.i0 + a + ng);
        stride = g.ex; n_d = g.ny; o_d = tc.j0;
    } else {
        z0 = ((long long)(tc.k0 + ng) * g.ey + (tc.j0 + b + ng)) * g.ex + (tc.i0 + a + ng);
        stride = g.plane_g; n_d = g.nz; o_d = tc.k0;
    }
    const bool ghost_lo = (o_d == 0), ghost_hi = (o_d + L == n_d);
    const double rd = (D == 0) ? g.rdx : (D == 1) ? g.rdy : g.rdz;

    PpmWindow w[5];
    double Uc[5], Fprev[5];
#pragma unroll
    for (int c = 0; c < 5; ++c) Uc[c] = Ub[c * g.comp_g + z0 - 3 * stride];

    for (int p = -3; p <= L + 2; ++p) {
        // prefetch the next zone of the pencil while this one is processed
        double Un[5];
        if (p < L + 2) {
            const long long zn = z0 + (long long)(p + 1) * stride;
#pragma unroll
            for (int c = 0; c < 5; ++c) Un[c] = Ub[c * g.comp_g + zn];
        }
        double W[5];
        const double r = cons_to_prim(g, Uc[0], Uc[1], Uc[2], Uc[3], Uc[4], W);
        if ((D == 2 && p >= 0 && p < L) || (p < 0 && ghost_lo) || (p >= L && ghost_hi))
            rinv_b[z0 + (long long)p * stride] = r;

        if (p == -3) {
#pragma unroll
            for (int c = 0; c < 5; ++c) w[c].start(W[c]);
        } else if (p == -2) {
#pragma unroll
            for (int c = 0; c < 5; ++c) w[c].warm1(W[c]);
        } else if (p == -1) {
#pragma unroll
            for (int c = 0; c < 5; ++c) w[c].warm2(W[c]);
        } else if (p == 0) {
#pragma unroll
            for (int c = 0; c < 5; ++c) w[c].warm3(W[c]);
        } else {
            if (FLAT) {                                  // optional CW84 flattening of the parabola of zone p-2
                const double x = chi_b[z0 + (long long)(p - 2) * stride];
#pragma unroll
                for (int c = 0; c < 5; ++c) w[c].push_flat(W[c], x);
            } else {
#pragma unroll
                for (int c = 0; c < 5; ++c) w[c].push(W[c]);
            }
            if (p >= 2) {
                // face f = p-2 between zones p-3 and p-2
                double WL[5], WR[5], F[5];
#pragma unroll
                for (int c = 0; c < 5; ++c) { WL[c] = w[c].qpL; WR[c] = w[c].qm; }
                WL[0] = fmax(WL[0], g.small_dens); WR[0] = fmax(WR[0], g.small_dens);
                WL[4] = fmax(WL[4], g.small_pres); WR[4] = fmax(WR[4], g.small_pres);
                hllc<D>(g, WL, WR, F);
                fm_tile[((D * (TILE + 1)) + (p - 2)) * NTHR + tid] = F[0];
                if (p >= 3) {
                    const int q = p - 3;                     // zone of the pencil that is now complete
                    int li, lj, lk;
                    if (D == 0) { li = q; lj = a; lk = b; }
                    else if (D == 1) { li = a; lj = q; lk = b; }
                    else { li = a; lj = b; lk = q; }
                    const int sp = (lk * TILE + lj) * PART_PITCH + li;
                    if (D == 0) {
#pragma unroll
                        for (int c = 0; c < 5; ++c) part[c * PART_COMP + sp] = -(F[c] - Fprev[c]) * rd;
                    } else if (D == 1) {
#pragma unroll
                        for (int c = 0; c < 5; ++c)
                            part[c * PART_COMP + sp] = fma(-(F[c] - Fprev[c]), rd, part[c * PART_COMP + sp]);
                    } else {
                        double A5[5];
#pragma unroll
                        for (int c = 0; c < 5; ++c) A5[c] = fma(-(F[c] - Fprev[c]), rd, part[c * PART_COMP + sp]);
                        const long long zc = z0 + (long long)q * stride;
                        const bool grav = (g.grav[0] != 0.0) || (g.grav[1] != 0.0) || (g.grav[2] != 0.0);
                        double Um[5];
                        if (grav || NR >= 0) {
#pragma unroll
                            for (int c = 0; c < 5; ++c) Um[c] = Ub[c * g.comp_g + zc];
                        }
                        if (grav) {     // S4 source: constant gravity from the zone-centre state
                            A5[1] = fma(Um[0], g.grav[0], A5[1]);
                            A5[2] = fma(Um[0], g.grav[1], A5[2]);
                            A5[3] = fma(Um[0], g.grav[2], A5[3]);
                            A5[4] += fma(Um[3], g.grav[2], fma(Um[2], g.grav[1], Um[1] * g.grav[0]));
                        }
                        const long long ia0 = (long long)tc.b * g.box_a +
                            ((long long)(tc.k0 + lk) * g.ny + (tc.j0 + lj)) * g.nx + (tc.i0 + li);
#pragma unroll
                        for (int c = 0; c < 5; ++c) {
                            const long long ia = ia0 + c * g.comp_a;
                            if (NR >= 0)
                                up.U_next[(long long)tc.b * g.box_g + c * g.comp_g + zc] =
                                    node_update<NR>(up, Um[c], A5[c], ia);
                            A[ia] = A5[c];
                        }
                    }
                }
#pragma unroll
                for (int c = 0; c < 5; ++c) Fprev[c] = F[c];
            }
        }
#pragma unroll
        for (int c = 0; c < 5; ++c) Uc[c] = Un[c];
    }
}

template <int NR, bool FLAT>
__global__ void __launch_bounds__(NTHR, 1)
k_advect_hydro(Geom g, TileGeom tg, const double* __restrict__ U, double* __restrict__ A,
               double* __restrict__ rinv, double* __restrict__ Fm, UpdArgs up, bool x_vec, const double* __restrict__ chi)
{
    extern __shared__ double part[];                   // [5][TILE][TILE][PART_PITCH]
    const TileCoord tc = tile_coord(g, tg, blockIdx.x);
    const double* Ub = U + (long long)tc.b * g.box_g;
    double* rinv_b = rinv + (long long)tc.b * g.comp_g;
    double* fm_tile = Fm + tc.tile * 3LL * (TILE + 1) * NTHR;
    const double* chi_b = FLAT ? chi + (long long)tc.b * g.comp_g : nullptr;
    const bool full = !FLAT && (tc.tx == TILE) && (tc.ty == TILE) && (tc.tz == TILE) && x_vec;   // flattening: general body only
    if (full) {
        hydro_sweep_full<0, NR>(g, tc, Ub, part, fm_tile, rinv_b, A, up);
        __syncthreads();
        hydro_sweep_full<1, NR>(g, tc, Ub, part, fm_tile, rinv_b, A, up);
        __syncthreads();
        hydro_sweep_full<2, NR>(g, tc, Ub, part, fm_tile, rinv_b, A, up);
    } else {
        hydro_sweep<0, NR, FLAT>(g, tc, Ub, part, fm_tile, rinv_b, A, up, chi_b);
        __syncthreads();
        hydro_sweep<1, NR, FLAT>(g, tc, Ub, part, fm_tile, rinv_b, A, up, chi_b);
        __syncthreads();
        hydro_sweep<2, NR, FLAT>(g, tc, Ub, part, fm_tile, rinv_b, A, up, chi_b);
    }
}

// <A(U)> (+ node update) of the hydro components with the CFL reduction of the SAME state folded into the z sweep
// (include/cst.h cst_advance_A_update_cfl): only for lattices made of full tiles; the max signal rate of the CTA's zones
// goes through warp shuffles and one atomicMax on the bit pattern of the non-negative double, as in cfl.cu.
template <int NR>
__global__ void __launch_bounds__(NTHR, 1)
k_advect_hydro_cfl(Geom g, TileGeom tg, const double* __restrict__ U, double* __restrict__ A,
                   double* __restrict__ rinv, double* __restrict__ Fm, UpdArgs up, double* __restrict__ cfl_scratch)
{
    extern __shared__ double part[];
    __shared__ double wmax[NTHR / 32];
    const TileCoord tc = tile_coord(g, tg, blockIdx.x);
    const double* Ub = U + (long long)tc.b * g.box_g;
    double* rinv_b = rinv + (long long)tc.b * g.comp_g;
    double* fm_tile = Fm + tc.tile * 3LL * (TILE + 1) * NTHR;
    hydro_sweep_full<0, NR>(g, tc, Ub, part, fm_tile, rinv_b, A, up);
    __syncthreads();
    hydro_sweep_full<1, NR>(g, tc, Ub, part, fm_tile, rinv_b, A, up);
    __syncthreads();
    double smax = hydro_sweep_full<2, NR, true>(g, tc, Ub, part, fm_tile, rinv_b, A, up);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, o));
    if ((threadIdx.x & 31) == 0) wmax[threadIdx.x >> 5] = smax;
    __syncthreads();
    if (threadIdx.x < 32) {
        double m = threadIdx.x < NTHR / 32 ? wmax[threadIdx.x] : 0.0;
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (threadIdx.x == 0)
            atomicMax(reinterpret_cast<unsigned long long*>(cfl_scratch), (unsigned long long)__double_as_longlong(m));
    }
}

template <int NR>
static int launch_hydro_cfl_nr(cst_ctx* ctx, const double* U, double* A, const UpdArgs& up, double* cfl_scratch, cudaStream_t st)
{
    const Geom& g = ctx->g;
    const TileGeom tg = make_tile_geom(g);
    const size_t smem = 5ull * PART_COMP * sizeof(double);
    if (cudaFuncSetAttribute(k_advect_hydro_cfl<NR>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return CST_ECUDA;
    k_advect_hydro_cfl<NR><<<(unsigned)tg.ntiles, NTHR, smem, st>>>(g, tg, U, A, ctx->ws, ctx->ws + ws_rinv_doubles(g), up, cfl_scratch);
    ctx->launches++;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}

// true when the fused kernel can serve this call: every tile full, 32-byte aligned rows, no flattening
bool hydro_cfl_eligible(const cst_ctx* ctx, const double* U)
{
    const Geom& g = ctx->g;
    return !ctx->flatten && (g.nx % TILE == 0) && (g.ny % TILE == 0) && (g.nz % TILE == 0) && (((uintptr_t)U & 31) == 0);
}

int launch_advect_hydro_cfl(cst_ctx* ctx, const double* U, double* A, const UpdArgs& up, double* cfl_scratch, cudaStream_t st)
{
    switch (up.nr) {
    case -1: return launch_hydro_cfl_nr<-1>(ctx, U, A, up, cfl_scratch, st);
    case 0: return launch_hydro_cfl_nr<0>(ctx, U, A, up, cfl_scratch, st);
    case 1: return launch_hydro_cfl_nr<1>(ctx, U, A, up, cfl_scratch, st);
    case 2: return launch_hydro_cfl_nr<2>(ctx, U, A, up, cfl_scratch, st);
    case 3: return launch_hydro_cfl_nr<3>(ctx, U, A, up, cfl_scratch, st);
    }
    return CST_EINVAL;
}

template <int NR>
static int launch_hydro_nr(cst_ctx* ctx, const double* U, double* A, const UpdArgs& up, cudaStream_t st)
{
    const Geom& g = ctx->g;
    const TileGeom tg = make_tile_geom(g);
    const size_t smem = 5ull * PART_COMP * sizeof(double);
    {   // per launch: the attribute belongs to the current device's instance of the kernel
        const cudaError_t e = ctx->flatten
            ? cudaFuncSetAttribute(k_advect_hydro<NR, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)
            : cudaFuncSetAttribute(k_advect_hydro<NR, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return CST_ECUDA;
    }
    double* rinv = ctx->ws;
    double* Fm = ctx->ws + ws_rinv_doubles(g);
    // 32-byte loads of the x sweep need rows that start on 32-byte boundaries
    const bool x_vec = (g.nx % 4 == 0) && (((uintptr_t)U & 31) == 0);
    if (ctx->flatten) {
        const double* chi = Fm + ws_fm_doubles(g);
        k_advect_hydro<NR, true><<<(unsigned)tg.ntiles, NTHR, smem, st>>>(g, tg, U, A, rinv, Fm, up, x_vec, chi);
    } else {
        k_advect_hydro<NR, false><<<(unsigned)tg.ntiles, NTHR, smem, st>>>(g, tg, U, A, rinv, Fm, up, x_vec, nullptr);
    }
    ctx->launches++;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}

int launch_advect_hydro(cst_ctx* ctx, const double* U, double* A, const UpdArgs& up, cudaStream_t st)
{
    switch (up.nr) {
    case -1: return launch_hydro_nr<-1>(ctx, U, A, up, st);
    case 0: return launch_hydro_nr<0>(ctx, U, A, up, st);
    case 1: return launch_hydro_nr<1>(ctx, U, A, up, st);
    case 2: return launch_hydro_nr<2>(ctx, U, A, up, st);
    case 3: return launch_hydro_nr<3>(ctx, U, A, up, st);
    }
    return CST_EINVAL;
}
