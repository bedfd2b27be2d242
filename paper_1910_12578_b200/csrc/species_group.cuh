// species_group.cuh -- fast path of k_advect_species for full 16^3 tiles: G species per pass.
//
// A CTA of 256 / PP threads owns one tile; every thread marches PP pencils of G species AT ONCE:
// G x PP independent PPM windows in registers give each warp the instruction-level parallelism that
// the FP64 pipe latency needs, the face mass fluxes Fm and 1/rho are fetched once per G species, and
// 2 G x 16^3 doubles of shared memory per CTA (unpadded: zone (k, j, i) sits in column i ^ j of its row, which
// keeps all three pencil orientations free of bank conflicts) leave room for several CTAs per SM, whose
// streaming phases (stage the next group / write out the previous one) overlap the sweeps of the others.
// The sweep is ONE body of code with the direction as a run-time argument (strides, bases), executed
// three times, and its march is a loop over groups of four zones: the kernel stays in the
// instruction cache.
// Same arithmetic, zone for zone, as species_sweep (advect_species.cu) and as the oracle's S1-S5.
#pragma once
#include "sweep.cuh"
#include "tile.cuh"

#ifndef SPG_SWZ
#define SPG_SWZ 1          // 1: unpadded tile arrays (2 x 32 KB per species), zone (k, j, i) stored in column i ^ j
#endif
#if SPG_SWZ
#define SPG_PITCH 16
#else
#define SPG_PITCH 17
#endif
#define SPG_TILE (TILE * TILE * SPG_PITCH)
#define SPG_HALO (3 * 6 * NTHR)         // halo X values of one species: [direction][n][pencil id]

__device__ __forceinline__ unsigned long long spg_policy_keep()
{
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ unsigned long long spg_policy_stream()
{
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ double spg_ldg(const double* a, unsigned long long pol)
{
    double v;
    asm volatile("ld.global.nc.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(a), "l"(pol));
    return v;
}
__device__ __forceinline__ double2 spg_ldg2(const double* a, unsigned long long pol)
{
    double2 v;
    asm volatile("ld.global.nc.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(a), "l"(pol));
    return v;
}
__device__ __forceinline__ double2 spg_ldg2(const double* a)
{
    double2 v;
    asm volatile("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(a));
    return v;
}
__device__ __forceinline__ void spg_stg2(double* a, double2 v, unsigned long long pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1,%2}, %3;" :: "l"(a), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}

// geometry of pencil number q of this thread (pencil id = threadIdx.x + q * blockDim.x) in direction d
// (run-time d, uniform over the CTA)
struct SpgPencil {
    long long z0;      // ghosted index (within a component of the box) of pencil position 0
    long long stride;  // ghosted stride along the pencil
    int s0, sst;       // shared-memory index of position 0 and stride along the pencil
    int M, X;          // SPG_SWZ: column of position pos is ((pos & M) ^ X) on top of s0 + pos * sst
    double nrd;        // -1/delta_d
};

__device__ __forceinline__ SpgPencil spg_pencil(const Geom& g, const TileCoord& tc, const int d, const int pid)
{
    const int ng = CST_NG;
    const int a = pid & (TILE - 1), b = pid >> 4;
    SpgPencil pc;
    const long long zt = ((long long)(tc.k0 + ng) * g.ey + (tc.j0 + ng)) * g.ex + (tc.i0 + ng);
    if (d == 0) {           // (a, b) = (j, k)
        pc.z0 = zt + b * g.plane_g + (long long)a * g.ex; pc.stride = 1;
        pc.s0 = (b * TILE + a) * SPG_PITCH; pc.sst = SPG_SWZ ? 0 : 1; pc.nrd = -g.rdx; pc.M = 15; pc.X = a;
    } else if (d == 1) {    // (a, b) = (i, k)
        pc.z0 = zt + b * g.plane_g + a; pc.stride = g.ex;
        pc.s0 = (b * TILE) * SPG_PITCH + (SPG_SWZ ? 0 : a); pc.sst = SPG_PITCH; pc.nrd = -g.rdy; pc.M = 15; pc.X = a;
    } else {                // (a, b) = (i, j)
        pc.z0 = zt + (long long)b * g.ex + a; pc.stride = g.plane_g;
        pc.s0 = b * SPG_PITCH + (SPG_SWZ ? 0 : a); pc.sst = TILE * SPG_PITCH; pc.nrd = -g.rdz; pc.M = 0; pc.X = a ^ b;
    }
    return pc;
}

// shared-memory offset of pencil position pos (0..15) inside a tile array
__device__ __forceinline__ int spg_off(const SpgPencil& pc, const int pos)
{
#if SPG_SWZ
    return pc.s0 + pos * pc.sst + ((pos & pc.M) ^ pc.X);
#else
    return pc.s0 + pos * pc.sst;
#endif
}

// raw halo operands of the PP pencils: positions -3..-1 (n = 0..2) and 16..18 (n = 3..5)
template <int G, int PP>
struct SpgHaloRaw {
    double u[G][PP][6];
    double r[PP][6];
};

template <int G, int PP>
__device__ __forceinline__ void spg_halo_load(const Geom& g, const double* __restrict__ Ub,
                                              const double* __restrict__ rinv_b, const SpgPencil (&pc)[PP],
                                              const int c0, const int ng_, SpgHaloRaw<G, PP>& h,
                                              const unsigned long long keep)
{
#pragma unroll
    for (int q = 0; q < PP; ++q)
#pragma unroll
        for (int n = 0; n < 6; ++n) {
            const long long z = pc[q].z0 + (long long)(n < 3 ? n - 3 : TILE - 3 + n) * pc[q].stride;
            h.r[q][n] = spg_ldg(rinv_b + z, keep);
#pragma unroll
            for (int s = 0; s < G; ++s)
                h.u[s][q][n] = (s < ng_) ? Ub[(long long)(c0 + s) * g.comp_g + z] : 0.0;
        }
}

// One sweep of G species x PP pencils along direction d (run-time): S2 window march, F = Fm * X(upwind),
// flux difference into the partial-sum arrays.  first = true for the x sweep (the partial sum starts).
// hx[s][q][n]: halo X values (n = 0..2: positions -3..-1, n = 3..5: positions 16..18).
template <int G, int PP>
__device__ __forceinline__ void spg_sweep(const SpgPencil (&pc)[PP], const bool first, const double* __restrict__ Xs,
                                          double* __restrict__ Ps, const double* __restrict__ fm_d,
                                          const double (&hx)[G][PP][6], const unsigned long long keep)
{
    const double nrd = pc[0].nrd;
    const int nthr = NTHR / PP;
    PpmWindow w[G][PP] = {};
    double Fprev[G][PP];
    const double* __restrict__ fm = fm_d + threadIdx.x;          // pencil q: + q * nthr

    auto face = [&](const int s, const int q, const double fmc) -> double {
        return fmc * (sign_bit(fmc) ? w[s][q].qm : w[s][q].qpL);
    };
    auto zone = [&](const int s, const int q, const int pos, const double dF) {
        double* p = Ps + s * SPG_TILE + spg_off(pc[q], pos);
        const double old = first ? 0.0 : *p;
        *p = fma(dF, nrd, old);
    };
    auto xval = [&](const int s, const int q, const int pos) -> double { return Xs[s * SPG_TILE + spg_off(pc[q], pos)]; };

    // ---- prologue: pencil positions -3 .. 3 (faces 0, 1; zone 0)
    // the face mass fluxes are requested two groups of four ahead of their use (they come from HBM)
    double f0[PP], f1[PP], fn[PP][4], fnn[PP][4];
#pragma unroll
    for (int q = 0; q < PP; ++q) {
        f0[q] = spg_ldg(fm + q * nthr, keep); f1[q] = spg_ldg(fm + q * nthr + NTHR, keep);
#pragma unroll
        for (int e = 0; e < 4; ++e) fn[q][e] = spg_ldg(fm + q * nthr + (2 + e) * NTHR, keep);
#pragma unroll
        for (int e = 0; e < 4; ++e) fnn[q][e] = spg_ldg(fm + q * nthr + (6 + e) * NTHR, keep);
    }
#pragma unroll
    for (int s = 0; s < G; ++s)
#pragma unroll
        for (int q = 0; q < PP; ++q) {
            PpmWindow& ww = w[s][q];
            ww.start(hx[s][q][0]); ww.warm1(hx[s][q][1]); ww.warm2(hx[s][q][2]);
            ww.warm3(xval(s, q, 0));
            ww.push(xval(s, q, 1));
            ww.push(xval(s, q, 2));
            const double F0 = face(s, q, f0[q]);
            ww.push(xval(s, q, 3));
            const double F1 = face(s, q, f1[q]);
            zone(s, q, 0, F1 - F0);
            Fprev[s][q] = F1;
        }
    // ---- positions 4 .. 15: three groups of four (faces p-2, zones p-3)
#pragma unroll 1
    for (int it = 1; it <= 3; ++it) {
        double fc[PP][4];
#pragma unroll
        for (int q = 0; q < PP; ++q)
#pragma unroll
            for (int e = 0; e < 4; ++e) {
                fc[q][e] = fn[q][e];
                fn[q][e] = fnn[q][e];
                if (it < 2 || (it == 2 && e < 3)) fnn[q][e] = spg_ldg(fm + q * nthr + (4 * it + 6 + e) * NTHR, keep);
            }
        const int p0 = 4 * it;
#pragma unroll
        for (int e = 0; e < 4; ++e)
#pragma unroll
            for (int s = 0; s < G; ++s)
#pragma unroll
                for (int q = 0; q < PP; ++q) {
                    w[s][q].push(xval(s, q, p0 + e));
                    const double F = face(s, q, fc[q][e]);
                    zone(s, q, p0 + e - 3, F - Fprev[s][q]);
                    Fprev[s][q] = F;
                }
    }
    // ---- epilogue: positions 16 .. 18 (faces 14..16, zones 13..15)
#pragma unroll
    for (int e = 0; e < 3; ++e)
#pragma unroll
        for (int s = 0; s < G; ++s)
#pragma unroll
            for (int q = 0; q < PP; ++q) {
                w[s][q].push(hx[s][q][3 + e]);
                const double F = face(s, q, fn[q][e]);
                zone(s, q, 13 + e, F - Fprev[s][q]);
                Fprev[s][q] = F;
            }
}

// streaming phase: write out the n_out species from c_out0 (A and, fused, U_next) out of Ps, stage the
// n_in species from c_in0 into Xs.  Rows of the tile are handled as 8 x 16-byte pieces: thread t takes
// piece cp = t % 8 of rows t / 8 + (32 / PP) n (row = 16 k + j): every global access is a 16-byte vector.
// With HS (PP = 1 only) the 3-deep halos of all three directions are staged too, into
// Hs[s][direction][n = 0..5][pencil id] (n < 3: positions -3..-1, n >= 3: positions 16..18).
template <int G, int PP, int NR, bool HS>
__device__ __forceinline__ void spg_stream(const Geom& g, const TileCoord& tc, const double* __restrict__ Ub,
                                           const double* __restrict__ rinv_b, double* __restrict__ Xs,
                                           const double* __restrict__ Ps, double* __restrict__ Hs,
                                           double* __restrict__ A, const UpdArgs& up,
                                           const int c_out0, const int n_out, const int c_in0, const int n_in,
                                           const unsigned long long keep)
{
    const int ng = CST_NG;
    const int tid = threadIdx.x, cp = tid & 7, r0 = tid >> 3;
    constexpr int RS = 32 / PP, NROW = 8 * PP;          // row stride and rows per thread
    const unsigned long long strm = spg_policy_stream();
    const long long zt = ((long long)(tc.k0 + ng) * g.ey + (tc.j0 + ng)) * g.ex + (tc.i0 + ng) + 2 * cp;
    if (n_in > 0) {
        // one batch: 1/rho and the G species of all eight rows.  Rows r0 + RS n of this thread differ by RS / 16
        // planes: running pointers, one 64-bit add per array and row
        double2 ri[NROW], u[G][NROW];
        const long long zrow = zt + (long long)(r0 >> 4) * g.plane_g + (long long)(r0 & 15) * g.ex;
        const long long zstep = (RS / 16) * g.plane_g;
        const double* pr = rinv_b + zrow;
        const double* pu[G];
#pragma unroll
        for (int s = 0; s < G; ++s) pu[s] = Ub + (long long)(c_in0 + s) * g.comp_g + zrow;
#pragma unroll
        for (int n = 0; n < NROW; ++n) {
            ri[n] = spg_ldg2(pr, keep);
            pr += zstep;
#pragma unroll
            for (int s = 0; s < G; ++s) {
                if (s < n_in) u[s][n] = spg_ldg2(pu[s]);
                pu[s] += zstep;
            }
        }
#pragma unroll
        for (int n = 0; n < NROW; ++n) {
            const int row = r0 + RS * n;
#if SPG_SWZ
            double* x = Xs + row * SPG_PITCH + ((2 * cp) ^ (row & 14));
            const bool odd = row & 1;                  // odd j: the two columns of the piece swap places
#pragma unroll
            for (int s = 0; s < G; ++s)
                if (s < n_in) {
                    const double vx = u[s][n].x * ri[n].x, vy = u[s][n].y * ri[n].y;
                    *reinterpret_cast<double2*>(x + s * SPG_TILE) = odd ? make_double2(vy, vx) : make_double2(vx, vy);
                }
#else
            double* x = Xs + row * SPG_PITCH + 2 * cp;
#pragma unroll
            for (int s = 0; s < G; ++s)
                if (s < n_in) { x[s * SPG_TILE] = u[s][n].x * ri[n].x; x[s * SPG_TILE + 1] = u[s][n].y * ri[n].y; }
#endif
        }
        if (HS) {
            const long long zt0 = zt - 2 * cp;
            // y halos (consumer pencil = 16 k + i) and z halos (consumer pencil = 16 j + i): 768 16-byte pieces each
#pragma unroll
            for (int m = 0; m < 3; ++m) {
                const int idx = tid + NTHR * m, hp = idx & 7, q = (idx >> 3) & 15, n = idx >> 7;
                const int off = n < 3 ? n - 3 : TILE - 3 + n;
                const long long zy = zt0 + q * g.plane_g + (long long)off * g.ex + 2 * hp;
                const long long zz = zt0 + off * g.plane_g + (long long)q * g.ex + 2 * hp;
                const double2 ry = spg_ldg2(rinv_b + zy, keep), rz = spg_ldg2(rinv_b + zz, keep);
#pragma unroll
                for (int s = 0; s < G; ++s)
                    if (s < n_in) {
                        const double* Us = Ub + (long long)(c_in0 + s) * g.comp_g;
                        const double2 uy = spg_ldg2(Us + zy), uz = spg_ldg2(Us + zz);
                        double* h = Hs + s * SPG_HALO;
                        *reinterpret_cast<double2*>(h + (6 + n) * NTHR + q * TILE + 2 * hp) = make_double2(uy.x * ry.x, uy.y * ry.y);
                        *reinterpret_cast<double2*>(h + (12 + n) * NTHR + q * TILE + 2 * hp) = make_double2(uz.x * rz.x, uz.y * rz.y);
                    }
            }
            // x halos of this thread's own x pencil (j = tid % 16, k = tid / 16): positions -3 | -2 -1 and 16 17 | 18
            const long long zx = zt0 + (tid >> 4) * g.plane_g + (long long)(tid & 15) * g.ex;
            const double rl = spg_ldg(rinv_b + zx - 3, keep), rh = spg_ldg(rinv_b + zx + TILE + 2, keep);
            const double2 rl2 = spg_ldg2(rinv_b + zx - 2, keep), rh2 = spg_ldg2(rinv_b + zx + TILE, keep);
#pragma unroll
            for (int s = 0; s < G; ++s)
                if (s < n_in) {
                    const double* Us = Ub + (long long)(c_in0 + s) * g.comp_g;
                    const double ul = Us[zx - 3], uh = Us[zx + TILE + 2];
                    const double2 ul2 = spg_ldg2(Us + zx - 2), uh2 = spg_ldg2(Us + zx + TILE);
                    double* h = Hs + s * SPG_HALO + tid;
                    h[0] = ul * rl; h[NTHR] = ul2.x * rl2.x; h[2 * NTHR] = ul2.y * rl2.y;
                    h[3 * NTHR] = uh2.x * rh2.x; h[4 * NTHR] = uh2.y * rh2.y; h[5 * NTHR] = uh * rh;
                }
        }
    }
    if (n_out > 0) {
        const long long ia0 = (long long)tc.b * g.box_a + ((long long)tc.k0 * g.ny + tc.j0) * g.nx + tc.i0 + 2 * cp;
        const long long iu0 = (long long)tc.b * g.box_g + zt;
#pragma unroll 1
        for (int s = 0; s < n_out; ++s) {
            const long long ias = ia0 + (long long)(c_out0 + s) * g.comp_a;
            const long long ius = iu0 + (long long)(c_out0 + s) * g.comp_g;
            const double* __restrict__ pss = Ps + s * SPG_TILE;
            // batches of four rows: every load of a batch is issued before its first store; running pointers
            const long long arow = ias + ((long long)(r0 >> 4) * g.ny + (r0 & 15)) * g.nx;
            const long long astep = (long long)(RS / 16) * g.ny * g.nx;
            const long long urow = ius + (long long)(r0 >> 4) * g.plane_g + (long long)(r0 & 15) * g.ex;
            const long long ustep = (RS / 16) * g.plane_g;
            const double* pum = up.U_m + urow;
            double* pun = up.U_next + urow;
            double* pa = A + arow;
            const double* pp[UPD_MAX_EXT];
#pragma unroll
            for (int r = 0; r < UPD_MAX_EXT; ++r) pp[r] = (r < NR) ? up.P[r] + arow : nullptr;
#pragma unroll
            for (int n0 = 0; n0 < NROW; n0 += 4) {
                double2 um[4], pv[4][UPD_MAX_EXT];
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    if (NR >= 0) {
                        um[e] = spg_ldg2(pum);
                        pum += ustep;
#pragma unroll
                        for (int r = 0; r < NR; ++r) { pv[e][r] = spg_ldg2(pp[r], strm); pp[r] += astep; }
                    }
                }
#pragma unroll
                for (int e = 0; e < 4; ++e) {
                    const int row = r0 + RS * (n0 + e);
#if SPG_SWZ
                    const double2 raw = *reinterpret_cast<const double2*>(pss + row * SPG_PITCH + ((2 * cp) ^ (row & 14)));
                    const double2 av = (row & 1) ? make_double2(raw.y, raw.x) : raw;
#else
                    const double* x = pss + row * SPG_PITCH + 2 * cp;
                    const double2 av = make_double2(x[0], x[1]);
#endif
                    if (NR >= 0) {
                        double2 acc = make_double2(fma(up.ca, av.x, um[e].x), fma(up.ca, av.y, um[e].y));
#pragma unroll
                        for (int r = 0; r < NR; ++r) {
                            acc.x = fma(up.c[r], pv[e][r].x, acc.x); acc.y = fma(up.c[r], pv[e][r].y, acc.y);
                        }
                        spg_stg2(pun, acc, strm);
                        pun += ustep;
                    }
                    spg_stg2(pa, av, strm);
                    pa += astep;
                }
            }
        }
    }
}

// the species [s_begin, s_end) of one full tile, G at a time
template <int G, int PP, int NR, bool HS>
__device__ __forceinline__ void spg_tile(const Geom& g, const TileCoord& tc, const double* __restrict__ Ub,
                                         const double* __restrict__ rinv_b, const double* __restrict__ fm_tile,
                                         double* __restrict__ A, const UpdArgs& up, double* __restrict__ sm,
                                         const int s_begin, const int s_end)
{
    static_assert(!(HS && SPG_SWZ), "halo staging is not written for the swizzled layout");
    static_assert(!HS || PP == 1, "halo staging in shared memory is written for one pencil per thread");
    double* Xs = sm;                    // [G][SPG_TILE]  X of the tile core
    double* Ps = sm + G * SPG_TILE;     // [G][SPG_TILE]  A under construction
    double* Hs = sm + 2 * G * SPG_TILE; // [G][SPG_HALO]  halo X values (HS only)
    const int tid = threadIdx.x, nthr = NTHR / PP;
    int c_prev = 0, n_prev = 0;
#pragma unroll 1
    for (int s0 = s_begin; s0 < s_end; s0 += G) {
        const int n_in = min(G, s_end - s0), c_in = 5 + s0;
        // 1/rho and Fm of this tile stay in L2 (evict_last) until the last species, which demotes them
        const unsigned long long keep = (s0 + G >= s_end) ? spg_policy_stream() : spg_policy_keep();
        __syncthreads();                                // z sweep of the previous group done
        spg_stream<G, PP, NR, HS>(g, tc, Ub, rinv_b, Xs, Ps, Hs, A, up, c_prev, n_prev, c_in, n_in, keep);
        SpgHaloRaw<G, PP> hr;
        SpgPencil pc[PP];
#pragma unroll
        for (int q = 0; q < PP; ++q) pc[q] = spg_pencil(g, tc, 0, tid + q * nthr);
        // without HS: halo operands of the x sweep (products formed after the barrier, when the loads have landed)
        if (!HS) spg_halo_load<G, PP>(g, Ub, rinv_b, pc, c_in, n_in, hr, keep);
        __syncthreads();
#pragma unroll 1
        for (int d = 0; d < 3; ++d) {
            double hx[G][PP][6];
            SpgPencil pcd[PP];
#pragma unroll
            for (int q = 0; q < PP; ++q) pcd[q] = pc[q];
            if (HS) {
#pragma unroll
                for (int s = 0; s < G; ++s)
#pragma unroll
                    for (int n = 0; n < 6; ++n) hx[s][0][n] = Hs[s * SPG_HALO + (d * 6 + n) * NTHR + tid];
                if (d < 2) pc[0] = spg_pencil(g, tc, d + 1, tid);
            } else {
#pragma unroll
                for (int s = 0; s < G; ++s)
#pragma unroll
                    for (int q = 0; q < PP; ++q)
#pragma unroll
                        for (int n = 0; n < 6; ++n) hx[s][q][n] = hr.u[s][q][n] * hr.r[q][n];
                if (d < 2) {                            // operands of the next sweep: in flight during this one
#pragma unroll
                    for (int q = 0; q < PP; ++q) pc[q] = spg_pencil(g, tc, d + 1, tid + q * nthr);
                    spg_halo_load<G, PP>(g, Ub, rinv_b, pc, c_in, n_in, hr, keep);
                }
            }
            spg_sweep<G, PP>(pcd, d == 0, Xs, Ps, fm_tile + (d * (TILE + 1)) * NTHR, hx, keep);
            if (d < 2) __syncthreads();
        }
        c_prev = c_in; n_prev = n_in;
    }
    __syncthreads();
    spg_stream<G, PP, NR, HS>(g, tc, Ub, rinv_b, Xs, Ps, Hs, A, up, c_prev, n_prev, 0, 0, spg_policy_stream());
}
