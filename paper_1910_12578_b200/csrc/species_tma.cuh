// species_tma.cuh -- fast path of the species kernel for boxes made of full 16^3 tiles (k_advect_species_tma).
//
// One CTA (256 threads) works on one 16^3 tile and a contiguous share of the species; two CTAs share an SM.  Per species:
//   * rho X of the tile core PLUS its x halos arrives by ONE tensor-map (TMA) tile load (box 24 x 16 x 16: zones -4 .. 19
//     of every x pencil -- a box must start on a 16-byte boundary, measured: an odd fp64 start coordinate faults),
//     completing on an mbarrier; the box was pulled into L2 by a tensor prefetch a whole species pass earlier and the
//     load itself is issued as soon as the previous species' z sweep has released the buffer, so it overlaps the
//     write-out of that species;
//   * the face mass fluxes Fm, 1/rho and the fused update's operands (A_old arrays) are pulled into L2 by bulk / tensor
//     prefetches one pass ahead of the loads that use them;
//   * X = rho X / rho is formed in place (halo columns included), then three sweeps (x, y, z), one pencil per thread
//     with the PPM window in registers (sweep.cuh), accumulate -div F into the partial-sum tile; the next pass writes
//     A (and U_next) out.
// Shared memory: the X tile has dense rows of 24 doubles (x = -4 .. 19), the partial-sum tile rows of 18 doubles (84 KB per
// CTA, 168 KB per SM: the L1 that is left still carries the remaining per-thread global loads -- at 216 KB the same
// kernel ran 1.4x slower).  Every access of every sweep is "pencil base + immediate"; rows stay 16-byte aligned; the x
// sweep reads and writes PAIRS of zones (16-byte accesses; the partial-sum rows are conflict free because 9 j mod 8 is a
// permutation, the twelve X reads per pencil pay a 4-way conflict: 3 % of the sweep); the y / z sweeps touch 16 consecutive
// doubles per half warp -- no swizzle arithmetic, and the x halos never travel through registers.
// Same arithmetic, zone for zone, as species_sweep (advect_species.cu) and as the oracle's S1-S5.
#pragma once
#include "sweep.cuh"
#include "tile.cuh"
#include "tma.cuh"

#define SPT_XW 24                             // X tile row: zones -4 .. 19 of the x pencil
#define SPT_XPLANE (TILE * SPT_XW)            // 384 doubles
#define SPT_XTILE (TILE * SPT_XPLANE)         // 6144 doubles
#define SPT_XTILE_BYTES (SPT_XTILE * 8)       // 49152 = the TMA box 24 x 16 x 16
#define SPT_PITCH 18                          // partial-sum tile row (zones 0 .. 15 + 2 pad)
#define SPT_PLANE (TILE * SPT_PITCH)          // 288 doubles
#define SPT_TILE (TILE * SPT_PLANE)           // 4608 doubles
#define SPT_SMEM (SPT_XTILE_BYTES + SPT_TILE * 8 + 128)   // X, P, one mbarrier

struct SptMaps {             // tensor maps of one call (host-encoded, passed as a __grid_constant__ kernel parameter)
    CUtensorMap u;           // U as [nbox*nvar*ez][ey][ex], box 24 x 16 x 16: tile core + x halos (load and L2 prefetch)
    CUtensorMap r;           // 1/rho workspace as [nbox*ez][ey][ex], box 24 x 22 x 22: L2 prefetch of the tile's star
    CUtensorMap p[UPD_MAX_EXT];   // external arrays of the fused update as [nbox*nvar*nz][ny][nx], box 16^3: L2 prefetch
};

__device__ __forceinline__ unsigned long long spt_policy_keep()
{
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ unsigned long long spt_policy_stream()
{
    unsigned long long p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ double spt_ldg(const double* a, unsigned long long pol)
{
    double v;
    asm volatile("ld.global.nc.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(a), "l"(pol));
    return v;
}
__device__ __forceinline__ double2 spt_ldg2(const double* a, unsigned long long pol)
{
    double2 v;
    asm volatile("ld.global.nc.L2::cache_hint.v2.f64 {%0,%1}, [%2], %3;" : "=d"(v.x), "=d"(v.y) : "l"(a), "l"(pol));
    return v;
}
__device__ __forceinline__ double2 spt_ldg2(const double* a)
{
    double2 v;
    asm volatile("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(a));
    return v;
}
__device__ __forceinline__ void spt_stg2(double* a, double2 v, unsigned long long pol)
{
    asm volatile("st.global.L2::cache_hint.v2.f64 [%0], {%1,%2}, %3;" :: "l"(a), "d"(v.x), "d"(v.y), "l"(pol) : "memory");
}

__device__ __forceinline__ void spt_stg(double* a, double v, unsigned long long pol)
{
    asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" :: "l"(a), "d"(v), "l"(pol) : "memory");
}

// Pencil of this thread in direction D: (a, b) = (tid % 16, tid / 16) = (j, k) | (i, k) | (i, j).
// X tile: zone (k, j, x) at k * SPT_XPLANE + j * SPT_XW + (x + 4), x = -4 .. 19; P tile: zone (k, j, i) at
// k * SPT_PLANE + j * SPT_PITCH + i.
template <int D> struct SptDir {
    static constexpr int XS = (D == 0) ? 1 : (D == 1) ? SPT_XW : SPT_XPLANE;        // X stride along the pencil
    static constexpr int PS = (D == 0) ? 1 : (D == 1) ? SPT_PITCH : SPT_PLANE;      // P stride along the pencil
};
template <int D>
__device__ __forceinline__ int spt_xbase(const int a, const int b)
{   // X index of pencil position 0 (D = 0: of position -4, the start of the row)
    return (D == 0) ? (b * TILE + a) * SPT_XW : (D == 1) ? b * SPT_XPLANE + a + 4 : b * SPT_XW + a + 4;
}
template <int D>
__device__ __forceinline__ int spt_pbase(const int a, const int b)
{
    return (D == 0) ? (b * TILE + a) * SPT_PITCH : (D == 1) ? b * SPT_PLANE + a : b * SPT_PITCH + a;
}

struct SptHalo { double u[6], r[6]; };      // raw rho X and 1/rho at pencil positions -3..-1 (0..2) and 16..18 (3..5)

// halo operands of this thread's y (d = 1) or z (d = 2) pencil, straight from global memory (16 consecutive doubles
// per half warp): requested one sweep before they are used
__device__ __forceinline__ void spt_halo_load(const Geom& g, const TileCoord& tc, const int d, const double* __restrict__ Us,
                                              const double* __restrict__ rinv_b, SptHalo& h, const unsigned long long keep)
{
    const int ng = CST_NG, a = threadIdx.x & (TILE - 1), b = threadIdx.x >> 4;
    const long long zt = ((long long)(tc.k0 + ng) * g.ey + (tc.j0 + ng)) * g.ex + (tc.i0 + ng);
    long long z0, stride;
    if (d == 1) { z0 = zt + b * g.plane_g + a; stride = g.ex; }
    else { z0 = zt + (long long)b * g.ex + a; stride = g.plane_g; }
#pragma unroll
    for (int n = 0; n < 6; ++n) {
        const long long z = z0 + (long long)(n < 3 ? n - 3 : TILE - 3 + n) * stride;
        h.r[n] = spt_ldg(rinv_b + z, keep);
        h.u[n] = Us[z];
    }
}

__device__ __forceinline__ double spt_face(const PpmWindow& w, const double fmc)
{   // F(rho X) = F(rho) * X(upwind side): the sign of the mass flux picks the side (Q8)
    return fmc * (sign_bit(fmc) ? w.qm : w.qpL);
}

// y or z sweep: X and P of pencil position p at Xp[p * XS], Pp[p * PS] (compile-time strides).  Face mass fluxes of
// the pencil: thread-private slots fm[f * NTHR], f = 0..16, requested two groups of four ahead of their use.
template <int D>
__device__ __forceinline__ void spt_sweep_yz(const double* __restrict__ Xp, double* __restrict__ Pp,
                                             const double* __restrict__ fm, const double (&hx)[6], const double nrd,
                                             const unsigned long long keep)
{
    constexpr int XS = SptDir<D>::XS, PS = SptDir<D>::PS;
    PpmWindow w;
    double fn[4], fnn[4];
    const double f0 = spt_ldg(fm, keep), f1 = spt_ldg(fm + NTHR, keep);
#pragma unroll
    for (int e = 0; e < 4; ++e) fn[e] = spt_ldg(fm + (2 + e) * NTHR, keep);
#pragma unroll
    for (int e = 0; e < 4; ++e) fnn[e] = spt_ldg(fm + (6 + e) * NTHR, keep);
    w.start(hx[0]); w.warm1(hx[1]); w.warm2(hx[2]);
    w.warm3(Xp[0]);
    w.push(Xp[XS]);
    w.push(Xp[2 * XS]);
    const double F0 = spt_face(w, f0);
    w.push(Xp[3 * XS]);
    double Fprev = spt_face(w, f1);
    Pp[0] = fma(Fprev - F0, nrd, Pp[0]);
#pragma unroll 1
    for (int it = 1; it <= 3; ++it) {                 // positions 4it .. 4it+3: faces 4it-2 .., zones 4it-3 ..
        double fc[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            fc[e] = fn[e];
            fn[e] = fnn[e];
            if (it < 2 || (it == 2 && e < 3)) fnn[e] = spt_ldg(fm + (4 * it + 6 + e) * NTHR, keep);
        }
        const double* __restrict__ xg = Xp + 4 * it * XS;
        double* __restrict__ pg = Pp + (4 * it - 3) * PS;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            w.push(xg[e * XS]);
            const double F = spt_face(w, fc[e]);
            pg[e * PS] = fma(F - Fprev, nrd, pg[e * PS]);
            Fprev = F;
        }
    }
#pragma unroll
    for (int e = 0; e < 3; ++e) {
        w.push(hx[3 + e]);
        const double F = spt_face(w, fn[e]);
        Pp[(13 + e) * PS] = fma(F - Fprev, nrd, Pp[(13 + e) * PS]);
        Fprev = F;
    }
}

// x sweep: starts the partial sum.  The pencil is one row of the X tile, halos included: Xr[o] = X at position o - 4,
// read as twelve pairs (positions (2m-4, 2m-3) in pair m); the row of P is written as eight pairs.
__device__ __forceinline__ void spt_sweep_x(const double* __restrict__ Xr, double* __restrict__ Pp,
                                            const double* __restrict__ fm, const double nrd, const unsigned long long keep)
{
    PpmWindow w;
    double fn[4], fnn[4];
    const double f0 = spt_ldg(fm, keep), f1 = spt_ldg(fm + NTHR, keep);
#pragma unroll
    for (int e = 0; e < 4; ++e) fn[e] = spt_ldg(fm + (2 + e) * NTHR, keep);
#pragma unroll
    for (int e = 0; e < 4; ++e) fnn[e] = spt_ldg(fm + (6 + e) * NTHR, keep);
    const double2 h0 = *reinterpret_cast<const double2*>(Xr), h1 = *reinterpret_cast<const double2*>(Xr + 2);
    const double2 xa = *reinterpret_cast<const double2*>(Xr + 4), xb = *reinterpret_cast<const double2*>(Xr + 6);
    w.start(h0.y); w.warm1(h1.x); w.warm2(h1.y);
    w.warm3(xa.x);
    w.push(xa.y);
    w.push(xb.x);
    const double F0 = spt_face(w, f0);
    w.push(xb.y);
    double Fprev = spt_face(w, f1);
    double pend = fma(Fprev - F0, nrd, 0.0);                    // zone 0, stored with zone 1
#pragma unroll 1
    for (int it = 1; it <= 3; ++it) {                 // positions 4it .. 4it+3: faces 4it-2 .., zones 4it-3 ..
        double fc[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            fc[e] = fn[e];
            fn[e] = fnn[e];
            if (it < 2 || (it == 2 && e < 3)) fnn[e] = spt_ldg(fm + (4 * it + 6 + e) * NTHR, keep);
        }
        const double2 xc = *reinterpret_cast<const double2*>(Xr + 4 + 4 * it), xd = *reinterpret_cast<const double2*>(Xr + 6 + 4 * it);
        double* __restrict__ pg = Pp + 4 * it - 4;                 // zones 4it-4 .. 4it-1 are complete after this group
        double F, z, hold;
        w.push(xc.x); F = spt_face(w, fc[0]); z = fma(F - Fprev, nrd, 0.0); Fprev = F;
        *reinterpret_cast<double2*>(pg) = make_double2(pend, z);
        w.push(xc.y); F = spt_face(w, fc[1]); hold = fma(F - Fprev, nrd, 0.0); Fprev = F;
        w.push(xd.x); F = spt_face(w, fc[2]); z = fma(F - Fprev, nrd, 0.0); Fprev = F;
        *reinterpret_cast<double2*>(pg + 2) = make_double2(hold, z);
        w.push(xd.y); F = spt_face(w, fc[3]); pend = fma(F - Fprev, nrd, 0.0); Fprev = F;
    }
    {
        const double2 xe = *reinterpret_cast<const double2*>(Xr + 20), xf = *reinterpret_cast<const double2*>(Xr + 22);
        double F, z, hold;
        w.push(xe.x); F = spt_face(w, fn[0]); z = fma(F - Fprev, nrd, 0.0); Fprev = F;
        *reinterpret_cast<double2*>(Pp + 12) = make_double2(pend, z);
        w.push(xe.y); F = spt_face(w, fn[1]); hold = fma(F - Fprev, nrd, 0.0); Fprev = F;
        w.push(xf.x); F = spt_face(w, fn[2]); z = fma(F - Fprev, nrd, 0.0);
        *reinterpret_cast<double2*>(Pp + 14) = make_double2(hold, z);
    }
}

// ---- variant kernels (cst_set_variant; species_tile V = 1, 2): the same arithmetic with fewer phases per species ----
// x sweep that also forms X = rho X / rho: the pencil's row of the raw tile (24 values, halos included) is multiplied by
// the row of 1/rho (twelve 16-byte loads requested up front, consumed in pencil order), fed to the window, and the core
// pairs are written back in place for the y / z sweeps.  Replaces spt_convert (one phase, one dependent round of L2
// loads and 2 x 48 KB of shared-memory traffic per species).  Same products, same order: results are bit-identical.
__device__ __forceinline__ double2 spt_conv_pair(double* __restrict__ Xr, const int o, const double2 r, const bool core)
{   // X of the two positions at row offset o; core pairs go back to the tile for the y / z sweeps
    double2 v = *reinterpret_cast<const double2*>(Xr + o);
    v.x *= r.x; v.y *= r.y;
    if (core) *reinterpret_cast<double2*>(Xr + o) = v;
    return v;
}
__device__ __forceinline__ void spt_sweep_x_conv(double* __restrict__ Xr, double* __restrict__ Pp, const double* __restrict__ fm,
                                                 const double* __restrict__ rrow, const double nrd, const unsigned long long keep)
{
    PpmWindow w;
    const double2 r0 = spt_ldg2(rrow, keep), r1 = spt_ldg2(rrow + 2, keep), r2 = spt_ldg2(rrow + 4, keep), r3 = spt_ldg2(rrow + 6, keep);
    double2 rn0 = spt_ldg2(rrow + 8, keep), rn1 = spt_ldg2(rrow + 10, keep);     // 1/rho of the next group of four
    double fn[4], fnn[4];
    const double f0 = spt_ldg(fm, keep), f1 = spt_ldg(fm + NTHR, keep);
#pragma unroll
    for (int e = 0; e < 4; ++e) fn[e] = spt_ldg(fm + (2 + e) * NTHR, keep);
#pragma unroll
    for (int e = 0; e < 4; ++e) fnn[e] = spt_ldg(fm + (6 + e) * NTHR, keep);
    const double2 h0 = spt_conv_pair(Xr, 0, r0, false), h1 = spt_conv_pair(Xr, 2, r1, false);
    const double2 xa = spt_conv_pair(Xr, 4, r2, true), xb = spt_conv_pair(Xr, 6, r3, true);
    w.start(h0.y); w.warm1(h1.x); w.warm2(h1.y);
    w.warm3(xa.x);
    w.push(xa.y);
    w.push(xb.x);
    const double F0 = spt_face(w, f0);
    w.push(xb.y);
    double Fprev = spt_face(w, f1);
    double pend = fma(Fprev - F0, nrd, 0.0);                    // zone 0, stored with zone 1
#pragma unroll 1
    for (int it = 1; it <= 3; ++it) {                 // positions 4it .. 4it+3: faces 4it-2 .., zones 4it-3 ..
        double fc[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            fc[e] = fn[e];
            fn[e] = fnn[e];
            if (it < 2 || (it == 2 && e < 3)) fnn[e] = spt_ldg(fm + (4 * it + 6 + e) * NTHR, keep);
        }
        const double2 rc0 = rn0, rc1 = rn1;
        rn0 = spt_ldg2(rrow + 8 + 4 * it, keep); rn1 = spt_ldg2(rrow + 10 + 4 * it, keep);   // it = 3: the pairs of the tail
        const double2 xc = spt_conv_pair(Xr, 4 + 4 * it, rc0, true), xd = spt_conv_pair(Xr, 6 + 4 * it, rc1, true);
        double* __restrict__ pg = Pp + 4 * it - 4;                 // zones 4it-4 .. 4it-1 are complete after this group
        double F, z, hold;
        w.push(xc.x); F = spt_face(w, fc[0]); z = fma(F - Fprev, nrd, 0.0); Fprev = F;
        *reinterpret_cast<double2*>(pg) = make_double2(pend, z);
        w.push(xc.y); F = spt_face(w, fc[1]); hold = fma(F - Fprev, nrd, 0.0); Fprev = F;
        w.push(xd.x); F = spt_face(w, fc[2]); z = fma(F - Fprev, nrd, 0.0); Fprev = F;
        *reinterpret_cast<double2*>(pg + 2) = make_double2(hold, z);
        w.push(xd.y); F = spt_face(w, fc[3]); pend = fma(F - Fprev, nrd, 0.0); Fprev = F;
    }
    {
        const double2 xe = spt_conv_pair(Xr, 20, rn0, false), xf = spt_conv_pair(Xr, 22, rn1, false);
        double F, z, hold;
        w.push(xe.x); F = spt_face(w, fn[0]); z = fma(F - Fprev, nrd, 0.0); Fprev = F;
        *reinterpret_cast<double2*>(Pp + 12) = make_double2(pend, z);
        w.push(xe.y); F = spt_face(w, fn[1]); hold = fma(F - Fprev, nrd, 0.0); Fprev = F;
        w.push(xf.x); F = spt_face(w, fn[2]); z = fma(F - Fprev, nrd, 0.0);
        *reinterpret_cast<double2*>(Pp + 14) = make_double2(hold, z);
    }
}

// z sweep that also writes the component out: the zone that a step completes gets A = P + z contribution and, fused,
// U_next = U_m + ca A + sum c_r P_r straight from the sweep (a half warp covers 16 consecutive zones of a row: full
// 128-byte segments), so the separate write-out phase of the next pass -- and its read of the partial-sum tile -- is gone.
// Operands of the update are requested one group of four zones ahead.  Same operations in the same order as
// spt_write_out: bit-identical results.
struct SptOut {              // per-thread addresses of the zone column (i, j, k = 0 .. 15) of component c
    const double* um; double* un; double* a; const double* p[UPD_MAX_EXT];
    long long ustep, astep;
};
template <int NR>
__device__ __forceinline__ void spt_sweep_z_out(const double* __restrict__ Xp, const double* __restrict__ Pp,
                                                const double* __restrict__ fm, const double (&hx)[6], const double nrd,
                                                const unsigned long long keep, const UpdArgs& up, SptOut o)
{
    constexpr int XS = SptDir<2>::XS, PS = SptDir<2>::PS;
    const unsigned long long strm = spt_policy_stream();
    PpmWindow w;
    double fn[4], fnn[4];
    const double f0 = spt_ldg(fm, keep), f1 = spt_ldg(fm + NTHR, keep);
#pragma unroll
    for (int e = 0; e < 4; ++e) fn[e] = spt_ldg(fm + (2 + e) * NTHR, keep);
#pragma unroll
    for (int e = 0; e < 4; ++e) fnn[e] = spt_ldg(fm + (6 + e) * NTHR, keep);
    // operands of zone 0 and of the first group (zones 1 .. 4)
    double um0 = 0.0, pv0[UPD_MAX_EXT] = {}, umn[4] = {}, pvn[4][UPD_MAX_EXT] = {};
    if (NR >= 0) {
        um0 = spt_ldg(o.um, strm);
#pragma unroll
        for (int r = 0; r < NR; ++r) pv0[r] = spt_ldg(o.p[r], strm);
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            umn[e] = spt_ldg(o.um + (1 + e) * o.ustep, strm);
#pragma unroll
            for (int r = 0; r < NR; ++r) pvn[e][r] = spt_ldg(o.p[r] + (1 + e) * o.astep, strm);
        }
    }
    auto emit = [&](const int q, const double av, const double um, const double (&pv)[UPD_MAX_EXT]) {
        if (NR >= 0) {
            double acc = fma(up.ca, av, um);
#pragma unroll
            for (int r = 0; r < NR; ++r) acc = fma(up.c[r], pv[r], acc);
            spt_stg(o.un + q * o.ustep, acc, strm);
        }
        spt_stg(o.a + q * o.astep, av, strm);
    };
    w.start(hx[0]); w.warm1(hx[1]); w.warm2(hx[2]);
    w.warm3(Xp[0]);
    w.push(Xp[XS]);
    w.push(Xp[2 * XS]);
    const double F0 = spt_face(w, f0);
    w.push(Xp[3 * XS]);
    double Fprev = spt_face(w, f1);
    emit(0, fma(Fprev - F0, nrd, Pp[0]), um0, pv0);
#pragma unroll 1
    for (int it = 1; it <= 3; ++it) {                 // positions 4it .. 4it+3: faces 4it-2 .., zones 4it-3 .. 4it
        double fc[4], umc[4] = {}, pvc[4][UPD_MAX_EXT] = {};
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            fc[e] = fn[e];
            fn[e] = fnn[e];
            if (it < 2 || (it == 2 && e < 3)) fnn[e] = spt_ldg(fm + (4 * it + 6 + e) * NTHR, keep);
            if (NR >= 0) {
                umc[e] = umn[e];
#pragma unroll
                for (int r = 0; r < NR; ++r) pvc[e][r] = pvn[e][r];
                const int qn = 4 * it + 1 + e;                     // zone of the next group (13 .. 15 in the tail)
                if (qn < TILE) {
                    umn[e] = spt_ldg(o.um + qn * o.ustep, strm);
#pragma unroll
                    for (int r = 0; r < NR; ++r) pvn[e][r] = spt_ldg(o.p[r] + qn * o.astep, strm);
                }
            }
        }
        const double* __restrict__ xg = Xp + 4 * it * XS;
        const double* __restrict__ pg = Pp + (4 * it - 3) * PS;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            w.push(xg[e * XS]);
            const double F = spt_face(w, fc[e]);
            emit(4 * it - 3 + e, fma(F - Fprev, nrd, pg[e * PS]), umc[e], pvc[e]);
            Fprev = F;
        }
    }
#pragma unroll
    for (int e = 0; e < 3; ++e) {
        w.push(hx[3 + e]);
        const double F = spt_face(w, fn[e]);
        emit(13 + e, fma(F - Fprev, nrd, Pp[(13 + e) * PS]), umn[e], pvn[e]);
        Fprev = F;
    }
}

// write out component c_out of the tile from the partial-sum tile: A and, fused, U_next = U_m + ca A + sum c_r P_r.
// Thread t takes the 16-byte piece t % 8 of rows t / 8 + 32 n (row = 16 k + j): every global access is a 16-byte vector.
template <int NR>
__device__ __forceinline__ void spt_write_out(const Geom& g, const TileCoord& tc, const double* __restrict__ Ps,
                                              double* __restrict__ A, const UpdArgs& up, const int c_out)
{
    const int ng = CST_NG;
    const int tid = threadIdx.x, cp = tid & 7, r0 = tid >> 3;
    const unsigned long long strm = spt_policy_stream();
    const long long zt = ((long long)(tc.k0 + ng) * g.ey + (tc.j0 + ng)) * g.ex + (tc.i0 + ng) + 2 * cp;
    const long long arow = (long long)tc.b * g.box_a + (long long)c_out * g.comp_a +
        ((long long)(tc.k0 + (r0 >> 4)) * g.ny + tc.j0 + (r0 & 15)) * g.nx + tc.i0 + 2 * cp;
    const long long astep = 2LL * g.ny * g.nx;
    const long long urow = (long long)tc.b * g.box_g + (long long)c_out * g.comp_g + zt +
        (long long)(r0 >> 4) * g.plane_g + (long long)(r0 & 15) * g.ex;
    const long long ustep = 2 * g.plane_g;
    const double* pum = up.U_m + urow;
    double* pun = up.U_next + urow;
    double* pa = A + arow;
    const double* pp[UPD_MAX_EXT];
#pragma unroll
    for (int r = 0; r < UPD_MAX_EXT; ++r) pp[r] = (r < NR) ? up.P[r] + arow : nullptr;
    const double* ps = Ps + r0 * SPT_PITCH + 2 * cp;
#pragma unroll
    for (int n0 = 0; n0 < 8; n0 += 4) {
        double2 um[4], pv[4][UPD_MAX_EXT];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            if (NR >= 0) {
                um[e] = spt_ldg2(pum);
                pum += ustep;
#pragma unroll
                for (int r = 0; r < NR; ++r) { pv[e][r] = spt_ldg2(pp[r], strm); pp[r] += astep; }
            }
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const double2 av = *reinterpret_cast<const double2*>(ps + 32 * (n0 + e) * SPT_PITCH);
            if (NR >= 0) {
                double2 acc = make_double2(fma(up.ca, av.x, um[e].x), fma(up.ca, av.y, um[e].y));
#pragma unroll
                for (int r = 0; r < NR; ++r) {
                    acc.x = fma(up.c[r], pv[e][r].x, acc.x); acc.y = fma(up.c[r], pv[e][r].y, acc.y);
                }
                spt_stg2(pun, acc, strm);
                pun += ustep;
            }
            spt_stg2(pa, av, strm);
            pa += astep;
        }
    }
}

// X = rho X / rho in place on the tile the TMA load has just delivered (waits for it on the mbarrier), x-halo columns
// included.  A k plane of the tile is 16 rows x 24 columns = 384 consecutive doubles of shared memory: thread t takes
// elements t (and t + 256 when below 384) of every plane; its (row, column) is the same in all 16 planes, and
// consecutive threads read consecutive zones of a row of 1/rho.
__device__ __forceinline__ void spt_convert(const Geom& g, const TileCoord& tc, double* __restrict__ Xs,
                                            const double* __restrict__ rinv_b, uint64_t* bar, const uint32_t parity,
                                            const unsigned long long keep)
{
    const int ng = CST_NG;
    const int tid = threadIdx.x;
    const long long zt = ((long long)(tc.k0 + ng) * g.ey + (tc.j0 + ng)) * g.ex + (tc.i0 + ng) - 4;
    const int j1 = tid / SPT_XW, c1 = tid - j1 * SPT_XW;
    const int e2 = tid + NTHR, j2 = e2 / SPT_XW, c2 = e2 - j2 * SPT_XW;
    const bool two = e2 < SPT_XPLANE;
    const double* p1 = rinv_b + zt + (long long)j1 * g.ex + c1;
    const double* p2 = rinv_b + zt + (long long)j2 * g.ex + c2;
    double r1[TILE], r2[TILE];
#pragma unroll
    for (int k = 0; k < TILE; ++k) r1[k] = spt_ldg(p1 + k * g.plane_g, keep);
    if (two) {
#pragma unroll
        for (int k = 0; k < TILE; ++k) r2[k] = spt_ldg(p2 + k * g.plane_g, keep);
    }
    mbar_wait(bar, parity);
#pragma unroll
    for (int k = 0; k < TILE; ++k) Xs[k * SPT_XPLANE + tid] *= r1[k];
    if (two) {
#pragma unroll
        for (int k = 0; k < TILE; ++k) Xs[k * SPT_XPLANE + e2] *= r2[k];
    }
}

// the species [s_begin, s_end) of one full tile
template <int NR>
__device__ __forceinline__ void spt_tile(const Geom& g, const TileCoord& tc, const SptMaps& maps,
                                         const double* __restrict__ Ub, const double* __restrict__ rinv_b,
                                         const double* __restrict__ fm_tile, double* __restrict__ A, const UpdArgs& up,
                                         double* __restrict__ sm, const int s_begin, const int s_end)
{
    const int ng = CST_NG;
    double* Xs = sm;                                  // [SPT_XTILE]
    double* PB = sm + SPT_XTILE;                      // [SPT_TILE]
    uint64_t* bar = reinterpret_cast<uint64_t*>(sm + SPT_XTILE + SPT_TILE);
    const int tid = threadIdx.x, a = tid & (TILE - 1), b = tid >> 4;
    const int tx = tc.i0 + ng - 4, ty = tc.j0 + ng;           // x, y coordinates of the tile box in the U tensor map
    const int zc0 = (tc.b * g.nvar) * g.ez + tc.k0 + ng;      // z coordinate of component 0
    const int za0 = (tc.b * g.nvar) * g.nz + tc.k0;           // ... in the A-like tensor maps
    if (tid == 0) {
        mbar_init(bar, 1);
        fence_mbar_init();
        mbar_expect_tx(bar, SPT_XTILE_BYTES);
        tma_load_3d(Xs, &maps.u, tx, ty, zc0 + (5 + s_begin) * g.ez, bar);
        // the tile's face mass fluxes and 1/rho star: one trip from HBM into L2 for all species passes
        bulk_prefetch_l2(fm_tile, 3 * (TILE + 1) * NTHR * 8);
        tma_prefetch_3d(&maps.r, tc.i0, tc.j0 + 1, tc.b * g.ez + tc.k0 + 1);
    }
    __syncthreads();
    const double nrdx = -g.rdx, nrdy = -g.rdy, nrdz = -g.rdz;
    const double* __restrict__ fm = fm_tile + tid;
    int n = 0;
#pragma unroll 1
    for (int s = s_begin; s < s_end; ++s, ++n) {
        const int c = 5 + s;
        const bool last = (s + 1 >= s_end);
        // 1/rho and Fm of this tile stay in L2 (evict_last) until the last species, which demotes them
        const unsigned long long keep = last ? spt_policy_stream() : spt_policy_keep();
        const double* Us = Ub + (long long)c * g.comp_g;
        if (n > 0) spt_write_out<NR>(g, tc, PB, A, up, c - 1);       // overlaps the tile load issued after the z sweep
        if (tid == 0) {                               // L2 prefetches a pass ahead: next species' tile, this species' write-out operands
            if (!last) tma_prefetch_3d(&maps.u, tx, ty, zc0 + (c + 1) * g.ez);
            if (NR > 0) {
#pragma unroll
                for (int r = 0; r < NR; ++r) tma_prefetch_3d(&maps.p[r], tc.i0, tc.j0, za0 + c * g.nz);
            }
        }
        spt_convert(g, tc, Xs, rinv_b, bar, n & 1, keep);
        SptHalo hr;
        spt_halo_load(g, tc, 1, Us, rinv_b, hr, keep);           // operands of the y sweep: in flight during the x sweep
        __syncthreads();                              // X complete; P free (written out)
        double hx[6];
        // ---- x sweep
        spt_sweep_x(Xs + spt_xbase<0>(a, b), PB + spt_pbase<0>(a, b), fm, nrdx, keep);
        __syncthreads();
        // ---- y sweep
#pragma unroll
        for (int m = 0; m < 6; ++m) hx[m] = hr.u[m] * hr.r[m];
        spt_halo_load(g, tc, 2, Us, rinv_b, hr, keep);
        spt_sweep_yz<1>(Xs + spt_xbase<1>(a, b), PB + spt_pbase<1>(a, b), fm + (TILE + 1) * NTHR, hx, nrdy, keep);
        __syncthreads();
        // ---- z sweep
#pragma unroll
        for (int m = 0; m < 6; ++m) hx[m] = hr.u[m] * hr.r[m];
        spt_sweep_yz<2>(Xs + spt_xbase<2>(a, b), PB + spt_pbase<2>(a, b), fm + 2 * (TILE + 1) * NTHR, hx, nrdz, keep);
        __syncthreads();                              // X released, P complete
        if (tid == 0 && !last) {                      // next species' tile (already in L2): lands during the write-out
            fence_proxy_async();
            mbar_expect_tx(bar, SPT_XTILE_BYTES);
            tma_load_3d(Xs, &maps.u, tx, ty, zc0 + (c + 1) * g.ez, bar);
        }
    }
    spt_write_out<NR>(g, tc, PB, A, up, 5 + s_end - 1);
}

// the species [s_begin, s_end) of one full tile, variant kernels: V = 1 forms X inside the x sweep (no conversion phase);
// V = 2 also writes each component out from its own z sweep (no write-out phase, one barrier fewer per species; the tile
// load of the next species is then issued right after the z sweep and is hidden only by the other CTA of the SM).
template <int NR, int V>
__device__ __forceinline__ void spt_tile_v(const Geom& g, const TileCoord& tc, const SptMaps& maps,
                                           const double* __restrict__ Ub, const double* __restrict__ rinv_b,
                                           const double* __restrict__ fm_tile, double* __restrict__ A, const UpdArgs& up,
                                           double* __restrict__ sm, const int s_begin, const int s_end)
{
    constexpr bool ZOUT = (V >= 2), LATE = (V == 3);     // V = 3: as 2, with the L2 prefetches issued one sweep ahead of their use
    const int ng = CST_NG;
    double* Xs = sm;                                  // [SPT_XTILE]
    double* PB = sm + SPT_XTILE;                      // [SPT_TILE]
    uint64_t* bar = reinterpret_cast<uint64_t*>(sm + SPT_XTILE + SPT_TILE);
    const int tid = threadIdx.x, a = tid & (TILE - 1), b = tid >> 4;
    const int tx = tc.i0 + ng - 4, ty = tc.j0 + ng;
    const int zc0 = (tc.b * g.nvar) * g.ez + tc.k0 + ng;
    const int za0 = (tc.b * g.nvar) * g.nz + tc.k0;
    if (tid == 0) {
        mbar_init(bar, 1);
        fence_mbar_init();
        mbar_expect_tx(bar, SPT_XTILE_BYTES);
        tma_load_3d(Xs, &maps.u, tx, ty, zc0 + (5 + s_begin) * g.ez, bar);
        bulk_prefetch_l2(fm_tile, 3 * (TILE + 1) * NTHR * 8);
        tma_prefetch_3d(&maps.r, tc.i0, tc.j0 + 1, tc.b * g.ez + tc.k0 + 1);
    }
    __syncthreads();                                  // the initialised barrier is visible to every waiter
    const double nrdx = -g.rdx, nrdy = -g.rdy, nrdz = -g.rdz;
    const double* __restrict__ fm = fm_tile + tid;
    // ghosted index of the tile origin; the x pencil (j = a, k = b) starts four zones to the left of it
    const long long zt = ((long long)(tc.k0 + ng) * g.ey + (tc.j0 + ng)) * g.ex + (tc.i0 + ng);
    const double* __restrict__ rrow = rinv_b + zt + (long long)b * g.plane_g + (long long)a * g.ex - 4;
    // z pencil (i = a, j = b): the column of zones this thread completes
    const long long ucol = (long long)tc.b * g.box_g + zt + (long long)b * g.ex + a;
    const long long acol = (long long)tc.b * g.box_a + ((long long)tc.k0 * g.ny + tc.j0 + b) * g.nx + tc.i0 + a;
    int n = 0;
#pragma unroll 1
    for (int s = s_begin; s < s_end; ++s, ++n) {
        const int c = 5 + s;
        const bool last = (s + 1 >= s_end);
        const unsigned long long keep = last ? spt_policy_stream() : spt_policy_keep();
        const double* Us = Ub + (long long)c * g.comp_g;
        if (!ZOUT && n > 0) spt_write_out<NR>(g, tc, PB, A, up, c - 1);
        if (tid == 0 && !LATE) {
            if (!last) tma_prefetch_3d(&maps.u, tx, ty, zc0 + (c + 1) * g.ez);
            if (NR > 0) {
#pragma unroll
                for (int r = 0; r < NR; ++r) tma_prefetch_3d(&maps.p[r], tc.i0, tc.j0, za0 + c * g.nz);
            }
        }
        SptHalo hr;
        spt_halo_load(g, tc, 1, Us, rinv_b, hr, keep);           // operands of the y sweep: in flight during the x sweep
        if (!ZOUT && n > 0) __syncthreads();          // P free (written out); with ZOUT the barrier after the z sweep did that
        mbar_wait(bar, n & 1);                        // the raw tile has landed (every thread reads only its own row next)
        double hx[6];
        // ---- x sweep (+ conversion)
        spt_sweep_x_conv(Xs + spt_xbase<0>(a, b), PB + spt_pbase<0>(a, b), fm, rrow, nrdx, keep);
        __syncthreads();
        if (LATE && tid == 0 && NR > 0) {             // operands of this component's update: read by the z sweep
#pragma unroll
            for (int r = 0; r < NR; ++r) tma_prefetch_3d(&maps.p[r], tc.i0, tc.j0, za0 + c * g.nz);
        }
        // ---- y sweep
#pragma unroll
        for (int m = 0; m < 6; ++m) hx[m] = hr.u[m] * hr.r[m];
        spt_halo_load(g, tc, 2, Us, rinv_b, hr, keep);
        spt_sweep_yz<1>(Xs + spt_xbase<1>(a, b), PB + spt_pbase<1>(a, b), fm + (TILE + 1) * NTHR, hx, nrdy, keep);
        __syncthreads();
        if (LATE && tid == 0 && !last) tma_prefetch_3d(&maps.u, tx, ty, zc0 + (c + 1) * g.ez);   // the tile loaded after the z sweep
        // ---- z sweep (+ write-out)
#pragma unroll
        for (int m = 0; m < 6; ++m) hx[m] = hr.u[m] * hr.r[m];
        if (ZOUT) {
            SptOut o;
            o.ustep = g.plane_g; o.astep = (long long)g.ny * g.nx;
            o.um = (NR >= 0) ? up.U_m + ucol + (long long)c * g.comp_g : nullptr;
            o.un = (NR >= 0) ? up.U_next + ucol + (long long)c * g.comp_g : nullptr;
            o.a = A + acol + (long long)c * g.comp_a;
#pragma unroll
            for (int r = 0; r < UPD_MAX_EXT; ++r) o.p[r] = (r < NR) ? up.P[r] + acol + (long long)c * g.comp_a : nullptr;
            spt_sweep_z_out<NR>(Xs + spt_xbase<2>(a, b), PB + spt_pbase<2>(a, b), fm + 2 * (TILE + 1) * NTHR, hx, nrdz, keep, up, o);
        } else {
            spt_sweep_yz<2>(Xs + spt_xbase<2>(a, b), PB + spt_pbase<2>(a, b), fm + 2 * (TILE + 1) * NTHR, hx, nrdz, keep);
        }
        __syncthreads();                              // X released (and, with ZOUT, P read)
        if (tid == 0 && !last) {
            fence_proxy_async();
            mbar_expect_tx(bar, SPT_XTILE_BYTES);
            tma_load_3d(Xs, &maps.u, tx, ty, zc0 + (c + 1) * g.ez, bar);
        }
    }
    if (!ZOUT) spt_write_out<NR>(g, tc, PB, A, up, 5 + s_end - 1);
}
