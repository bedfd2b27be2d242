// tile.cuh -- tiling of a box into 16^3-zone tiles and the pencil <-> thread map shared by the
// hydro and species kernels of <A(U)>.
//
// One CTA of 256 threads owns one tile of up to 16 x 16 x 16 interior zones of one box.  In the
// sweep along direction d every thread owns one PENCIL of the tile (a line of zones along d) and
// marches along it with the PPM stencil in a register window:
//     x sweep: thread (a, b) = (j, k)      y sweep: (a, b) = (i, k)      z sweep: (a, b) = (i, j)
// with a = tid % 16, b = tid / 16.  The face mass fluxes F(rho) that couple the species to the
// hydro are exchanged through a THREAD-PRIVATE slot array in the workspace:
//     Fm[((tile * 3 + d) * (TILE + 1) + f) * NTHR + tid],   f = 0 .. L  (face f lies between zones f-1, f)
// which is written and read with the same thread map, so every access is fully coalesced.
#pragma once
#include "common.cuh"

#define TILE 16
#define NTHR 256

struct TileGeom {
    int ntx, nty, ntz;        // tiles per box in each direction
    int tiles_per_box;
    long long ntiles;         // nbox * tiles_per_box
};

__host__ __device__ inline TileGeom make_tile_geom(const Geom& g)
{
    TileGeom t;
    t.ntx = (g.nx + TILE - 1) / TILE;
    t.nty = (g.ny + TILE - 1) / TILE;
    t.ntz = (g.nz + TILE - 1) / TILE;
    t.tiles_per_box = t.ntx * t.nty * t.ntz;
    t.ntiles = (long long)g.nbox * t.tiles_per_box;
    return t;
}

// workspace layout (doubles): [ rinv : nbox * comp_g ][ Fm : ntiles * 3 * (TILE+1) * NTHR ]
__host__ __device__ inline long long ws_rinv_doubles(const Geom& g) { return (long long)g.nbox * g.comp_g; }
__host__ __device__ inline long long ws_fm_doubles(const Geom& g)
{
    return make_tile_geom(g).ntiles * 3LL * (TILE + 1) * NTHR;
}

struct TileCoord {
    int b;                    // box
    int i0, j0, k0;           // interior origin of the tile inside the box
    int tx, ty, tz;           // extents (<= TILE)
    long long tile;           // global tile index
};

// blockIdx -> tile.  Tiles are numbered x-fastest inside a box (that number addresses the Fm workspace),
// but a big box is WALKED brick by brick (8 x 8 x 4 tiles): the ~300 tiles that are resident on the GPU
// at one time then form a compact brick whose halo reads hit in L2, instead of a one-tile-thick slab
// whose z neighbours were evicted long ago.
#define BRICK_X 8
#define BRICK_Y 8
#define BRICK_Z 4
__device__ __forceinline__ TileCoord tile_coord(const Geom& g, const TileGeom& tg, long long blk)
{
    TileCoord t;
    t.b = (int)(blk / tg.tiles_per_box);
    int r = (int)(blk - (long long)t.b * tg.tiles_per_box);
    int ti, tj, tk;
    if ((tg.ntx % BRICK_X == 0) && (tg.nty % BRICK_Y == 0) && (tg.ntz % BRICK_Z == 0)) {
        const int per = BRICK_X * BRICK_Y * BRICK_Z;
        const int brick = r / per, w = r - brick * per;
        const int nbx = tg.ntx / BRICK_X, nby = tg.nty / BRICK_Y;
        const int bz = brick / (nbx * nby), br = brick - bz * nbx * nby, by = br / nbx, bx = br - by * nbx;
        const int wz = w / (BRICK_X * BRICK_Y), wr = w - wz * BRICK_X * BRICK_Y, wy = wr / BRICK_X, wx = wr - wy * BRICK_X;
        ti = bx * BRICK_X + wx; tj = by * BRICK_Y + wy; tk = bz * BRICK_Z + wz;
    } else {
        tk = r / (tg.ntx * tg.nty);
        r -= tk * tg.ntx * tg.nty;
        tj = r / tg.ntx; ti = r - tj * tg.ntx;
    }
    t.tile = (long long)t.b * tg.tiles_per_box + ((long long)tk * tg.nty + tj) * tg.ntx + ti;
    t.i0 = ti * TILE; t.j0 = tj * TILE; t.k0 = tk * TILE;
    t.tx = min(TILE, g.nx - t.i0); t.ty = min(TILE, g.ny - t.j0); t.tz = min(TILE, g.nz - t.k0);
    return t;
}

#define UPD_MAX_EXT 3        // external arrays the fused update can read (more -> unfused calls)

// The SDC node update fused behind A (S5, Eq. (2) of the paper with R = 0):
//   U_next = U_m + dt_m (A_new - A_old) + sum_q w_q A_q
// normalised on the host into  U_next = U_m + ca * A_new + sum_{r < nr} c[r] * P[r]
// where every occurrence of the A_new buffer among A_old / A_q is folded into ca and equal
// pointers are merged (advect.cu make_upd).  nr = -1: no update (plain cst_advance_A).
struct UpdArgs {
    int nr;
    const double* U_m;        // the state A is evaluated on (ghosted layout)
    double* U_next;
    const double* A_base;     // the A_new array (index origin of the A-like arrays)
    double ca;
    const double* P[UPD_MAX_EXT];
    double c[UPD_MAX_EXT];
};

template <int NR>
__device__ __forceinline__ double node_update(const UpdArgs& up, double um, double a, long long ia)
{
    double acc = fma(up.ca, a, um);
#pragma unroll
    for (int r = 0; r < NR; ++r) acc = fma(up.c[r], up.P[r][ia], acc);
    return acc;
}
