// exchange.cu -- the box lattice sharded over ranks ("MPI distribute the AMR grids across nodes";
// SURVEY 8(e); include/cst.h cst_set_sublattice, cst_exchange_*).
//
// The global lattice of gnbx x gnby x gnbz boxes is cut into part[0] x part[1] x part[2] equal bricks, one per rank
// (rank = pi + part[0] * (pj + part[1] * pk)).  Within one <A(U)> evaluation every box is independent once its ghost
// shell is filled, so the only data that crosses ranks is the 4-deep shell of boxes on a brick surface:
//   * cst_fill_ghosts fills every ghost zone whose SOURCE box is local (ghost_fill.cu, global zone map);
//   * the remaining ghost zones are described by SEGMENTS: one per (destination box, one of its 26 shell regions)
//     whose source box lives on another rank.  Because a box is at least as wide as the shell (n >= ng) a region
//     has exactly one source box, and along each direction the source index runs with step +1 (neighbour box or
//     periodic wrap), 0 (outflow: every ghost copies the boundary zone) or -1 (reflecting mirror, with the
//     wall-normal momentum negated);
//   * the sender packs the source zones of a segment in the DESTINATION's zone order, signs applied
//     (k_exchange_pack), so the receiver's unpack is a plain copy into the region (k_exchange_unpack);
//   * all segments between one (sender, receiver) pair travel as ONE message, in a canonical order both sides derive
//     on their own: destination boxes in the receiver's local order, regions in (rz, ry, rx) order.
// The plan is pure host arithmetic (cst_exchange_plan needs no GPU and is what the CPU tests check against a
// brute-force ghost map); the kernels only walk the segment table.
#include <algorithm>
#include <new>
#include <vector>
#include "common.cuh"

namespace {

struct Lattice {
    int n[3], gnb[3], part[3], lb[3];      // zones per box, global boxes, ranks, boxes per brick
    int bc_lo[3], bc_hi[3];
    int nvar;
};

struct DimMap { int sbox; int lo; int step; int flip; };

// direction d, destination box at global lattice coordinate gb, shell region r = -1 / 0 / +1:
// source box (global coordinate), ghosted index of the source of the region's first zone, step, sign flip
DimMap map_region(const Lattice& L, int d, int gb, int r)
{
    const int ng = CST_NG, n = L.n[d], G = L.gnb[d];
    if (r == 0) return { gb, ng, 1, 0 };
    if (r < 0) {
        if (gb > 0) return { gb - 1, n, 1, 0 };
        if (L.bc_lo[d] == CST_BC_PERIODIC) return { G - 1, n, 1, 0 };
        if (L.bc_lo[d] == CST_BC_OUTFLOW) return { 0, ng, 0, 0 };
        return { 0, 2 * ng - 1, -1, 1 };
    }
    if (gb < G - 1) return { gb + 1, ng, 1, 0 };
    if (L.bc_hi[d] == CST_BC_PERIODIC) return { 0, ng, 1, 0 };
    if (L.bc_hi[d] == CST_BC_OUTFLOW) return { G - 1, ng + n - 1, 0, 0 };
    return { G - 1, ng + n - 1, -1, 1 };
}

int rank_of_box(const Lattice& L, const int gb[3])
{
    return gb[0] / L.lb[0] + L.part[0] * (gb[1] / L.lb[1] + L.part[1] * (gb[2] / L.lb[2]));
}
void rank_coords(const Lattice& L, int rank, int p[3])
{
    p[0] = rank % L.part[0]; p[1] = (rank / L.part[0]) % L.part[1]; p[2] = rank / (L.part[0] * L.part[1]);
}

// all segments whose destination box lives on rank `dst_rank`, canonical order; each with the owner of its source
struct RawSeg { int dst_box, src_box, src_rank; int dlo[3], slo[3], step[3], ext[3], flip[3]; };
void enumerate_dst(const Lattice& L, int dst_rank, std::vector<RawSeg>& out)
{
    const int ng = CST_NG;
    int p[3];
    rank_coords(L, dst_rank, p);
    for (int bk = 0; bk < L.lb[2]; ++bk)
    for (int bj = 0; bj < L.lb[1]; ++bj)
    for (int bi = 0; bi < L.lb[0]; ++bi) {
        const int lb3[3] = { bi, bj, bk };
        int gb[3];
        for (int d = 0; d < 3; ++d) gb[d] = p[d] * L.lb[d] + lb3[d];
        for (int rz = -1; rz <= 1; ++rz)
        for (int ry = -1; ry <= 1; ++ry)
        for (int rx = -1; rx <= 1; ++rx) {
            if (!rx && !ry && !rz) continue;
            const int r[3] = { rx, ry, rz };
            RawSeg s;
            int sgb[3];
            for (int d = 0; d < 3; ++d) {
                const DimMap m = map_region(L, d, gb[d], r[d]);
                sgb[d] = m.sbox; s.slo[d] = m.lo; s.step[d] = m.step; s.flip[d] = m.flip;
                s.dlo[d] = r[d] < 0 ? 0 : r[d] == 0 ? ng : ng + L.n[d];
                s.ext[d] = r[d] == 0 ? L.n[d] : ng;
            }
            s.src_rank = rank_of_box(L, sgb);
            int sp[3];
            rank_coords(L, s.src_rank, sp);
            s.src_box = (sgb[0] - sp[0] * L.lb[0]) + L.lb[0] * ((sgb[1] - sp[1] * L.lb[1]) + L.lb[1] * (sgb[2] - sp[2] * L.lb[2]));
            s.dst_box = bi + L.lb[0] * (bj + L.lb[1] * bk);
            out.push_back(s);
        }
    }
}

bool make_lattice(const cst_params* gp, const int part[3], Lattice& L)
{
    if (!gp || !part || gp->ng != CST_NG) return false;
    const int n[3] = { gp->nx, gp->ny, gp->nz }, gnb[3] = { gp->nbx, gp->nby, gp->nbz };
    for (int d = 0; d < 3; ++d) {
        if (part[d] < 1 || gnb[d] < 1 || gnb[d] % part[d] || n[d] < CST_NG) return false;
        L.n[d] = n[d]; L.gnb[d] = gnb[d]; L.part[d] = part[d]; L.lb[d] = gnb[d] / part[d];
        L.bc_lo[d] = gp->bc_lo[d]; L.bc_hi[d] = gp->bc_hi[d];
        if (L.bc_lo[d] < 0 || L.bc_lo[d] > 2 || L.bc_hi[d] < 0 || L.bc_hi[d] > 2) return false;
        if ((L.bc_lo[d] == CST_BC_PERIODIC) != (L.bc_hi[d] == CST_BC_PERIODIC)) return false;
    }
    L.nvar = 5 + gp->nspec;
    return gp->nspec >= 0 && gp->nspec <= CST_MAX_NSPEC;
}

// the ranks whose bricks touch (or wrap onto) the brick of `rank`, itself excluded, ascending
std::vector<int> neighbour_ranks(const Lattice& L, int rank)
{
    int p[3];
    rank_coords(L, rank, p);
    std::vector<int> v;
    for (int dz = -1; dz <= 1; ++dz)
    for (int dy = -1; dy <= 1; ++dy)
    for (int dx = -1; dx <= 1; ++dx) {
        const int q[3] = { (p[0] + dx + L.part[0]) % L.part[0], (p[1] + dy + L.part[1]) % L.part[1],
                           (p[2] + dz + L.part[2]) % L.part[2] };
        const int r = q[0] + L.part[0] * (q[1] + L.part[1] * q[2]);
        if (r != rank) v.push_back(r);
    }
    std::sort(v.begin(), v.end());
    v.erase(std::unique(v.begin(), v.end()), v.end());
    return v;
}

// segments of `rank`: recv = 1: its own ghost regions with a remote source; recv = 0: regions of other ranks' boxes
// whose source box is local.  Grouped by peer (ascending), canonical order inside; offset = doubles from the start
// of that peer's message.
void plan_segments(const Lattice& L, int rank, int recv, std::vector<cst_xseg>& out)
{
    std::vector<RawSeg> raw;
    if (recv) {
        enumerate_dst(L, rank, raw);
        std::vector<int> peers;
        for (const RawSeg& s : raw) if (s.src_rank != rank) peers.push_back(s.src_rank);
        std::sort(peers.begin(), peers.end());
        peers.erase(std::unique(peers.begin(), peers.end()), peers.end());
        for (int q : peers) {
            long long off = 0;
            for (const RawSeg& s : raw) {
                if (s.src_rank != q) continue;
                cst_xseg x;
                x.peer = q; x.box = s.dst_box; x.offset = off; x.rbox = s.src_box;
                for (int d = 0; d < 3; ++d) { x.lo[d] = s.dlo[d]; x.step[d] = 1; x.ext[d] = s.ext[d]; x.flip[d] = 0; x.rlo[d] = s.slo[d]; }
                off += (long long)L.nvar * s.ext[0] * s.ext[1] * s.ext[2];
                out.push_back(x);
            }
        }
    } else {
        for (int q : neighbour_ranks(L, rank)) {
            raw.clear();
            enumerate_dst(L, q, raw);
            long long off = 0;
            for (const RawSeg& s : raw) {
                if (s.src_rank != rank) continue;
                cst_xseg x;
                x.peer = q; x.box = s.src_box; x.offset = off; x.rbox = s.dst_box;
                for (int d = 0; d < 3; ++d) { x.lo[d] = s.slo[d]; x.step[d] = s.step[d]; x.ext[d] = s.ext[d]; x.flip[d] = s.flip[d]; x.rlo[d] = s.dlo[d]; }
                off += (long long)L.nvar * s.ext[0] * s.ext[1] * s.ext[2];
                out.push_back(x);
            }
        }
    }
}

struct DevSeg {
    int box;
    int lo[3], step[3], ext[3], flip[3];
    int peer_slot, rbox, rlo[3];   // send segments: index of the peer in the plan's peer list, destination box / first zone there
    long long off;            // doubles from the start of the whole send / receive buffer
    long long zone_start;     // first zone (all components) of this segment in the flat thread index
};

}  // namespace

struct XPlan {
    std::vector<int> peers;
    std::vector<long long> send_off, send_len, recv_off, recv_len;      // doubles, per peer
    DevSeg *d_send = nullptr, *d_recv = nullptr;
    long long n_send = 0, n_recv = 0, zones_send = 0, zones_recv = 0;
};

extern "C" long long cst_exchange_plan(const cst_params* gp, const int part[3], int rank, int recv,
                                       cst_xseg* segs, long long cap)
{
    Lattice L;
    if (!make_lattice(gp, part, L)) return CST_EINVAL;
    if (rank < 0 || rank >= part[0] * part[1] * part[2]) return CST_EINVAL;
    std::vector<cst_xseg> v;
    plan_segments(L, rank, recv ? 1 : 0, v);
    if (segs) for (long long n = 0; n < (long long)v.size() && n < cap; ++n) segs[n] = v[n];
    return (long long)v.size();
}

static long long upload(const std::vector<cst_xseg>& v, const std::vector<int>& peers, const std::vector<long long>& base,
                        int nvar, DevSeg** d_out, long long* zones)
{
    std::vector<DevSeg> h(v.size());
    long long z = 0;
    for (size_t n = 0; n < v.size(); ++n) {
        DevSeg& s = h[n];
        s.box = v[n].box;
        for (int d = 0; d < 3; ++d) { s.lo[d] = v[n].lo[d]; s.step[d] = v[n].step[d]; s.ext[d] = v[n].ext[d]; s.flip[d] = v[n].flip[d]; }
        const size_t pi = std::lower_bound(peers.begin(), peers.end(), v[n].peer) - peers.begin();
        s.off = base[pi] + v[n].offset;
        s.peer_slot = (int)pi; s.rbox = v[n].rbox;
        for (int d = 0; d < 3; ++d) s.rlo[d] = v[n].rlo[d];
        s.zone_start = z;
        z += (long long)s.ext[0] * s.ext[1] * s.ext[2];
    }
    (void)nvar;
    *zones = z;
    *d_out = nullptr;
    if (h.empty()) return 0;
    if (cudaMalloc((void**)d_out, h.size() * sizeof(DevSeg)) != cudaSuccess) return -1;
    if (cudaMemcpyAsync(*d_out, h.data(), h.size() * sizeof(DevSeg), cudaMemcpyHostToDevice, 0) != cudaSuccess ||
        cudaStreamSynchronize(0) != cudaSuccess)
        return -1;
    return (long long)h.size();
}

void xplan_destroy(cst_ctx* ctx)
{
    if (!ctx->xplan) return;
    if (ctx->xplan->d_send) cudaFree(ctx->xplan->d_send);
    if (ctx->xplan->d_recv) cudaFree(ctx->xplan->d_recv);
    delete ctx->xplan;
    ctx->xplan = nullptr;
}

int xplan_create(cst_ctx* ctx, const int global_nb[3], const int part[3], int rank)
{
    Geom& g = ctx->g;
    cst_params gp = ctx->p;
    gp.nbx = global_nb[0]; gp.nby = global_nb[1]; gp.nbz = global_nb[2];
    Lattice L;
    if (!make_lattice(&gp, part, L)) return CST_EINVAL;
    if (L.lb[0] != g.nbx || L.lb[1] != g.nby || L.lb[2] != g.nbz) return CST_EINVAL;
    if (rank < 0 || rank >= part[0] * part[1] * part[2]) return CST_EINVAL;
    xplan_destroy(ctx);
    XPlan* xp = new (std::nothrow) XPlan();
    if (!xp) return CST_ENOMEM;
    std::vector<cst_xseg> snd, rcv;
    plan_segments(L, rank, 0, snd);
    plan_segments(L, rank, 1, rcv);
    for (const cst_xseg& s : snd) xp->peers.push_back(s.peer);
    for (const cst_xseg& s : rcv) xp->peers.push_back(s.peer);
    std::sort(xp->peers.begin(), xp->peers.end());
    xp->peers.erase(std::unique(xp->peers.begin(), xp->peers.end()), xp->peers.end());
    const size_t np = xp->peers.size();
    xp->send_off.assign(np, 0); xp->send_len.assign(np, 0); xp->recv_off.assign(np, 0); xp->recv_len.assign(np, 0);
    auto lens = [&](const std::vector<cst_xseg>& v, std::vector<long long>& len) {
        for (const cst_xseg& s : v) {
            const size_t pi = std::lower_bound(xp->peers.begin(), xp->peers.end(), s.peer) - xp->peers.begin();
            len[pi] = std::max(len[pi], s.offset + (long long)g.nvar * s.ext[0] * s.ext[1] * s.ext[2]);
        }
    };
    lens(snd, xp->send_len); lens(rcv, xp->recv_len);
    for (size_t n = 1; n < np; ++n) {
        xp->send_off[n] = xp->send_off[n - 1] + xp->send_len[n - 1];
        xp->recv_off[n] = xp->recv_off[n - 1] + xp->recv_len[n - 1];
    }
    xp->n_send = upload(snd, xp->peers, xp->send_off, g.nvar, &xp->d_send, &xp->zones_send);
    xp->n_recv = upload(rcv, xp->peers, xp->recv_off, g.nvar, &xp->d_recv, &xp->zones_recv);
    ctx->xplan = xp;
    if (xp->n_send < 0 || xp->n_recv < 0) { xplan_destroy(ctx); return CST_ECUDA; }
    int p[3];
    rank_coords(L, rank, p);
    g.gnbx = global_nb[0]; g.gnby = global_nb[1]; g.gnbz = global_nb[2];
    g.obx = p[0] * L.lb[0]; g.oby = p[1] * L.lb[1]; g.obz = p[2] * L.lb[2];
    return CST_OK;
}

int xplan_info(const cst_ctx* ctx, int* npeers, int* peers, long long* send_off, long long* send_len,
               long long* recv_off, long long* recv_len, int cap)
{
    const XPlan* xp = ctx->xplan;
    if (!xp || !npeers) return CST_EINVAL;
    *npeers = (int)xp->peers.size();
    for (int n = 0; n < *npeers && n < cap; ++n) {
        if (peers) peers[n] = xp->peers[n];
        if (send_off) send_off[n] = xp->send_off[n];
        if (send_len) send_len[n] = xp->send_len[n];
        if (recv_off) recv_off[n] = xp->recv_off[n];
        if (recv_len) recv_len[n] = xp->recv_len[n];
    }
    return CST_OK;
}

// One thread per zone of a segment, all NVAR components (the zone map is computed once).  PACK: buffer <- U (source
// order with steps, momentum signs applied); !PACK: U <- buffer (plain copy into the ghost region).
template <bool PACK>
__global__ void __launch_bounds__(256)
k_exchange(Geom g, const DevSeg* __restrict__ segs, int nseg, long long zones, double* __restrict__ U,
           double* __restrict__ buf)
{
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < zones; t += (long long)gridDim.x * blockDim.x) {
        int lo = 0, hi = nseg - 1;                    // last segment with zone_start <= t
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (segs[mid].zone_start <= t) lo = mid; else hi = mid - 1;
        }
        const DevSeg& s = segs[lo];
        const long long z = t - s.zone_start;
        const int ix = (int)(z % s.ext[0]);
        const long long r = z / s.ext[0];
        const int iy = (int)(r % s.ext[1]), iz = (int)(r / s.ext[1]);
        const long long nz = (long long)s.ext[0] * s.ext[1] * s.ext[2];
        const long long u0 = uidx(g, s.box, 0, s.lo[2] + s.step[2] * iz, s.lo[1] + s.step[1] * iy, s.lo[0] + s.step[0] * ix);
        double* __restrict__ b = buf + s.off + z;
        for (int c = 0; c < g.nvar; ++c) {
            if (PACK) {
                const double v = U[u0 + c * g.comp_g];
                const bool neg = (c >= 1 && c <= 3) && s.flip[c - 1];
                b[c * nz] = neg ? -v : v;
            } else {
                U[u0 + c * g.comp_g] = b[c * nz];
            }
        }
    }
}

// The exchange WITHOUT staging buffers: every zone a peer's ghost shell reads from this brick is written straight into
// the peer's array through a peer-mapped pointer (NVLink stores; the caller obtained the pointers with cst_ipc_import
// or, in one process, passes the arrays themselves).  Same zone map and signs as pack + unpack.
struct PeerPtrs { double* p[CST_MAX_PEERS]; };
__global__ void __launch_bounds__(256)
k_exchange_push(Geom g, const DevSeg* __restrict__ segs, int nseg, long long zones, const double* __restrict__ U, PeerPtrs peers)
{
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < zones; t += (long long)gridDim.x * blockDim.x) {
        int lo = 0, hi = nseg - 1;
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (segs[mid].zone_start <= t) lo = mid; else hi = mid - 1;
        }
        const DevSeg& s = segs[lo];
        const long long z = t - s.zone_start;
        const int ix = (int)(z % s.ext[0]);
        const long long r = z / s.ext[0];
        const int iy = (int)(r % s.ext[1]), iz = (int)(r / s.ext[1]);
        const long long u0 = uidx(g, s.box, 0, s.lo[2] + s.step[2] * iz, s.lo[1] + s.step[1] * iy, s.lo[0] + s.step[0] * ix);
        const long long d0 = uidx(g, s.rbox, 0, s.rlo[2] + iz, s.rlo[1] + iy, s.rlo[0] + ix);     // every brick has the same shape
        double* __restrict__ dst = peers.p[s.peer_slot] + d0;
        for (int c = 0; c < g.nvar; ++c) {
            const double v = U[u0 + c * g.comp_g];
            const bool neg = (c >= 1 && c <= 3) && s.flip[c - 1];
            dst[c * g.comp_g] = neg ? -v : v;
        }
    }
}

int launch_exchange_push(cst_ctx* ctx, const double* U, double* const* peer_U, int npeers, cudaStream_t st)
{
    const XPlan* xp = ctx->xplan;
    if (!xp || npeers != (int)xp->peers.size() || npeers > CST_MAX_PEERS) return CST_EINVAL;
    if (xp->zones_send == 0) return CST_OK;
    PeerPtrs pp{};
    for (int n = 0; n < npeers; ++n) { if (!peer_U[n]) return CST_EINVAL; pp.p[n] = peer_U[n]; }
    long long nb = (xp->zones_send + 255) / 256;
    const long long cap = (long long)ctx->sm_count * 16;
    if (nb > cap) nb = cap;
    k_exchange_push<<<(unsigned)nb, 256, 0, st>>>(ctx->g, xp->d_send, (int)xp->n_send, xp->zones_send, U, pp);
    ctx->launches++;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}

static int launch_exchange(cst_ctx* ctx, double* U, double* buf, bool pack, cudaStream_t st)
{
    const XPlan* xp = ctx->xplan;
    if (!xp) return CST_EINVAL;
    const long long zones = pack ? xp->zones_send : xp->zones_recv;
    const long long nseg = pack ? xp->n_send : xp->n_recv;
    if (zones == 0) return CST_OK;
    long long nb = (zones + 255) / 256;
    const long long cap = (long long)ctx->sm_count * 16;
    if (nb > cap) nb = cap;
    if (pack) k_exchange<true><<<(unsigned)nb, 256, 0, st>>>(ctx->g, xp->d_send, (int)nseg, zones, U, buf);
    else      k_exchange<false><<<(unsigned)nb, 256, 0, st>>>(ctx->g, xp->d_recv, (int)nseg, zones, U, buf);
    ctx->launches++;
    return cudaGetLastError() == cudaSuccess ? CST_OK : CST_ECUDA;
}

int launch_exchange_pack(cst_ctx* ctx, const double* U, double* sendbuf, cudaStream_t st)
{
    return launch_exchange(ctx, const_cast<double*>(U), sendbuf, true, st);
}
int launch_exchange_unpack(cst_ctx* ctx, double* U, const double* recvbuf, cudaStream_t st)
{
    return launch_exchange(ctx, U, const_cast<double*>(recvbuf), false, st);
}
