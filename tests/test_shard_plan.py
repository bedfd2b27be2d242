"""The ghost-exchange plan of the sharded box lattice (include/cst.h cst_exchange_plan)
on the CPU: the plan is a pure host function of libcst.so, so it can be checked without a GPU.

For every rank of a partition, numpy executes the plan (pack from the sender's INTERIOR zones, unpack into the
receiver's ghost regions) and the result is compared with the oracle's ghost fill of the whole lattice, bit for bit;
a brute-force restatement of the S0 zone map, written out here, says which ghost zones have a remote source: the
plan must cover exactly those.  A world-size-2 gloo run sends the same messages through torch.distributed with the
product's GhostExchange plumbing (paper_1910_12578_b200/shard.py).
"""
import os
import sys

import numpy as np
import pytest

from oracle import orc
from paper_1910_12578_b200 import binding, shard, workloads as wl
from test_oracle_pins import small_cfg

NG = 4


def brute_source(cfg, gz, d):
    """S0 map of one direction written out: global zone index (may be outside) -> in-domain source index."""
    n = (cfg["nx"], cfg["ny"], cfg["nz"])[d] * (cfg["nbx"], cfg["nby"], cfg["nbz"])[d]
    if gz < 0:
        return {0: gz % n, 1: 0, 2: -1 - gz}[cfg["bc_lo"][d]]
    if gz >= n:
        return {0: gz % n, 1: n - 1, 2: 2 * n - 1 - gz}[cfg["bc_hi"][d]]
    return gz


def remote_mask(cfg, part, rank):
    """[local box][k][j][i] -> True where the zone is a ghost whose source box belongs to another rank."""
    lc = shard.local_config(cfg, part)
    n = (cfg["nx"], cfg["ny"], cfg["nz"])
    lb = (lc["nbx"], lc["nby"], lc["nbz"])
    p = shard.rank_coords(part, rank)
    mask = np.zeros((lb[0] * lb[1] * lb[2], n[2] + 2 * NG, n[1] + 2 * NG, n[0] + 2 * NG), bool)
    for bk in range(lb[2]):
        for bj in range(lb[1]):
            for bi in range(lb[0]):
                b = bi + lb[0] * (bj + lb[1] * bk)
                own = []
                for d, l in enumerate((bi, bj, bk)):
                    gb = p[d] * lb[d] + l
                    src = np.array([brute_source(cfg, gb * n[d] + i - NG, d) // n[d] for i in range(n[d] + 2 * NG)])
                    own.append((src // lb[d]) == p[d])                     # source brick coordinate == mine
                local = own[2][:, None, None] & own[1][None, :, None] & own[0][None, None, :]
                mask[b] = ~local
    return mask


def run_plan_numpy(cfg, part, U_global_filled):
    """Executes the plan for every rank with numpy; returns per rank (U_local after unpack, coverage mask)."""
    world = part[0] * part[1] * part[2]
    lc = shard.local_config(cfg, part)
    loc = []
    for r in range(world):
        U = U_global_filled[shard.local_boxes(cfg, part, r)].copy()
        ghost = np.ones(U.shape, bool)
        ghost[:, :, NG:-NG, NG:-NG, NG:-NG] = False
        U[ghost] = np.nan                                                # only interiors are known before the exchange
        loc.append(U)
    N = wl.nvar(cfg)
    # pack
    msgs = {}
    for s in range(world):
        for seg in binding.exchange_plan(cfg, part, s, recv=False):
            ext = tuple(seg.ext)
            idx = [seg.lo[d] + seg.step[d] * np.arange(ext[d]) for d in range(3)]
            assert all((i >= NG).all() and (i < NG + (cfg["nx"], cfg["ny"], cfg["nz"])[d]).all() for d, i in enumerate(idx)), \
                "a source zone is not an interior zone"
            blk = loc[s][seg.box][:, idx[2][:, None, None], idx[1][None, :, None], idx[0][None, None, :]].copy()
            for d in range(3):
                if seg.flip[d]:
                    blk[1 + d] *= -1.0
            m = msgs.setdefault((s, seg.peer), {})
            assert seg.offset not in m
            m[seg.offset] = blk.ravel()
    out = []
    for r in range(world):
        U = loc[r]
        cover = np.zeros(U.shape[:1] + U.shape[2:], int)
        for seg in binding.exchange_plan(cfg, part, r, recv=True):
            data = msgs[(seg.peer, r)].pop(seg.offset)                   # same offset on both sides
            ext = tuple(seg.ext)
            assert data.size == N * ext[0] * ext[1] * ext[2] and tuple(seg.step) == (1, 1, 1)
            sl = tuple(slice(seg.lo[d], seg.lo[d] + ext[d]) for d in (2, 1, 0))
            U[seg.box][(slice(None),) + sl] = data.reshape(N, ext[2], ext[1], ext[0])
            cover[seg.box][sl] += 1
        out.append((U, cover))
    assert all(len(m) == 0 for m in msgs.values()), "a packed segment was never received"
    return out


CASES = [
    # (n, global lattice, bc per direction, partition)
    ((4, 5, 6), (2, 2, 2), (0, 0, 0), (2, 1, 1)),
    ((4, 5, 6), (2, 2, 2), (0, 0, 0), (2, 2, 2)),
    ((6, 4, 4), (4, 2, 1), (0, 1, 2), (2, 2, 1)),
    ((4, 4, 7), (2, 3, 4), (2, 0, 1), (1, 3, 2)),
    ((5, 4, 4), (4, 1, 2), (1, 2, 0), (4, 1, 1)),
    ((4, 4, 4), (3, 3, 3), (0, 0, 0), (3, 3, 3)),
    ((8, 4, 4), (2, 2, 4), (0, 0, 2), (1, 1, 1)),        # one rank: nothing is remote
]


@pytest.mark.parametrize("n,gnb,bc,part", CASES)
def test_plan_reproduces_the_global_ghost_fill(n, gnb, bc, part):
    cfg = small_cfg(n=n, nb=gnb, nspec=2, bc=bc)
    Ug = orc.fill_ghosts(cfg, wl.random_state(cfg, 31))
    for r, (U, cover) in enumerate(run_plan_numpy(cfg, part, Ug)):
        expect = Ug[shard.local_boxes(cfg, part, r)]
        remote = remote_mask(cfg, part, r)
        assert np.array_equal(cover == 1, remote), "the plan must cover exactly the ghost zones with a remote source, once"
        got = U[:, :, :, :, :]
        m5 = np.broadcast_to(remote[:, None], got.shape)
        assert np.array_equal(got[m5], expect[m5]), "exchanged ghost zones differ from the single-lattice fill"


@pytest.mark.parametrize("n,gnb,bc,part", CASES[:5])
def test_push_form_of_the_plan_reproduces_the_global_ghost_fill(n, gnb, bc, part):
    """The send segments also name the destination (rbox, rlo): executing them as direct stores into the peers' arrays
    (what cst_exchange_push does on the device) must give the same shells as pack + message + unpack."""
    cfg = small_cfg(n=n, nb=gnb, nspec=1, bc=bc)
    Ug = orc.fill_ghosts(cfg, wl.random_state(cfg, 33))
    world = part[0] * part[1] * part[2]
    loc = []
    for r in range(world):
        U = Ug[shard.local_boxes(cfg, part, r)].copy()
        U[np.broadcast_to(remote_mask(cfg, part, r)[:, None], U.shape)] = np.nan
        loc.append(U)
    for s in range(world):
        for seg in binding.exchange_plan(cfg, part, s, recv=False):
            ext = tuple(seg.ext)
            idx = [seg.lo[d] + seg.step[d] * np.arange(ext[d]) for d in range(3)]
            blk = loc[s][seg.box][:, idx[2][:, None, None], idx[1][None, :, None], idx[0][None, None, :]].copy()
            for d in range(3):
                if seg.flip[d]:
                    blk[1 + d] *= -1.0
            sl = tuple(slice(seg.rlo[d], seg.rlo[d] + ext[d]) for d in (2, 1, 0))
            loc[seg.peer][seg.rbox][(slice(None),) + sl] = blk
    for r in range(world):
        assert np.array_equal(loc[r], Ug[shard.local_boxes(cfg, part, r)]), r


def test_message_sizes_agree_between_the_two_sides():
    cfg = small_cfg(n=(4, 6, 5), nb=(4, 2, 2), nspec=1, bc=(0, 2, 1))
    part = (2, 2, 1)
    N = wl.nvar(cfg)
    size = lambda segs, peer: sum(N * s.ext[0] * s.ext[1] * s.ext[2] for s in segs if s.peer == peer)
    for a in range(4):
        for b in range(4):
            if a != b:
                assert size(binding.exchange_plan(cfg, part, a, False), b) == size(binding.exchange_plan(cfg, part, b, True), a)


def test_plan_rejects_bad_partitions():
    cfg = small_cfg(n=(4, 4, 4), nb=(3, 2, 2))
    with pytest.raises(binding.CstError):
        binding.exchange_plan(cfg, (2, 1, 1), 0, True)          # 3 boxes cannot be cut in two
    with pytest.raises(binding.CstError):
        binding.exchange_plan(cfg, (3, 1, 1), 3, True)          # rank out of range


def test_brick_partition():
    assert shard.brick_partition((16, 8, 4), 1) == (1, 1, 1)
    assert shard.brick_partition((16, 8, 4), 2) == (2, 1, 1)
    assert shard.brick_partition((16, 8, 4), 4) == (2, 2, 1)
    assert shard.brick_partition((16, 8, 4), 8) == (4, 2, 1)
    assert shard.brick_partition((2, 2, 2), 8) == (2, 2, 2)
    with pytest.raises(ValueError):
        shard.brick_partition((3, 1, 1), 2)
    seen = np.concatenate([shard.local_boxes(dict(nbx=4, nby=2, nbz=2), (2, 2, 1), r) for r in range(4)])
    assert sorted(seen) == list(range(16))


# ------------------------------------------------------------------ world size 2, gloo: the message plumbing ----
class NumpyBrickCtx:
    """Stand-in for binding.Context in the CPU test: the same five calls GhostExchange makes, executed with numpy
    from the library's host-side plan (the CUDA pack / unpack kernels are covered by tests/test_next_gpu_shard.py)."""

    def __init__(self, cfg_global, local_filled):
        self.cfg, self.local_filled = cfg_global, local_filled

    def set_sublattice(self, gnb, part, rank):
        self.part, self.rank = part, rank
        self.snd = binding.exchange_plan(self.cfg, part, rank, False)
        self.rcv = binding.exchange_plan(self.cfg, part, rank, True)
        N = wl.nvar(self.cfg)
        self.peers = sorted({s.peer for s in self.snd} | {s.peer for s in self.rcv})
        ln = lambda segs, p: sum(N * s.ext[0] * s.ext[1] * s.ext[2] for s in segs if s.peer == p)
        self.sl = [ln(self.snd, p) for p in self.peers]
        self.rl = [ln(self.rcv, p) for p in self.peers]

    def exchange_info(self):
        so = np.concatenate([[0], np.cumsum(self.sl)[:-1]]).astype(int)
        ro = np.concatenate([[0], np.cumsum(self.rl)[:-1]]).astype(int)
        return [(p, int(so[i]), self.sl[i], int(ro[i]), self.rl[i]) for i, p in enumerate(self.peers)]

    def fill_ghosts(self, U, stream=None):
        pass                                                      # local-source ghosts: not under test here

    def exchange_pack(self, U, buf, stream=None):
        base = {i[0]: i[1] for i in self.exchange_info()}
        Un = U.numpy()
        for s in self.snd:
            idx = [s.lo[d] + s.step[d] * np.arange(s.ext[d]) for d in range(3)]
            blk = Un[s.box][:, idx[2][:, None, None], idx[1][None, :, None], idx[0][None, None, :]].copy()
            for d in range(3):
                if s.flip[d]:
                    blk[1 + d] *= -1.0
            o = base[s.peer] + s.offset
            buf.numpy()[o:o + blk.size] = blk.ravel()

    def exchange_unpack(self, U, buf, stream=None):
        base = {i[0]: i[3] for i in self.exchange_info()}
        N = wl.nvar(self.cfg)
        for s in self.rcv:
            n = N * s.ext[0] * s.ext[1] * s.ext[2]
            o = base[s.peer] + s.offset
            sl = tuple(slice(s.lo[d], s.lo[d] + s.ext[d]) for d in (2, 1, 0))
            U.numpy()[s.box][(slice(None),) + sl] = buf.numpy()[o:o + n].reshape(N, s.ext[2], s.ext[1], s.ext[0])


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = small_cfg(n=(4, 5, 6), nb=(2, 2, 1), nspec=1, bc=(0, 2, 1))
    part = shard.brick_partition((2, 2, 1), world)
    Ug = orc.fill_ghosts(cfg, wl.random_state(cfg, 32))
    expect = Ug[shard.local_boxes(cfg, part, rank)]
    U = torch.from_numpy(expect.copy())
    ghost = torch.ones(U.shape, dtype=torch.bool)
    ghost[:, :, NG:-NG, NG:-NG, NG:-NG] = False
    remote = torch.from_numpy(np.broadcast_to(remote_mask(cfg, part, rank)[:, None], U.shape).copy())
    U[remote] = float("nan")                                      # what the exchange has to deliver
    ex = shard.GhostExchange(NumpyBrickCtx(cfg, expect), cfg, part, rank, lambda n: torch.zeros(n, dtype=torch.float64))
    ex.fill_ghosts(U)
    dtmin = shard.allreduce_min(0.1 * (rank + 1), "cpu")
    out.put((rank, bool(np.array_equal(U.numpy(), expect)), int(remote.sum()), dtmin))
    dist.destroy_process_group()


def test_two_rank_ghost_exchange_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + (os.getpid() + 7) % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, same, nremote, dtmin in res:
        assert same and nremote > 0 and dtmin == 0.1
