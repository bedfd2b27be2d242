"""The sharded box lattice on ONE GPU: every rank of a partition is a separate Context holding its brick; the
messages that NCCL would carry are copied between the ranks' send / receive buffers here (kernels that wait on one
another are never launched, /opt/skills B200 recipe).  After the exchange every rank's ghost shell must equal the
oracle's fill of the whole lattice bit for bit, and <A(U)> + the node update evaluated per rank must equal the
single-lattice evaluation BITWISE (a box never sees which rank it lives on).  SURVEY 8(e)."""
import numpy as np
import pytest
import torch

from oracle import orc
from paper_1910_12578_b200 import Context, CstError, shard, workloads as wl
from test_oracle_pins import small_cfg

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def sharded_fill(cfg, part, U_host):
    """-> list per rank of (ctx, U_local on the device, filled through local fill + pack / copy / unpack)."""
    world = part[0] * part[1] * part[2]
    lc = shard.local_config(cfg, part)
    ranks = []
    for r in range(world):
        ctx = Context(lc)
        ctx.set_sublattice((cfg["nbx"], cfg["nby"], cfg["nbz"]), part, r)
        info = ctx.exchange_info()
        U = dev(U_host[shard.local_boxes(cfg, part, r)])
        snd = torch.full((max(1, sum(i[2] for i in info)),), float("nan"), dtype=torch.float64, device=DEV)
        rcv = torch.full((max(1, sum(i[4] for i in info)),), float("nan"), dtype=torch.float64, device=DEV)
        ctx.fill_ghosts(U)
        ctx.exchange_pack(U, snd)
        ranks.append(dict(ctx=ctx, U=U, info=info, snd=snd, rcv=rcv))
    torch.cuda.synchronize()
    for r, me in enumerate(ranks):                 # the transport: peer p's message for me -> my receive buffer
        for peer, so, sl, ro, rl in me["info"]:
            src = ranks[peer]
            pso, psl = next((i[1], i[2]) for i in src["info"] if i[0] == r)
            assert psl == rl
            me["rcv"][ro:ro + rl].copy_(src["snd"][pso:pso + psl])
    for me in ranks:
        me["ctx"].exchange_unpack(me["U"], me["rcv"])
    torch.cuda.synchronize()
    return ranks


@pytest.mark.parametrize("n,gnb,bc,part,nspec", [
    ((16, 16, 16), (2, 2, 2), (0, 0, 0), (2, 1, 1), 3),         # full tiles: the TMA species kernel
    ((8, 6, 5), (2, 2, 2), (0, 0, 0), (2, 2, 2), 2),
    ((6, 4, 4), (4, 2, 1), (0, 1, 2), (2, 2, 1), 1),
    ((4, 4, 7), (2, 3, 4), (2, 0, 1), (1, 3, 2), 0),
    ((5, 4, 4), (4, 1, 2), (1, 2, 0), (4, 1, 1), 2),
])
def test_sharded_lattice_equals_single_lattice_bitwise(n, gnb, bc, part, nspec):
    cfg = small_cfg(n=n, nb=gnb, nspec=nspec, bc=bc, gamma=5 / 3, grav=(0.0, 0.1, -0.3))
    U_host = wl.random_state(cfg, 41)
    Uo = orc.fill_ghosts(cfg, U_host.copy())
    # single lattice on the device
    ctx1 = Context(cfg)
    U1 = dev(U_host)
    ctx1.fill_ghosts(U1)
    assert np.array_equal(U1.cpu().numpy(), Uo)
    dt = ctx1.cfl_dt(U1, 0.5)
    A1 = torch.full(wl.a_shape(cfg), float("nan"), dtype=torch.float64, device=DEV)
    Un1 = torch.full(wl.u_shape(cfg), 7.0, dtype=torch.float64, device=DEV)
    ctx1.advance_A_update(U1, A1, Un1, dt, A1, [A1, A1], [0.5 * dt, 0.5 * dt])
    A1h, Un1h = A1.cpu().numpy(), Un1.cpu().numpy()
    # the same lattice cut into bricks
    dts = []
    for r, me in enumerate(sharded_fill(cfg, part, U_host)):
        boxes = shard.local_boxes(cfg, part, r)
        assert np.array_equal(me["U"].cpu().numpy(), Uo[boxes]), f"rank {r}: ghost shell differs from the global fill"
        ctx, U = me["ctx"], me["U"]
        dts.append(ctx.cfl_dt(U, 0.5))
        lc = shard.local_config(cfg, part)
        A = torch.full(wl.a_shape(lc), float("nan"), dtype=torch.float64, device=DEV)
        Un = torch.full(wl.u_shape(lc), 7.0, dtype=torch.float64, device=DEV)
        ctx.advance_A_update(U, A, Un, dt, A, [A, A], [0.5 * dt, 0.5 * dt])
        assert np.array_equal(A.cpu().numpy(), A1h[boxes]), f"rank {r}: A differs from the single-lattice A"
        assert np.array_equal(Un.cpu().numpy(), Un1h[boxes])
        ctx.destroy()
    assert min(dts) == dt                                   # MIN over ranks of the local CFL steps
    ctx1.destroy()


@pytest.mark.parametrize("n,gnb,bc,part", [
    ((8, 6, 5), (2, 2, 2), (0, 0, 0), (2, 2, 2)),
    ((6, 4, 4), (4, 2, 1), (0, 1, 2), (2, 2, 1)),
    ((4, 4, 7), (2, 3, 4), (2, 0, 1), (1, 3, 2)),
])
def test_push_exchange_through_peer_pointers_equals_global_fill(n, gnb, bc, part):
    """cst_exchange_push: every rank stores straight into the other ranks' arrays (here all in one process, so the
    "peer-mapped" pointers are the arrays themselves); no buffers, no unpack."""
    cfg = small_cfg(n=n, nb=gnb, nspec=2, bc=bc)
    U_host = wl.random_state(cfg, 42)
    Uo = orc.fill_ghosts(cfg, U_host.copy())
    world = part[0] * part[1] * part[2]
    lc = shard.local_config(cfg, part)
    ranks = []
    for r in range(world):
        ctx = Context(lc)
        ctx.set_sublattice((cfg["nbx"], cfg["nby"], cfg["nbz"]), part, r)
        ranks.append(dict(ctx=ctx, U=dev(U_host[shard.local_boxes(cfg, part, r)])))
    for me in ranks:
        me["ctx"].fill_ghosts(me["U"])
    torch.cuda.synchronize()
    for me in ranks:
        peers = [ranks[i[0]]["U"] for i in me["ctx"].exchange_info()]
        me["ctx"].exchange_push(me["U"], peers)
    torch.cuda.synchronize()
    for r, me in enumerate(ranks):
        assert np.array_equal(me["U"].cpu().numpy(), Uo[shard.local_boxes(cfg, part, r)]), f"rank {r}"
        with pytest.raises(CstError):
            me["ctx"].exchange_push(me["U"], [])                 # wrong number of peers
        me["ctx"].destroy()


def test_sublattice_errors():
    cfg = small_cfg(n=(4, 4, 4), nb=(2, 1, 1))
    ctx = Context(cfg)
    with pytest.raises(CstError):
        ctx.exchange_info()                                 # no plan yet
    with pytest.raises(CstError):
        ctx.set_sublattice((3, 1, 1), (2, 1, 1), 0)         # 3 boxes cannot be cut in two
    with pytest.raises(CstError):
        ctx.set_sublattice((4, 1, 1), (4, 1, 1), 0)         # brick (1,1,1) != the context's lattice (2,1,1)
    with pytest.raises(CstError):
        ctx.set_sublattice((4, 1, 1), (2, 1, 1), 2)         # rank out of range
    ctx.set_sublattice((4, 1, 1), (2, 1, 1), 1)
    assert [i[0] for i in ctx.exchange_info()] == [0]       # periodic x: both neighbours are rank 0
    ctx.destroy()
