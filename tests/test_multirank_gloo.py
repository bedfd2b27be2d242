"""The N > 1 path of bench.py on CPU: world_size 2, gloo.  The box lattice is sharded over the ranks (DESIGN.md
section 9): the scalar reductions (MIN of dt, MAX of the device time), the sharded workload and each rank's share of
the seeded input are checked here; the ghost exchange itself in tests/test_shard_plan.py (gloo) and
tests/test_next_gpu_shard.py (kernels)."""
import os
import sys

import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    dt = bench.allreduce_scalar(0.01 * (rank + 1), "min", "cpu", world)
    ms = bench.allreduce_scalar(10.0 + rank, "max", "cpu", world)
    out.put((rank, dt, ms, bench.aggregate_value(1000, world, ms)))
    dist.destroy_process_group()


def test_two_rank_reductions_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for rank, dt, ms, val in res:
        assert dt == 0.01 and ms == 11.0              # MIN over ranks, MAX over ranks
        assert abs(val - 2 * 1000 / 11e-3) < 1e-6     # both ranks' zones over the slowest rank's time


def test_single_rank_is_identity():
    import bench
    assert bench.allreduce_scalar(3.5, "min", "cpu", 1) == 3.5
    assert bench.aggregate_value(10, 1, 1.0) == 10 / 1e-3


def test_sharded_workloads_keep_the_domain_and_the_state():
    """bench.py's multi-rank workloads: same global domain as the single-GPU config, equal bricks, and every rank's
    host input is exactly its boxes of the global seeded state."""
    import numpy as np
    import bench
    from paper_1910_12578_b200 import shard, workloads as wl
    g3, part3 = bench.sharded_config(wl.make_config(3), 8)
    assert wl.domain(g3) == (512, 512, 512) and (g3["nbx"], g3["nby"], g3["nbz"]) == (2, 2, 2) and part3 == (2, 2, 2)
    assert g3["dx"] == wl.make_config(3)["dx"]
    g4, part4 = bench.sharded_config(wl.make_config(4), 4)
    assert (g4["nbx"], g4["nby"], g4["nbz"]) == (16, 8, 4) and part4 == (2, 2, 1)
    # small version: the single box and its 2x2x2 decomposition hold the same zones
    one = wl.make_config(3, n=16, nspec=2)
    g, part = bench.sharded_config(one, 2)
    assert wl.domain(g) == wl.domain(one) and part == (2, 1, 1)
    G1 = wl.to_global(one, wl.initial_state(one), ghosted=True)
    full = wl.initial_state(g)
    assert np.array_equal(wl.to_global(g, full, ghosted=True), G1)
    for rank in range(2):
        lc = shard.local_config(g, part)
        pc = shard.rank_coords(part, rank)
        lat = (lc["nbx"], lc["nby"], lc["nbz"])
        U = np.zeros(wl.u_shape(lc))
        bench.fill_host_state(g, U, threads=2, brick=(tuple(pc[d] * lat[d] for d in range(3)), lat))
        ref = np.nan_to_num(full[shard.local_boxes(g, part, rank)], nan=0.0)
        assert np.array_equal(U, ref)


def test_probe_falls_back_to_the_default_path_when_the_child_fails():
    """bench.probe_configurations: the tunable configurations (species variants, fused CFL) are offered to the timed run
    only if a child process has checked them on the device; a child that cannot run (here: no GPU) must leave both off
    with a note, never raise."""
    import torch
    import bench
    res = bench.probe_configurations(0)
    assert isinstance(res["variants_ok"], bool) and isinstance(res["fused_cfl_ok"], bool) and res["note"]
    if not torch.cuda.is_available():
        assert res["variants_ok"] is False and res["fused_cfl_ok"] is False
        assert "default path only" in res["note"]
