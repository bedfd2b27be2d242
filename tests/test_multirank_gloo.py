"""The N > 1 path of bench.py on CPU: world_size 2, gloo.  The path shards as independent replicas
(DESIGN.md section 9); the only cross-rank traffic is MIN of dt and MAX of the device time."""
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
