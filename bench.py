#!/usr/bin/env python
"""bench.py -- zone-updates/s of the fp64 A(U)+SDC hot path on B200 (BASELINE.json metric).

One "step" = one pass of the whole hot path over the workload:
    cst_fill_ghosts(U) -> cst_advance_A_update(U -> A_new, U_next) -> cst_cfl_dt_device(U)
with the state not evolving between steps (outputs go to second buffers), inputs resident in HBM.
Default run: BASELINE.json configs[3] (512^3 periodic box, NVAR = 18) is the headline line, and -- after its
buffers are freed -- configs[4] (the XRB-shaped batch of 512 boxes of 64^3) is timed the same way and reported
inside the same line under "also" (both halves of the north-star target get a number from one driver run).
--workload K times configs[K] only.  Prints ONE JSON line (rank 0).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 3|4] [--impl ours|reference]
Multi-GPU (launched by torchrun, one rank per GPU): the box lattice is SHARDED over the ranks in equal bricks
(strong scaling: the global domain is fixed; paper_1910_12578_b200/shard.py, csrc/exchange.cu).  configs[3]'s 512^3
domain is then a 2 x 2 x 2 lattice of 256^3 boxes, configs[4] keeps its 16 x 8 x 4 boxes of 64^3.  Per step every rank
fills its local ghost zones, exchanges the 4-deep shells on its brick surface with the neighbouring ranks
(NCCL send/recv), advances its boxes and MIN-reduces dt; `value` = zones of the whole domain / max-over-ranks time.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time
from concurrent.futures import ThreadPoolExecutor

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1910_12578_b200 import workloads as wl  # noqa: E402

METRIC = "zone-updates/s of fp64 A(U)+SDC update"
UNIT = "zone-updates/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", type=int, default=None, choices=[0, 1, 2, 3, 4],
                    help="time this config only (default: configs[3], then configs[4] under \"also\")")
    ap.add_argument("--n", type=int, default=None, help="override zones per box side (debug only; marks the line)")
    ap.add_argument("--no-tune", action="store_true", help="keep species-kernel variant 0 instead of timing the variants")
    ap.add_argument("--probe", action="store_true",
                    help="(internal) child process: check every tunable configuration bitwise against variant 0, print one JSON line")
    ap.add_argument("--exchange", default="sendrecv", choices=["sendrecv", "p2p"],
                    help="multi-GPU ghost exchange: NCCL send/recv of packed messages, or direct stores into peer-mapped memory")
    ap.add_argument("--next", action="store_true",
                    help="time the kernels of the rows beyond S0-S6 (reactions, diffusion, flattening, fourth order, CTU) "
                         "on configs[3]'s distribution at 256^3 instead of the headline path; one JSON line, 1 GPU")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


# ------------------------------------------------------------------------------------ bytes ----
def alg_bytes(cfg):
    """Algorithmic bytes per zone-update, strict count."""
    ng, nx, ny, nz, N = cfg["ng"], cfg["nx"], cfg["ny"], cfg["nz"], wl.nvar(cfg)
    G = (nx + 2 * ng) * (ny + 2 * ng) * (nz + 2 * ng) / (nx * ny * nz)
    G3 = 1.0 + 6.0 * (1.0 / nx + 1.0 / ny + 1.0 / nz)
    fill = 2.0 * (G - 1.0) * N * 8.0                 # read source + write ghost, full shell
    adv = (G3 + 4.0) * N * 8.0                       # U (+3-deep face ghosts), A_old^m, A_old^other, A_new, U_next
    cfl = 5.0 * 8.0                                  # hydro components of the interior
    # the advance runs as two kernels: the 5 hydro components and the nspec species components
    return dict(fill=fill, advance=adv, cfl=cfl, step=fill + adv + cfl, balg=fill + adv, G=G, G3=G3,
                advance_hydro=(G3 + 4.0) * 5 * 8.0, advance_species=(G3 + 4.0) * (N - 5) * 8.0)


def measured_peaks():
    try:
        mp = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        return float(mp["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ----------------------------------------------------------------------------------- inputs ----
def fill_host_state(cfg, U_host_np, threads=8, brick=None):
    """Seeded synthetic state of the config, plane by plane, into the host array (ghosts zero).  brick = (origin,
    lattice) in box coordinates: only that rank's boxes (the planes are generated for the global domain)."""
    Dz = wl.domain(cfg)[2]
    planes = range(Dz) if brick is None else range(brick[0][2] * cfg["nz"], (brick[0][2] + brick[1][2]) * cfg["nz"])

    def one(kg):
        wl.scatter_plane(cfg, U_host_np, kg, wl.cons_plane(cfg, kg), brick)
    with ThreadPoolExecutor(threads) as ex:
        list(ex.map(one, planes))


def host_mem_available():
    """Bytes of host memory this process may still take (MemAvailable, capped by the cgroup limit)."""
    avail = 1 << 62
    try:
        for line in open("/proc/meminfo"):
            if line.startswith("MemAvailable"):
                avail = int(line.split()[1]) * 1024
    except Exception:
        pass
    try:
        lim = open("/sys/fs/cgroup/memory.max").read().strip()
        cur = int(open("/sys/fs/cgroup/memory.current").read().strip())
        if lim != "max":
            avail = min(avail, int(lim) - cur)
    except Exception:
        pass
    return avail


# ----------------------------------------------------------------------------------- clocks ----
class ClockSampler:
    FIELDS = ["clocks.sm", "clocks.max.sm", "power.draw", "clocks_event_reasons.hw_slowdown",
              "clocks_event_reasons.hw_thermal_slowdown", "clocks_event_reasons.sw_thermal_slowdown",
              "clocks_event_reasons.sw_power_cap"]

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(index), "--query-gpu=" + ",".join(self.FIELDS),
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if t0 <= t <= t1 + 0.1] or [r for (_, r) in self.rows]
        sm, mx, reasons = [], [], set()
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# ------------------------------------------------------------------------------ CPU baseline ----
def oracle_sample_cfg(cfg):
    """A bounded sample of the same workload for the CPU oracle (~10-30 s of CPU work)."""
    if cfg["index"] == 4:
        c = wl.make_config(4, n=(cfg["nx"], cfg["ny"], cfg["nz"]), nb=(2, 2, cfg["nbz"]), nspec=cfg["nspec"])
        what = f"{c['nbx'] * c['nby'] * c['nbz']} of the {cfg['nbx'] * cfg['nby'] * cfg['nbz']} boxes (2x2 columns, full height)"
    else:
        n = min(cfg["nx"], 144)
        c = wl.make_config(cfg["index"], n=n, nspec=cfg["nspec"])
        what = f"same input distribution on a {n}^3 box ({n ** 3 / (cfg['nx'] * cfg['ny'] * cfg['nz']):.3f} of the zones)"
    return c, what


def time_oracle(cfg, steps, warmup):
    from oracle import orc   # the one other place the oracle may run: the timed CPU baseline
    c, what = oracle_sample_cfg(cfg)
    U = wl.initial_state(c, ghost_value=0.0)
    Un = U.copy()
    A_old0, A_old1 = np.zeros(wl.a_shape(c)), np.zeros(wl.a_shape(c))
    times = []
    for s in range(warmup + steps):
        t0 = time.perf_counter()
        orc.fill_ghosts(c, U)
        dt = orc.cfl_dt(c, U, 0.5)
        A = orc.advance_A(c, U)
        orc.sdc_update(c, Un, U, dt, A, A_old0, [A_old0, A_old1], [0.5 * dt, 0.5 * dt])
        if s >= warmup:
            times.append(time.perf_counter() - t0)
    zones = wl.nzones(c)
    return dict(value=zones / float(np.mean(times)), unit=UNIT, cores=orc.num_threads(), kind="oracle",
                sample=what + f"; {steps} timed passes of fill_ghosts+cfl+A+update, {zones} zones each"), float(np.mean(times))


def run_reference(args, cfg, rank):
    if rank != 0:
        return
    steps, warmup = max(1, min(args.steps, 3)), max(0, min(args.warmup, 1))
    cb, sec = time_oracle(cfg, steps, warmup)
    line = {"impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
            "scaling": "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"configs[{cfg['index']}] {cfg['name']} (bounded sample: {cb['sample']})"},
            "cpu_baseline": cb,
            "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------- multi-rank ----
def allreduce_scalar(x, op, device, world):
    """MIN / MAX of a host scalar over the ranks (dt: MIN, device time: MAX).  The path shards as
    independent replicas of the box lattice: these two scalars are the only
    things that cross ranks.  Works with any torch.distributed backend (nccl on GPUs, gloo in tests)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MIN if op == "min" else dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(zones_per_rank, world, ms_step_max):
    """whole-job zone-updates/s: every rank advances its own zones_per_rank zones (its brick of the sharded
    lattice) in ms_step_max, the slowest rank's time."""
    return zones_per_rank * world / (ms_step_max * 1e-3)


def sharded_config(cfg, world):
    """The config a multi-rank run shards (same global domain and seeded state as the single-GPU workload) and its
    partition into bricks.  configs[3]'s single 512^3 box becomes 2 x 2 x 2 boxes of 256^3 (a box is the unit of
    distribution); the batched configs keep their lattice."""
    from paper_1910_12578_b200 import shard
    if cfg["nbx"] * cfg["nby"] * cfg["nbz"] == 1 and world > 1:
        f = 2 if world <= 8 else 4
        cfg = wl.make_config(cfg["index"], n=(cfg["nx"] // f, cfg["ny"] // f, cfg["nz"] // f), nb=(f, f, f), nspec=cfg["nspec"])
    part = shard.brick_partition((cfg["nbx"], cfg["nby"], cfg["nbz"]), world)
    return cfg, part


# -------------------------------------------------------------------------------------- main ----
def probe_child():
    """Runs in a CHILD process before anything is timed (see probe_configurations): on two reduced versions of the timed
    workloads -- configs[3] as one 128 x 128 x 64 box, configs[4] as 2 x 2 x 2 boxes of 64^3 -- every configuration the tuner
    may pick (species variants 1-3, 2 / 3 / 4 CTAs per tile, the CFL reduction folded into the advance) must reproduce
    variant 0 with the separate CFL pass BIT FOR BIT.  Prints {"variants_ok": b, "fused_cfl_ok": b, ...}.  The product
    path only: no oracle here (the oracle comparison of the same configurations is tests/test_next_gpu_variants.py)."""
    import torch
    from paper_1910_12578_b200 import Context
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    out = {"variants_ok": True, "fused_cfl_ok": True, "checked": 0, "failed": []}
    for index, kw in ((3, {"n": (128, 128, 64)}), (4, {"nb": (2, 2, 2)})):
        cfg = wl.make_config(index, **kw)
        U_host = np.zeros(wl.u_shape(cfg))
        fill_host_state(cfg, U_host)
        U = torch.from_numpy(U_host).to(dev)
        ctx = Context(cfg)
        ctx.fill_ghosts(U)
        dt_dev = torch.zeros(1, dtype=torch.float64, device=dev)
        ctx.cfl_dt_device(U, 0.5, dt_dev)
        dt_ref = float(dt_dev.cpu()[0])
        A0 = torch.zeros(wl.a_shape(cfg), dtype=torch.float64, device=dev)
        ctx.advance_A(U, A0)
        A1 = A0 * 0.9
        w = [0.5 * dt_ref, 0.5 * dt_ref]

        def run(variant, split, fused):
            ctx.set_variant(variant)
            ctx.set_species_split(split)
            A = torch.full_like(A0, 7.0)
            Un = U.clone()
            dt_f = None
            if fused:
                dt_dev.zero_()
                ctx.advance_A_update_cfl(U, A, Un, dt_ref, A0, [A0, A1], w, 0.5, dt_dev)
                dt_f = float(dt_dev.cpu()[0])
            else:
                ctx.advance_A_update(U, A, Un, dt_ref, A0, [A0, A1], w)
            torch.cuda.synchronize()
            return A, Un, dt_f

        A_ref, Un_ref, _ = run(0, 3, False)
        if not bool(torch.isfinite(A_ref).all()):
            raise SystemExit("probe: variant 0 gave a non-finite A")
        for variant in (0, 1, 2, 3):
            for split in (2, 3, 4):
                for fused in (False, True):
                    if (variant, split, fused) == (0, 3, False):
                        continue
                    A, Un, dt_f = run(variant, split, fused)
                    same = torch.equal(A, A_ref) and torch.equal(Un, Un_ref)
                    if fused:
                        same = same and dt_f is not None and abs(dt_f - dt_ref) <= 1e-14 * dt_ref
                    out["checked"] += 1
                    if not same:
                        out["failed"].append([cfg["name"], variant, split, fused])
                        if fused:
                            out["fused_cfl_ok"] = False
                        else:
                            out["variants_ok"] = False
        ctx.destroy()
    print("PROBE " + json.dumps(out), flush=True)


def probe_configurations(local):
    """None of the tunable configurations (cst_tune_advance's variants, the fused CFL step) is ever timed unless a child
    process has first run all of them on THIS device and found them bit-identical to the default path: a kernel fault
    in a variant then ends the child, not the benchmark, and the timed run keeps variant 0 with the separate CFL pass."""
    bad = {"variants_ok": False, "fused_cfl_ok": False}
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    env["LOCAL_RANK"] = str(local)
    try:
        r = subprocess.run([sys.executable, os.path.abspath(__file__), "--probe"], env=env, capture_output=True, text=True, timeout=420)
    except Exception as exc:
        return dict(bad, note=f"probe did not finish ({type(exc).__name__}); default path only")
    for ln in r.stdout.splitlines():
        if ln.startswith("PROBE "):
            res = json.loads(ln[6:])
            res["note"] = "every tunable configuration checked bitwise against variant 0 in a child process on this device"
            return res
    tail = (r.stderr or "").strip().splitlines()[-1:] or [""]
    return dict(bad, note=f"probe exited {r.returncode} ({tail[0][:200]}); default path only")


def measure(cfg, args, rank, world, local, dev, want_e2e, want_cpu_baseline):
    """Times one workload (W warm-up + K timed steps) and returns the JSON line as a dict (rank 0; None elsewhere).
    Every device buffer is local to this function, so the memory is free again when it returns."""
    import torch
    import torch.distributed as dist
    from paper_1910_12578_b200 import Context

    from paper_1910_12578_b200 import shard
    gcfg, part, brick = cfg, (1, 1, 1), None          # gcfg: the global lattice; cfg: this rank's brick of it
    if world > 1:
        gcfg, part = sharded_config(cfg, world)
        cfg = shard.local_config(gcfg, part)
        pc = shard.rank_coords(part, rank)
        lat = (cfg["nbx"], cfg["nby"], cfg["nbz"])
        brick = (tuple(pc[d] * lat[d] for d in range(3)), lat)
    ctx = Context(cfg)
    ctx_sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    N, zones = wl.nvar(cfg), wl.nzones(cfg)
    ushape, ashape = wl.u_shape(cfg), wl.a_shape(cfg)
    ubytes, abytes = int(np.prod(ushape)) * 8, int(np.prod(ashape)) * 8

    # ---- host input (pinned if possible), seeded + synthetic --------------------------------
    pinned = True
    try:
        U_host = torch.zeros(ushape, dtype=torch.float64, pin_memory=True)
    except Exception:
        pinned = False
        U_host = torch.zeros(ushape, dtype=torch.float64)
    fill_host_state(gcfg, U_host.numpy(), brick=brick)

    U = torch.empty(ushape, dtype=torch.float64, device=dev)
    U.copy_(U_host, non_blocking=True)
    U_next = U.clone()
    A_new = torch.empty(ashape, dtype=torch.float64, device=dev)
    A_old0 = torch.zeros(ashape, dtype=torch.float64, device=dev)
    A_old1 = torch.zeros(ashape, dtype=torch.float64, device=dev)
    dt_dev = torch.zeros(1, dtype=torch.float64, device=dev)
    ex = None
    if world > 1:                 # ghost zones with a source on another rank travel through NCCL send/recv
        mode = getattr(args, "exchange", "sendrecv")
        ex = shard.GhostExchange(ctx, gcfg, part, rank, lambda n: torch.empty(n, dtype=torch.float64, device=dev), mode=mode)
        if mode == "p2p":
            ex.register(U)          # IPC handles of U to the peers; raises if the allocation cannot be shared
    fill = (lambda: ex.fill_ghosts(U)) if ex else (lambda: ctx.fill_ghosts(U))
    fill()
    dt = ctx.cfl_dt(U, 0.5)
    dt = allreduce_scalar(dt, "min", dev, world)
    # A_old buffers hold plausible values: A of the initial state and a perturbation of it
    ctx.advance_A(U, A_old0)
    A_old1.copy_(A_old0).mul_(0.9)
    w = [0.5 * dt, 0.5 * dt]

    # kernel variants of the species half (cst_tune_advance): every variant is timed on these buffers before the
    # warm-up steps and the fastest is kept; all variants give bit-identical results (tests/test_next_gpu_variants.py)
    tuned = {"species_variant": 0, "ms": None, "note": "not tuned"}
    safe = getattr(args, "safe", {"variants_ok": False, "fused_cfl_ok": False})
    if not safe["variants_ok"]:
        tuned["note"] = "not tuned: " + str(safe.get("note", "no probe"))
    if not getattr(args, "no_tune", False) and N > 5 and safe["variants_ok"]:
        try:
            for _ in range(3):      # clocks and caches warm before the first variant is timed (variant 0 goes first)
                ctx.advance_A_update(U, A_new, U_next, dt, A_old0, [A_old0, A_old1], w)
            v, ms_v = ctx.tune_advance(U, A_new, U_next, dt, A_old0, [A_old0, A_old1], w, repeats=2)
            tuned = {"species_variant": v, "species_split": ctx.get_species_split() or 3, "ms": ms_v,
                     "note": "cst_tune_advance: ms of the fused advance (hydro + species kernels), min of 2 runs: variants "
                             "0, 1, 2, 3 with three CTAs per tile, then the winner with 2 and 4"}
        except Exception as exc:
            ctx.set_variant(0)
            tuned = {"species_variant": 0, "ms": None, "note": f"tuning failed ({exc}); variant 0"}

    ev = lambda: torch.cuda.Event(enable_timing=True)
    k_ev, k_ms2 = [], []
    ctx.set_timing(True)      # CUDA events around the two kernels of the advance, on this stream (cst.h)

    step_ev = []
    fused_cfl = {"on": False, "ms_separate": None, "ms_fused": None}

    def step(timed):
        if timed:
            step_ev.append(ev()); step_ev[-1].record()
        fill()
        if timed:
            e0, e1 = ev(), ev()
            e0.record()
        if fused_cfl["on"]:       # S1-S6 in one call: the CFL max is gathered inside the hydro kernel's z sweep
            ctx.advance_A_update_cfl(U, A_new, U_next, dt, A_old0, [A_old0, A_old1], w, 0.5, dt_dev)
        else:
            ctx.advance_A_update(U, A_new, U_next, dt, A_old0, [A_old0, A_old1], w)
        if timed:
            e1.record()
            k_ev.append((e0, e1))
        if not fused_cfl["on"]:
            ctx.cfl_dt_device(U, 0.5, dt_dev)
        if world > 1:
            dist.all_reduce(dt_dev, op=dist.ReduceOp.MIN)

    def sync_all():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    if not getattr(args, "no_tune", False) and safe["fused_cfl_ok"]:
        # the step with the CFL reduction folded into the advance against the step with the separate CFL pass: 3 runs each
        # after one untimed run, the faster composition is kept (same results: tests/test_next_gpu_variants.py)
        try:
            for key, on in (("ms_separate", False), ("ms_fused", True)):
                fused_cfl["on"] = on
                step(False)
                torch.cuda.synchronize()
                t0e, t1e = ev(), ev()
                t0e.record()
                for _ in range(3):
                    step(False)
                t1e.record()
                torch.cuda.synchronize()
                fused_cfl[key] = t0e.elapsed_time(t1e) / 3
            fused_cfl["on"] = fused_cfl["ms_fused"] < fused_cfl["ms_separate"]
        except Exception as exc:
            fused_cfl.update(on=False, note=f"comparison failed ({exc})")
        if world > 1:             # every rank must run the same composition: all take rank 0's choice
            flag = torch.tensor([1.0 if fused_cfl["on"] else 0.0], dtype=torch.float64, device=dev)
            dist.broadcast(flag, 0)
            fused_cfl["on"] = bool(flag.item() > 0.5)
    for _ in range(args.warmup):
        step(False)
    sync_all()
    sampler = ClockSampler(local) if rank == 0 else None
    l0 = ctx.launch_count()
    t_wall0 = time.time()
    s0, s1 = ev(), ev()
    s0.record()
    for _ in range(args.steps):
        step(True)
    s1.record()
    sync_all()
    k_ms2.append(ctx.last_advance_ms())      # (hydro, species) of the last timed step
    t_wall1 = time.time()
    launches = ctx.launch_count() - l0
    ms = s0.elapsed_time(s1)
    ms = allreduce_scalar(ms, "max", dev, world)
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    ms_step = ms / args.steps
    per_step = [a.elapsed_time(b) for a, b in zip(step_ev, step_ev[1:] + [s1])]
    value = aggregate_value(zones, world, ms_step)
    k_ms = float(np.mean([a.elapsed_time(b) for a, b in k_ev]))

    # ---- roofline of the dominant kernel: k_advect_species (the species components of the fused
    #      A + node update); k_advect_hydro and the whole advance call are reported beside it
    ab = alg_bytes(cfg)
    peak, peak_src = measured_peaks()
    ms_hydro, ms_species = k_ms2[-1]
    traffic, prof = None, {}
    try:
        prof = json.load(open(os.path.join(ROOT, "profiles", "traffic.json"))).get(f"configs[{cfg['index']}]", {})
        traffic = prof.get("k_advect_species_dram_bytes_per_launch")
    except Exception:
        pass
    if tuned["species_variant"] != 0 or args.n:
        # the ncu annotations were captured on variant 0 of the species kernel at full size: they do not describe this run
        traffic = None
        prof = {k: v for k, v in prof.items() if "species" not in k}
    if N > 5:
        vname = "k_advect_species_tma<2>" if tuned["species_variant"] == 0 else f"k_advect_species_tma_v<2, {tuned['species_variant']}>"
        dom, dom_ms, dom_bytes = f"{vname} (S1-S5, species components)", ms_species, ab["advance_species"]
    else:
        dom, dom_ms, dom_bytes = "k_advect_hydro<2> (S1-S5, hydro components)", ms_hydro, ab["advance_hydro"]
    achieved = dom_bytes * zones / (dom_ms * 1e-3) / 1e9
    # `frac` is the dominant KERNEL's (the contract's roofline entry).  The figure the north-star's 0.60 target is read
    # against is whole_step_frac_balg: SURVEY 8(d)'s B_alg (ghost fill + fused advance, no CFL bytes) x zones / step time.
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak,
                "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                "traffic_source": "static annotation: ncu --set full capture of this kernel, profiles/traffic.json "
                                  "(not measured in this run)",
                "peak_source": peak_src, "alg_bytes_per_zone": dom_bytes, "kernel_ms": dom_ms,
                "other_kernels": {"k_advect_hydro_ms": ms_hydro, "k_advect_species_ms": ms_species,
                                  "advance_call_ms": k_ms,
                                  "advance_call_frac": ab["advance"] * zones / (k_ms * 1e-3) / 1e9 / peak},
                "whole_step_frac_balg": ab["balg"] * zones / (ms_step * 1e-3) / 1e9 / peak,
                "balg_bytes_per_zone": ab["balg"],
                "whole_step_frac_with_cfl_bytes": ab["step"] * zones / (ms_step * 1e-3) / 1e9 / peak}
    # second roof (BASELINE.json north_star: "the slower of bytes/HBM bandwidth and FP64 flops/peak"): instruction issue
    # and the FP64 pipe.  Instruction counts per launch are STATIC ncu annotations (profiles/traffic.json); the peaks are
    # SMs x 4 schedulers x SM clock (issue) and SMs x 64 FP64 lanes x SM clock (FP64 instructions).
    sm_hz = (clocks or {}).get("sm_mhz") or 1965.0
    issue_peak = ctx_sm_count * 4 * sm_hz * 1e6
    fp64_peak = ctx_sm_count * 64 * sm_hz * 1e6
    if prof.get("k_advect_species_warp_instr_per_launch") and prof.get("k_advect_hydro_warp_instr_per_launch"):
        roofline["issue"] = {
            "k_advect_species_issue_frac": prof["k_advect_species_warp_instr_per_launch"] / (ms_species * 1e-3) / issue_peak,
            "k_advect_hydro_issue_frac": prof["k_advect_hydro_warp_instr_per_launch"] / (ms_hydro * 1e-3) / issue_peak,
            "fp64_pipe_active_pct_ncu": {"species": prof.get("k_advect_species_fp64_pipe_active_pct_ncu"),
                                         "hydro": prof.get("k_advect_hydro_fp64_pipe_active_pct_ncu")},
            "source": "static annotation (ncu counts in profiles/traffic.json), not measured in this run"}
        if prof.get("k_advect_species_fp64_thread_instr_per_launch"):
            roofline["issue"]["k_advect_species_fp64_frac"] = \
                prof["k_advect_species_fp64_thread_instr_per_launch"] / (ms_species * 1e-3) / fp64_peak

    # ---- end to end through the C ABI with HOST buffers (H2D + D2H inside the timed region) --
    e2e = None
    need = 2 * ubytes + abytes
    if want_e2e and host_mem_available() < 1.3 * (need - ubytes) + 8e9:
        e2e = {"value": None, "unit": UNIT, "skipped": f"host has {host_mem_available() / 1e9:.0f} GB available, "
               f"needs {need / 1e9:.0f} GB of host buffers"}
    elif want_e2e:
        try:
            A_host = torch.empty(ashape, dtype=torch.float64, pin_memory=pinned)
            Un_host = torch.empty(ushape, dtype=torch.float64, pin_memory=pinned)
        except Exception:
            pinned = False
            A_host = torch.empty(ashape, dtype=torch.float64)
            Un_host = torch.empty(ushape, dtype=torch.float64)
        n_e2e = max(1, min(args.steps, 2))

        def host_step():
            if ex is None:                  # one C-ABI call with HOST buffers
                ctx.step_host(U_host, A_host, Un_host, U, U_next, A_new, dt)
            else:                           # sharded: the same sequence with the ghost exchange between H2D and the advance
                U.copy_(U_host, non_blocking=True)
                ex.fill_ghosts(U)
                ctx.advance_A_update(U, A_new, U_next, dt, A_new, [A_new, A_new], w)
                A_host.copy_(A_new, non_blocking=True)
                Un_host.copy_(U_next, non_blocking=True)
                torch.cuda.synchronize()
        host_step()                         # warm-up
        sync_all()
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            host_step()
        sync_all()
        sec = (time.perf_counter() - t0) / n_e2e
        sec = allreduce_scalar(sec, "max", dev, world)
        e2e = {"value": zones * world / sec, "unit": UNIT, "h2d_bytes_per_step": ubytes * world,
               "d2h_bytes_per_step": (abytes + ubytes) * world, "steps": n_e2e, "host_memory": "pinned" if pinned else "pageable",
               "call": "cst_step_host (H2D U, fill_ghosts, advance_A_update, D2H A and U_next)" if ex is None else
                       "H2D U, fill_ghosts + ghost exchange, cst_advance_A_update, D2H A and U_next (per rank, its brick)"}
        del A_host, Un_host

    cpu_baseline = None
    if rank == 0 and world == 1 and want_cpu_baseline:
        cpu_baseline, _ = time_oracle(cfg, 3, 1)

    line = None
    if rank == 0:
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": f"configs[{gcfg['index']}] {gcfg['name']}: {gcfg['nbx'] * gcfg['nby'] * gcfg['nbz']} box(es) of "
                                       f"{gcfg['nx']}x{gcfg['ny']}x{gcfg['nz']}+{gcfg['ng']} ghosts, NVAR={N}",
                           "zones_per_gpu": zones, "zones_total": zones * world,
                           "step": ("fill_ghosts + advance_A_update_cfl" if fused_cfl["on"] else
                                    "fill_ghosts + advance_A_update + cfl_dt_device") if ex is None else
                                   ("fill_ghosts + exchange_pack + NCCL send/recv + exchange_unpack" if ex.mode == "sendrecv" else
                                    "barrier + fill_ghosts + exchange_push (stores into peer-mapped memory) + barrier")
                                   + " + advance_A_update + cfl_dt_device + all_reduce(MIN) of dt",
                           "ghost_exchange_bytes_per_rank_per_step": ex.bytes_per_fill if ex else 0,
                           "l2": f"inputs larger than L2 ({(ubytes + 3 * abytes) / 1e9:.1f} GB touched per step)"
                                 if ubytes > 4e8 else "inputs fit in L2 (debug size)",
                           "parallelism": f"box lattice sharded over {world} ranks, bricks {part[0]}x{part[1]}x{part[2]}" if world > 1
                                          else "single GPU",
                           "ms_per_step_best": float(min(per_step)), "ms_per_step_median": float(np.median(per_step)),
                           "tuned": tuned, "fused_cfl": fused_cfl, "probe": safe, "debug_size_override": bool(args.n)},
                "clocks": clocks, "e2e": e2e, "gpu_launches": launches, "roofline": roofline,
                "cpu_baseline": cpu_baseline}
    ctx.destroy()
    return line


def measure_next(args, dev):
    """--next: each operator of SURVEY 8(f) on one mid-size box (configs[3]'s distribution, 256^3 by default, NVAR = 18),
    device-resident, CUDA events, with the strict algorithmic byte count (what the operator must read and write once)
    beside the time, and the oracle's twin timed on a 48^3 sample.  None of these kernels is tuned: the fractions say
    how far the straightforward multi-pass versions are from a fused treatment."""
    import torch
    from paper_1910_12578_b200 import Context
    from oracle import orc
    n = args.n or 256
    cfg = wl.make_config(3, n=n)
    N, zones = wl.nvar(cfg), wl.nzones(cfg)
    peak, peak_src = measured_peaks()
    U_host = torch.zeros(wl.u_shape(cfg), dtype=torch.float64)
    fill_host_state(cfg, U_host.numpy())
    U = U_host.to(dev)
    mk = lambda: torch.zeros(wl.a_shape(cfg), dtype=torch.float64, device=dev)
    A, A2, R, R2 = mk(), mk(), mk(), mk()
    Un = U.clone()
    scfg = wl.make_config(3, n=48)
    Us = orc.fill_ghosts(scfg, wl.initial_state(scfg))
    react = wl.react_params(cfg["nspec"])
    Zs = np.zeros(wl.a_shape(scfg))
    ev = lambda: torch.cuda.Event(enable_timing=True)
    out = {}

    def timed(name, fn, alg_bytes_per_zone, oracle_fn, launches_ctx):
        for _ in range(max(1, args.warmup)):
            fn()
        torch.cuda.synchronize()
        l0 = launches_ctx.launch_count()
        e0, e1 = ev(), ev()
        e0.record()
        for _ in range(args.steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.steps
        t0 = time.perf_counter()
        oracle_fn()
        sec = time.perf_counter() - t0
        gbs = alg_bytes_per_zone * zones / (ms * 1e-3) / 1e9
        out[name] = {"ms": ms, "zone_updates_per_s": zones / (ms * 1e-3), "alg_bytes_per_zone": alg_bytes_per_zone,
                     "achieved_gbs": gbs, "frac_of_hbm_peak": gbs / peak,
                     "launches_per_call": (launches_ctx.launch_count() - l0) // args.steps,
                     "oracle_zone_updates_per_s": wl.nzones(scfg) / sec}

    ctx = Context(cfg)
    ctx.fill_ghosts(U)
    dt = ctx.cfl_dt(U, 0.5)
    ctx.advance_A(U, A)
    # NEXT-3: the implicit node update (reads U_m, A_new, A_old, R_old, 2 x (A_q + R_q); writes U_next, R_new)
    ctx.set_reactions(react)
    ctx.react_R(U, R)
    timed("sdc_update_react", lambda: ctx.sdc_update_react(Un, U, dt, A, A, R, [A, A], [R, R], [0.5 * dt, 0.5 * dt], R2),
          10 * N * 8, lambda: orc.sdc_update_react(scfg, react, Us.copy(), Us, 1e-3, Zs, Zs, orc.react_R(scfg, react, Us),
                                                   [Zs, Zs], [Zs, Zs], [5e-4, 5e-4]), ctx)
    # NEXT-4: the diffusion term alone = (A with it) - (A without it): time both, report the difference
    timed("advance_A (reference point: second-order path)", lambda: ctx.advance_A(U, A2), 2 * N * 8,
          lambda: orc.advance_A(scfg, Us), ctx)
    ctx.set_diffusion(0.01, 1.5)
    timed("advance_A + diffusion", lambda: ctx.advance_A(U, A2), 2 * N * 8 , lambda: orc.advance_A_diffuse(scfg, 0.01, 1.5, Us), ctx)
    ctx.set_diffusion(0.0, 1.5)
    ctx.destroy()
    del ctx
    # NEXT-2 (i): flattening (general kernels)
    ctx = Context(cfg, workspace=None)
    ctx.set_flattening(True)
    ctx.set_workspace(torch.empty(ctx.workspace_bytes(), dtype=torch.uint8, device=dev))
    timed("advance_A + flattening", lambda: ctx.advance_A(U, A2), 2 * N * 8, lambda: orc.advance_A_flat(scfg, Us), ctx)
    ctx.destroy()
    del ctx
    torch.cuda.empty_cache()
    # NEXT-1: fourth order
    ctx = Context(cfg, workspace=None)
    ctx.set_order(4)
    ws = torch.empty(ctx.workspace_bytes(), dtype=torch.uint8, device=dev)
    ctx.set_workspace(ws)
    timed("advance_A order 4", lambda: ctx.advance_A(U, A2), 2 * N * 8, lambda: orc.advance_A4(scfg, Us), ctx)
    ctx.destroy()
    del ctx, ws
    torch.cuda.empty_cache()
    # NEXT-2 (ii): CTU
    ctx = Context(cfg)
    ws = torch.empty(ctx.ctu_workspace_bytes(), dtype=torch.uint8, device=dev)
    timed("advance_ctu", lambda: ctx.advance_ctu(U, dt, A2, ws), 2 * N * 8, lambda: orc.advance_ctu(scfg, Us, 1e-3), ctx)
    ctx.destroy()
    return {"metric": "kernels of the rows beyond S0-S6 (SURVEY 8(f)): ms per call, zone-updates/s, strict algorithmic bytes",
            "unit": "ms", "n_gpus": 1, "steps": args.steps, "warmup": max(1, args.warmup), "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"configs[3] distribution on one {n}^3 box, NVAR={N}", "zones": zones,
                       "oracle_sample": "48^3 box, one call, all host threads"},
            "peak_gbs": peak, "peak_source": peak_src, "kernels": out}


def main():
    args = parse()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    head = 3 if args.workload is None else args.workload
    cfg = wl.make_config(head, n=args.n) if args.n else wl.make_config(head)

    if args.probe:
        probe_child()
        return
    if args.impl == "reference":
        run_reference(args, cfg, rank)
        return

    import torch
    import torch.distributed as dist

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    args.safe = {"variants_ok": False, "fused_cfl_ok": False, "note": "not probed"}
    if not args.no_tune and not getattr(args, "next", False):
        args.safe = probe_configurations(local)       # a child process per rank, before this one has a CUDA context
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
        for key in ("variants_ok", "fused_cfl_ok"):   # a configuration is used only if every rank's device passed it
            args.safe[key] = bool(allreduce_scalar(1.0 if args.safe[key] else 0.0, "min", dev, world) > 0.5)

    if getattr(args, "next", False):
        if rank == 0:
            print(json.dumps(measure_next(args, dev)), flush=True)
        if world > 1:
            dist.destroy_process_group()
        return

    line = measure(cfg, args, rank, world, local, dev, not args.no_e2e, not args.no_cpu_baseline)
    if args.workload is None and not args.n:
        # second half of the north-star target: the batched-box config, same protocol, device-resident numbers only
        import gc
        gc.collect()
        torch.cuda.empty_cache()
        try:
            also = measure(wl.make_config(4), args, rank, world, local, dev, False, False)
            if rank == 0:
                keep = ("value", "unit", "ms_per_step", "steps", "warmup", "config", "clocks", "gpu_launches", "roofline")
                line["also"] = {"configs[4]": {k: also[k] for k in keep}}
        except Exception as exc:    # the headline line must still be printed
            if rank == 0:
                line["also"] = {"configs[4]": {"error": f"{type(exc).__name__}: {exc}"}}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
