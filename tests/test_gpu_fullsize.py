"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (the fused
cst_advance_A_update with two distinct A_old arrays), on SAMPLED outputs: sub-boxes of the domain
are cut out of the GPU's ghost-filled state (with their 4-deep halo), the oracle evaluates A and the
node update on each sub-box as a stand-alone box, and the GPU's A / U_next are compared there.
Gate as everywhere: per component max|gpu - orc| / max|orc| <= 1e-12 (over the sampled zones)."""
import numpy as np
import pytest
import torch

from oracle import orc
from paper_1910_12578_b200 import Context, workloads as wl

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
TOL = 1e-12


def need_gb(gb):
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < gb * 1e9:
        pytest.skip(f"needs {gb} GB of free device memory, has {free / 1e9:.0f}")


def device_state(cfg):
    """Seeded state of the config, built plane by plane straight into device memory."""
    U = torch.zeros(wl.u_shape(cfg), dtype=torch.float64, device=DEV)
    for kg in range(wl.domain(cfg)[2]):
        wl.scatter_plane(cfg, U, kg, torch.from_numpy(wl.cons_plane(cfg, kg)).to(DEV))
    return U


def check_samples(cfg, samples, sub=16):
    """samples: list of (box, k0, j0, i0) interior origins of sub x sub x sub sub-boxes."""
    ctx = Context(cfg)
    U = device_state(cfg)
    ctx.fill_ghosts(U)
    dt = ctx.cfl_dt(U, 0.5)
    ash = wl.a_shape(cfg)
    A, A0, A1 = (torch.empty(ash, dtype=torch.float64, device=DEV) for _ in range(3))
    ctx.advance_A(U, A0)                       # plausible A_old values, as in bench.py
    A1.copy_(A0).mul_(0.9)
    Un = torch.zeros_like(U)
    w = [0.5 * dt, 0.5 * dt]
    ctx.advance_A_update(U, A, Un, dt, A0, [A0, A1], w)
    torch.cuda.synchronize()
    N, ng = wl.nvar(cfg), 4
    sc = dict(cfg, nx=sub, ny=sub, nz=sub, nbx=1, nby=1, nbz=1)
    numA, denA, numU, denU = (np.zeros(N) for _ in range(4))
    for (b, k0, j0, i0) in samples:
        Us = U[b, :, k0:k0 + sub + 2 * ng, j0:j0 + sub + 2 * ng, i0:i0 + sub + 2 * ng].cpu().numpy()[None].copy()
        sl = (b, slice(None), slice(k0, k0 + sub), slice(j0, j0 + sub), slice(i0, i0 + sub))
        Ao = orc.advance_A(sc, Us)
        Ag, A0s, A1s = (x[sl].cpu().numpy()[None] for x in (A, A0, A1))
        # the GPU's A_old0 was computed by the GPU; the update is checked from bit-identical inputs
        Uno = Us.copy()
        orc.sdc_update(sc, Uno, Us, dt, Ao, A0s, [A0s, A1s], w)
        Ung = Un[b, :, k0 + ng:k0 + ng + sub, j0 + ng:j0 + ng + sub, i0 + ng:i0 + ng + sub].cpu().numpy()
        Uni = Uno[0, :, ng:ng + sub, ng:ng + sub, ng:ng + sub]
        ax = (1, 2, 3)
        numA = np.maximum(numA, np.abs(Ag[0] - Ao[0]).max(axis=ax)); denA = np.maximum(denA, np.abs(Ao[0]).max(axis=ax))
        numU = np.maximum(numU, np.abs(Ung - Uni).max(axis=ax)); denU = np.maximum(denU, np.abs(Uni).max(axis=ax))
    eA, eU = (numA / denA).max(), (numU / denU).max()
    print(cfg["name"], "sampled sub-boxes", len(samples), "A err", eA, "U_next err", eU)
    assert eA <= TOL and eU <= TOL, (numA / denA, numU / denU)
    ctx.destroy()


def test_configs3_512_sampled():
    need_gb(110)
    cfg = wl.make_config(3)
    s = [(0, 0, 0, 0), (0, 496, 496, 496), (0, 248, 8, 496), (0, 100, 300, 16), (0, 8, 250, 250), (0, 333, 77, 129)]
    check_samples(cfg, s)


def test_configs4_boxes_sampled():
    need_gb(122)
    cfg = wl.make_config(4)
    # boxes at the reflecting z walls, at periodic x/y wraps and in the interior; sub-boxes touching box faces
    s = [(0, 0, 0, 0), (511, 48, 48, 48), (16 * 8 * 3 + 5, 48, 0, 20), (130, 20, 48, 0), (257, 24, 24, 24), (15, 0, 30, 48)]
    check_samples(cfg, s)


def test_configs2_256_sampled():
    need_gb(8)
    cfg = wl.make_config(2)
    s = [(0, 120, 120, 120), (0, 0, 0, 0), (0, 240, 240, 240), (0, 128, 100, 150), (0, 112, 128, 128)]
    check_samples(cfg, s)


def test_configs1_128_sampled():
    cfg = wl.make_config(1)
    s = [(0, 56, 56, 56), (0, 0, 0, 0), (0, 112, 112, 112), (0, 40, 60, 80)]
    check_samples(cfg, s)
