"""Parity of the unsplit CTU PPM operator (include/cst.h cst_advance_ctu) with the oracle's
orc_advance_ctu from bit-identical inputs, and the exact one-zone shift at unit CFL on the GPU itself."""
import numpy as np
import pytest
import torch

from oracle import orc
from paper_1910_12578_b200 import Context, CstError, workloads as wl
from test_oracle_pins import small_cfg
from test_oracle_ctu import cfl_dt_ctu

pytestmark = pytest.mark.gpu
TOL = 1e-12
DEV = "cuda:0"


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def comp_err(gpu, ref):
    axes = (0, 2, 3, 4)
    num, den = np.abs(gpu - ref).max(axis=axes), np.abs(ref).max(axis=axes)
    return np.where(den > 0, num / np.where(den > 0, den, 1.0), num)


def run_ctu(ctx, cfg, U, dt):
    ws = torch.empty(ctx.ctu_workspace_bytes(), dtype=torch.uint8, device=DEV)
    A = torch.full(wl.a_shape(cfg), float("nan"), dtype=torch.float64, device=DEV)
    ctx.advance_ctu(dev(U), dt, A, ws)
    return A.cpu().numpy()


@pytest.mark.parametrize("n,nb,ns,bc,amp", [
    ((16, 16, 16), (1, 1, 1), 2, (0, 0, 0), 0.3),
    ((20, 9, 12), (1, 1, 1), 13, (1, 2, 0), 0.3),             # the paper's species count; outflow / reflecting shells
    ((8, 6, 5), (2, 2, 1), 1, (2, 0, 1), 0.6),                # box lattice; supersonic zones (every tracing branch)
    ((24, 4, 4), (1, 1, 1), 0, (1, 0, 0), 0.6),
    ((4, 4, 4), (1, 1, 2), 3, (0, 0, 0), 0.3),                # minimum size
])
def test_ctu_matches_oracle(n, nb, ns, bc, amp):
    cfg = small_cfg(n=n, nb=nb, nspec=ns, gamma=1.4, bc=bc, grav=(0.05, 0.0, -0.1))
    U = orc.fill_ghosts(cfg, wl.random_state(cfg, 131, amp=amp))
    ctx = Context(cfg)
    for cfl in (0.8, 0.3):
        dt = cfl_dt_ctu(cfg, U, cfl)
        Ao = orc.advance_ctu(cfg, U, dt)
        assert np.isfinite(Ao).all()
        e = comp_err(run_ctu(ctx, cfg, U, dt), Ao)
        assert e.max() <= TOL, (cfl, e)
    with pytest.raises(CstError):
        ctx.advance_ctu(dev(U), 0.01, torch.empty(wl.a_shape(cfg), dtype=torch.float64, device=DEV),
                        torch.empty(16, dtype=torch.uint8, device=DEV))                        # workspace too small
    ctx.destroy()


def test_unit_cfl_advection_is_an_exact_shift_on_the_gpu():
    rng = np.random.default_rng(3)
    n = (16, 12, 8)
    cfg = small_cfg(n=n, nspec=2, gamma=1.4)
    dt = 0.05
    W = np.zeros((7, n[2], n[1], n[0]))
    W[0] = np.exp(0.5 * rng.standard_normal(W[0].shape))
    W[1], W[2], W[3] = cfg["dx"] / dt, cfg["dy"] / dt, cfg["dz"] / dt
    W[4] = 1.0
    W[5] = rng.random(W[0].shape)
    W[6] = 1 - W[5]
    Ug = wl.cons_from_prim(cfg, W)
    ctx = Context(cfg)
    A = wl.to_global(cfg, run_ctu(ctx, cfg, orc.fill_ghosts(cfg, wl.from_global(cfg, Ug)), dt))
    exact = (np.roll(Ug, (1, 1, 1), axis=(1, 2, 3)) - Ug) / dt
    assert np.abs(A - exact).max() <= 1e-13 * np.abs(exact).max()
    ctx.destroy()
