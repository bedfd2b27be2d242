"""Parity of the fourth-order finite-volume <A(U)> (include/cst.h cst_set_order(ctx, 4)) with the
oracle's orc_advance_A4 from bit-identical inputs, and the paper's fourth-order scheme (3 Simpson nodes, 4 iterations)
assembled from library calls against the oracle's driver."""
import numpy as np
import pytest
import torch

from oracle import orc
from paper_1910_12578_b200 import Context, CstError, sdc_step_nodes, workloads as wl
from test_oracle_pins import small_cfg

pytestmark = pytest.mark.gpu
TOL = 1e-12
DEV = "cuda:0"


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def comp_err(gpu, ref):
    axes = (0, 2, 3, 4)
    num, den = np.abs(gpu - ref).max(axis=axes), np.abs(ref).max(axis=axes)
    return np.where(den > 0, num / np.where(den > 0, den, 1.0), num)


def stepped_state(cfg, seed):
    """Mild white noise times piecewise-constant density / pressure plateaux (contrast 4) and velocity jumps: every
    branch of the limiter fires, yet U^c = <U> - Lap<U>/24 stays a physical state."""
    Dx, Dy, Dz = wl.domain(cfg)
    G = wl.to_global(cfg, wl.random_state(cfg, seed, amp=0.1), ghosted=True)
    z, y, x = np.meshgrid(np.arange(Dz), np.arange(Dy), np.arange(Dx), indexing="ij")
    w = lambda D, k: max(D // k, 4)                                    # plateaux at least four zones wide
    fr = np.where((x // w(Dx, 3) + y // w(Dy, 2)) % 2 == 0, 1.0, 4.0)
    fp = np.where((y // w(Dy, 3) + z // w(Dz, 2) + x // w(Dx, 2)) % 2 == 0, 1.0, 4.0)
    rho, v = G[0] * fr, G[1:4] / G[0] + 0.5 * np.where(x > Dx // 2, -1.0, 1.0)
    p = (cfg["gamma"] - 1) * (G[4] - 0.5 * (G[1:4] ** 2).sum(axis=0) / G[0]) * fp
    W = np.concatenate([rho[None], v, p[None], G[5:] / G[0]])
    return wl.from_global(cfg, wl.cons_from_prim(cfg, W))


def ctx4(cfg):
    ctx = Context(cfg, workspace=None)
    with pytest.raises(CstError):
        ctx.set_order(3)
    ctx.set_order(4)
    ctx.set_workspace(torch.empty(ctx.workspace_bytes(), dtype=torch.uint8, device=DEV))
    return ctx


@pytest.mark.parametrize("n,nb,ns,bc,state", [
    ((16, 16, 16), (1, 1, 1), 2, (0, 0, 0), "noise"),
    ((20, 9, 12), (1, 1, 1), 13, (1, 2, 0), "noise"),          # the paper's species count; outflow / reflecting shells
    ((8, 6, 5), (2, 2, 1), 1, (2, 0, 1), "shocks"),            # box lattice, strong jumps: every limiter branch
    ((24, 4, 4), (1, 1, 1), 0, (1, 0, 0), "shocks"),
    ((4, 4, 4), (1, 1, 2), 3, (0, 0, 0), "noise"),             # minimum size
])
def test_A4_matches_oracle(n, nb, ns, bc, state):
    cfg = small_cfg(n=n, nb=nb, nspec=ns, gamma=1.4, bc=bc, grav=(0.05, 0.0, -0.1))
    if state == "noise":
        U = orc.fill_ghosts(cfg, wl.random_state(cfg, 101))
    else:
        U = orc.fill_ghosts(cfg, stepped_state(cfg, 102))
    Ao = orc.advance_A4(cfg, U)
    assert np.isfinite(Ao).all()
    assert comp_err(Ao, orc.advance_A(cfg, U)).max() > 1e-3           # a different operator from the PPM path
    ctx = ctx4(cfg)
    Ud = dev(U)
    Ad = torch.full(wl.a_shape(cfg), float("nan"), dtype=torch.float64, device=DEV)
    ctx.advance_A(Ud, Ad)
    eA = comp_err(Ad.cpu().numpy(), Ao)
    assert eA.max() <= TOL, eA
    print("A4 error", eA.max())
    # the "fused" call: A4 followed by the plain node update
    dt = 0.3 * orc.cfl_dt(cfg, U, 0.5)
    rng = np.random.default_rng(5)
    Aold = Ao + 0.1 * rng.standard_normal(Ao.shape) * np.abs(Ao).max()
    Uno = np.full_like(U, 3.0)
    orc.sdc_update(cfg, Uno, U, dt, Ao, Aold, [Aold, Ao], [0.25 * dt, 0.75 * dt])
    Af, Uf = torch.empty_like(Ad), torch.full(wl.u_shape(cfg), 3.0, dtype=torch.float64, device=DEV)
    Aoldd = dev(Aold)
    ctx.advance_A_update(Ud, Af, Uf, dt, Aoldd, [Aoldd, Af], [0.25 * dt, 0.75 * dt])
    assert comp_err(Af.cpu().numpy(), Ao).max() <= TOL
    assert comp_err(Uf.cpu().numpy(), Uno).max() <= 10 * TOL
    ctx.destroy()


def test_fourth_order_sdc_step_matches_oracle_driver():
    """Simpson nodes + A4 = the paper's fourth-order scheme, one step, GPU driver against the oracle's."""
    cfg = small_cfg(n=(12, 8, 8), nspec=1, gamma=5 / 3)
    U0 = wl.random_state(cfg, 103, amp=0.1)
    dt = orc.cfl_dt(cfg, orc.fill_ghosts(cfg, U0.copy()), 0.5)
    Uo = orc.sdc_step_nodes(cfg, U0, dt, M=3, K=4, A_fn=lambda V: orc.advance_A4(cfg, V))
    ctx = ctx4(cfg)
    Ud = dev(np.nan_to_num(U0, nan=0.0))
    sdc_step_nodes(ctx, Ud, dt, M=3, K=4)
    I = (slice(None), slice(None), slice(4, -4), slice(4, -4), slice(4, -4))
    e = comp_err(Ud.cpu().numpy()[I], Uo[I])
    assert e.max() <= 10 * TOL, e
    ctx.destroy()
