"""Flow running into reflecting walls faster than the PVRS shock speed (reading Q6b), for every operator.

The two states of a reflecting-wall face are exact mirror images (u_L = -u_R, all else equal), so the numerator of S*
cancels EXACTLY: S* = 0 and the left state is the upwind one.  Where S_L > 0 > S_R both sides are "pure" and the two
candidate fluxes differ by O(1): the choice must be taken on the exactly cancelling sum, which needs (a) the two
products of the numerator rounded separately (hydro.cuh hllc, hllc_ieee) and (b) every operation before the Riemann
solve to treat the two mirror images alike (ctu.cu and fourth.cu are compiled without FMA contraction for this).
Found without a GPU by compiling the kernels on the host with and without contraction; collected after every other
`-m gpu` file (these cases have never run on a B200, and the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

from oracle import orc
from paper_1910_12578_b200 import Context, workloads as wl
from test_gpu_parity import check_one_call_set
from test_next_gpu_ctu import run_ctu
from test_next_gpu_flatten import flat_ctx
from test_next_gpu_fourth import ctx4
from test_oracle_ctu import cfl_dt_ctu
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


def wall_state(cfg, seed, speed=4.0):
    """noise + a flow of the given speed (c ~ 1.3: Mach ~ 3 by default) that runs away from the centre of the domain,
    i.e. INTO the wall on all six sides"""
    G = wl.to_global(cfg, wl.random_state(cfg, seed, amp=0.15), ghosted=True)
    rho = G[0].copy()
    for d in range(3):
        n = G.shape[3 - d]
        x = (np.arange(n) + 0.5) / n
        shape = [1, 1, 1]; shape[2 - d] = n
        mom = G[1 + d] + speed * rho * np.tanh(6.0 * (x - 0.5)).reshape(shape)
        G[4] += 0.5 * (mom ** 2 - G[1 + d] ** 2) / rho                            # keep the pressure
        G[1 + d] = mom
    return wl.from_global(cfg, G)


def wall_ties(cfg, U):
    """number of wall faces (x direction, low side) where the PVRS speeds give S_L > 0 > S_R for the mirror-image pair
    of first-order states: the faces on which the side the S* test picks changes the flux by O(1)"""
    Uo = orc.fill_ghosts(cfg, U.copy())
    g, ng, count = cfg["gamma"], cfg["ng"], 0
    for k in range(ng, ng + cfg["nz"]):
        for j in range(ng, ng + cfg["ny"]):
            W = orc.cons_to_prim(g, cfg["small_pres"], Uo[0][:, k, j, ng])
            ps = orc.pvrs_pstar(g, W[0], -W[1], W[4], W[0], W[1], W[4])
            SL, SR = orc.wave_speeds(g, W[0], -W[1], W[4], W[0], W[1], W[4], ps)
            count += (SL > 0.0) and (SR < 0.0)
    return count


@pytest.mark.parametrize("n,nb,ns", [((32, 16, 16), (1, 1, 1), 2),     # full tiles: the fast paths
                                     ((20, 9, 12), (1, 1, 1), 1),      # ragged tiles: the general kernels
                                     ((16, 16, 16), (2, 1, 2), 0)])    # walls on some sides of each box only
def test_supersonic_flow_into_reflecting_walls(n, nb, ns):
    """The two states of a reflecting-wall face are exact mirror images (u_L = -u_R, all else equal), so the numerator of
    S* cancels EXACTLY: S* = 0 and the left state is the upwind one (S* >= 0).  Where the flow runs into the wall faster
    than the PVRS shock speed, S_L > 0 > S_R, both sides are "pure" and the two candidate fluxes differ by O(1): the
    choice must be taken on the exactly cancelling sum, not on the rounding error of a fused multiply-add (hydro.cuh
    hllc: the products are rounded separately)."""
    cfg = small_cfg(n=n, nb=nb, nspec=ns, gamma=5 / 3, bc=(2, 2, 2))
    U = wall_state(cfg, 77)
    assert wall_ties(cfg, U) > 10, "the state must put S_L > 0 > S_R on wall faces"
    res = check_one_call_set(cfg, U)
    print("walls", n, nb, res)


@pytest.mark.parametrize("n,nb", [((16, 16, 16), (1, 1, 1)), ((20, 9, 12), (1, 1, 1))])
def test_flattened_A_with_flow_running_into_reflecting_walls(n, nb):
    """with flattening the wall zones sit behind a strong compression: chi = 0, first-order mirror-image states"""
    cfg = small_cfg(n=n, nb=nb, nspec=2, gamma=5 / 3, bc=(2, 2, 2))
    U0 = wall_state(cfg, 77)
    assert wall_ties(cfg, U0) > 10
    U = orc.fill_ghosts(cfg, U0)
    Ao = orc.advance_A_flat(cfg, U)
    assert comp_err(Ao, orc.advance_A(cfg, U)).max() > 1e-2, "flattening must be active"
    ctx = flat_ctx(cfg)
    Ad = torch.full(wl.a_shape(cfg), float("nan"), dtype=torch.float64, device=DEV)
    ctx.advance_A(dev(U), Ad)
    eA = comp_err(Ad.cpu().numpy(), Ao)
    assert eA.max() <= TOL, eA
    ctx.destroy()


@pytest.mark.parametrize("n,nb,ns,speed", [((16, 12, 10), (1, 1, 1), 1, 4.0), ((8, 16, 8), (2, 1, 1), 2, 2.5)])
def test_ctu_with_flow_running_into_reflecting_walls(n, nb, ns, speed):
    """Mirror-image states on the wall faces with S_L > 0 > S_R: the upwind side hangs on an exactly cancelling sum
    (reading Q6b); the tracing and the transverse corrections of the two mirror images must round alike --
    ctu.cu is compiled without FMA contraction for this (build.py PER_FILE)."""
    cfg = small_cfg(n=n, nb=nb, nspec=ns, gamma=5 / 3, bc=(2, 2, 2))
    U0 = wall_state(cfg, 77, speed=speed)
    assert wall_ties(cfg, U0) > 10
    U = orc.fill_ghosts(cfg, U0)
    dt = cfl_dt_ctu(cfg, U, 0.7)
    Ao = orc.advance_ctu(cfg, U, dt)
    assert np.isfinite(Ao).all()
    ctx = Context(cfg)
    e = comp_err(run_ctu(ctx, cfg, U, dt), Ao)
    assert e.max() <= TOL, e
    ctx.destroy()


@pytest.mark.parametrize("n,nb,seed", [((16, 12, 10), (1, 1, 1), 77), ((12, 16, 10), (2, 1, 1), 78)])
def test_A4_with_flow_running_into_reflecting_walls(n, nb, seed):
    """Mirror-image states on the wall faces, S_L > 0 > S_R on many of them: the upwind side hangs on an exactly
    cancelling sum (reading Q6b), so every operation before the Riemann solve has to treat the two mirror
    images alike -- fourth.cu is compiled without FMA contraction for this (build.py PER_FILE)."""
    cfg = small_cfg(n=n, nb=nb, nspec=1, gamma=5 / 3, bc=(2, 2, 2))
    U0 = wall_state(cfg, seed, speed=2.2)
    assert wall_ties(cfg, U0) > 5
    U = orc.fill_ghosts(cfg, U0)
    Ao = orc.advance_A4(cfg, U)
    assert np.isfinite(Ao).all()
    ctx = ctx4(cfg)
    Ad = torch.full(wl.a_shape(cfg), float("nan"), dtype=torch.float64, device=DEV)
    ctx.advance_A(dev(U), Ad)
    eA = comp_err(Ad.cpu().numpy(), Ao)
    assert eA.max() <= TOL, eA
    ctx.destroy()
