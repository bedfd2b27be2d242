"""Pins of the oracle's optional shock flattening (oracle/orc.c S2b, readings F1-F4; CW84 appendix; SURVEY 8(f)
NEXT-2 (i)).  No test here calls the CUDA path."""
import os

import numpy as np
import pytest

from oracle import orc
from paper_1910_12578_b200 import workloads as wl
from test_oracle_pins import small_cfg, relmax
from test_oracle_scheme import uniform_W, state_from_prims

GOLD = os.path.join(os.path.dirname(__file__), "golden")


# ---------------------------------------------------------------- F1-F2 on hand-computed lines ----
def test_line_coefficients_worked_out_by_hand():
    # a three-zone compression shock: zone 5 has z = 9/9 = 1 -> zeta = 0; its neighbours have z <= 2/3 -> zeta = 1
    p = np.array([1, 1, 1, 1, 1, 4, 10, 10, 10, 10, 10, 10], float)
    u = np.array([1, 1, 1, 1, 1, 0.5, 0, 0, 0, 0, 0, 0], float)
    chi = orc.flatten_line(p, u)
    assert list(chi[3:8]) == [1.0, 1.0, 0.0, 0.0, 1.0]         # F2: zone 6 looks at its low-pressure neighbour 5
    chi_m = orc.flatten_line(p[::-1].copy(), -u[::-1].copy())   # mirror image
    assert np.array_equal(chi_m[3:9], chi[::-1][3:9])
    # the same pressure profile in an expansion (u increasing): no shock, no flattening
    assert np.all(orc.flatten_line(p, -u) == 1.0)
    # a weak jump: |dp| / min(p) <= 1/3 everywhere
    pw = 1.0 + 0.1 * (p - 1.0) / 9.0
    assert np.all(orc.flatten_line(pw, u) == 1.0)
    # an intermediate value: zone 5 has dp = 4, dp2 = 5 -> z = 0.8 -> zeta = 0.5
    p2 = np.array([1, 1, 1, 1, 2, 5, 6, 6, 6, 6, 6], float)
    u2 = np.array([1, 1, 1, 1, 0.8, 0.3, 0, 0, 0, 0, 0], float)
    c2 = orc.flatten_line(p2, u2)
    assert abs(c2[5] - 0.5) < 1e-13
    # zone 4: dp = 5 - 1 = 4, dp2 = 6 - 1 = 5 as well -> 0.5; zone 6: dp = 1, dp2 = 4 -> z = 0.25 -> 1, but F2 (dp > 0)
    # takes the smaller of its own and zone 5's
    assert abs(c2[4] - 0.5) < 1e-13 and abs(c2[6] - 0.5) < 1e-13 and c2[7] == 1.0 and c2[3] == 1.0


# ---------------------------------------------------------------- the scheme with flattening ----
def run_sod(nx, flat, t_end=0.2):
    cfg = small_cfg(n=(nx, 4, 4), bc=(1, 0, 0), gamma=1.4, L=(1.0, 4.0 / nx, 4.0 / nx))
    W = uniform_W(cfg, [1, 0, 0, 0, 1])
    x = (np.arange(nx) + 0.5) / nx
    W[0] = np.where(x < 0.5, 1.0, 0.125)[None, None, :]
    W[4] = np.where(x < 0.5, 1.0, 0.1)[None, None, :]
    U = orc.fill_ghosts(cfg, state_from_prims(cfg, W))
    Af = (lambda V: orc.advance_A_flat(cfg, V)) if flat else None
    t, steps = 0.0, 0
    while t < t_end - 1e-14:
        dt = min(orc.cfl_dt(cfg, U, 0.5), t_end - t)
        U = orc.sdc_step_nodes(cfg, U, dt, M=2, K=2, A_fn=Af)
        t += dt
        steps += 1
    rho = wl.to_global(cfg, U, ghosted=True)[0]
    assert np.abs(rho - rho[0:1, 0:1, :]).max() == 0.0
    re, _, _ = orc.exact_riemann_sample(1.4, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, (x - 0.5) / t_end)
    return steps, np.abs(rho[0, 0] - re).mean()


def survey_values():
    rows = [l.split() for l in open(os.path.join(GOLD, "survey_sod_l1.txt")) if l.strip() and not l.startswith("#")]
    return {int(r[0]): (int(r[1]), float(r[2]), float(r[3])) for r in rows}


@pytest.mark.parametrize("nx", [64, 128])
def test_sod_errors_reproduce_the_surveys_independent_prototype(nx):
    """SURVEY.md Appendix A prints the L1 errors of an independent implementation of the same readings, with and
    without flattening, to four digits; both must come out of this oracle (tests/golden/survey_sod_l1.txt)."""
    steps, plain, flat = survey_values()[nx]
    s0, e0 = run_sod(nx, False)
    s1, e1 = run_sod(nx, True)
    assert s0 == steps
    assert abs(e0 - plain) <= 6e-4 * plain, (e0, plain)        # printed to 4 digits
    assert abs(e1 - flat) <= 6e-4 * flat, (e1, flat)
    assert abs(s1 - steps) <= 1


def test_smooth_flow_is_not_touched_bitwise():
    cfg = wl.make_config(2, n=24)                                 # the Gaussian pulse: p uniform
    U = orc.fill_ghosts(cfg, wl.initial_state(cfg))
    assert np.array_equal(orc.advance_A_flat(cfg, U), orc.advance_A(cfg, U))


def shocked_state(cfg, seed):
    """White noise with strong pressure contrasts (log-normal sigma 1.2): many zones pass the shock test."""
    Dx, Dy, Dz = wl.domain(cfg)
    rng = np.random.default_rng(seed)
    W = np.zeros((wl.nvar(cfg), Dz, Dy, Dx))
    W[0] = np.exp(0.3 * rng.standard_normal((Dz, Dy, Dx)))
    W[1:4] = 0.8 * rng.standard_normal((3, Dz, Dy, Dx))
    W[4] = np.exp(1.2 * rng.standard_normal((Dz, Dy, Dx)))
    if cfg["nspec"]:
        E = rng.standard_exponential((cfg["nspec"], Dz, Dy, Dx))
        W[5:] = E / E.sum(axis=0)
    return W


def test_invariants_with_active_flattening():
    cfg = small_cfg(n=(12, 12, 12), nspec=2, gamma=1.4)
    W = shocked_state(cfg, 5)
    U = orc.fill_ghosts(cfg, wl.from_global(cfg, wl.cons_from_prim(cfg, W)))
    A, A0 = orc.advance_A_flat(cfg, U), orc.advance_A(cfg, U)
    assert relmax(A, A0).max() > 1e-2, "flattening must be active in this test"
    # conservation on the periodic domain
    for c in range(wl.nvar(cfg)):
        assert abs(A[:, c].sum()) <= 1e-12 * np.abs(A[:, c]).sum()
    # axis permutation x <-> z (swap velocity components as well)
    Wp = W.transpose(0, 3, 2, 1).copy()
    Wp[[1, 3]] = Wp[[3, 1]]
    Ap = orc.advance_A_flat(cfg, orc.fill_ghosts(cfg, wl.from_global(cfg, wl.cons_from_prim(cfg, Wp))))
    G, Gp = wl.to_global(cfg, A), wl.to_global(cfg, Ap).transpose(0, 3, 2, 1).copy()
    Gp[[1, 3]] = Gp[[3, 1]]
    assert np.abs(G - Gp).max() <= 1e-13 * np.abs(G).max()
    # mirror in x
    Wm = W[:, :, :, ::-1].copy()
    Wm[1] *= -1.0
    Am = orc.advance_A_flat(cfg, orc.fill_ghosts(cfg, wl.from_global(cfg, wl.cons_from_prim(cfg, Wm))))
    Gm = wl.to_global(cfg, Am)[:, :, :, ::-1].copy()
    Gm[1] *= -1.0
    assert np.abs(G - Gm).max() <= 1e-13 * np.abs(G).max()
    # uniform state: exactly zero
    Uu = state_from_prims(cfg, uniform_W(cfg, [1.3, 0.4, -0.2, 0.1, 0.7, 0.25, 0.75]))
    assert np.all(orc.advance_A_flat(cfg, orc.fill_ghosts(cfg, Uu)) == 0.0)


def test_box_lattice_equals_single_box_bitwise_with_flattening():
    one = small_cfg(n=(16, 8, 8), nspec=1, gamma=1.4, bc=(1, 0, 2))
    cut = small_cfg(n=(8, 4, 8), nb=(2, 2, 1), nspec=1, gamma=1.4, bc=(1, 0, 2))
    G = wl.cons_from_prim(one, shocked_state(one, 6))
    A1 = orc.advance_A_flat(one, orc.fill_ghosts(one, wl.from_global(one, G)))
    A2 = orc.advance_A_flat(cut, orc.fill_ghosts(cut, wl.from_global(cut, G)))
    assert np.array_equal(wl.to_global(one, A1), wl.to_global(cut, A2))
