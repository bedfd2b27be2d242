"""Pins of the oracle's unsplit CTU PPM operator (oracle/orc_ctu.c, readings C1-C9; "the main unsplit
PPM hydrodynamics scheme [15, 16]").  No test here calls the CUDA path."""
import numpy as np
import pytest

from oracle import orc
from paper_1910_12578_b200 import workloads as wl
from test_oracle_pins import small_cfg, relmax
from test_oracle_scheme import uniform_W, state_from_prims


def cfl_dt_ctu(cfg, U, cfl):
    """dt = cfl * min_d Delta_d / max(|u_d| + c): the per-direction rule a CTU scheme is stable with (cfl <= 1)."""
    Ui = U[:, :, 4:-4, 4:-4, 4:-4]
    rho = Ui[:, 0]
    v = Ui[:, 1:4] / rho[:, None]
    p = (cfg["gamma"] - 1) * (Ui[:, 4] - 0.5 * rho * (v ** 2).sum(axis=1))
    c = np.sqrt(cfg["gamma"] * p / rho)
    h = (cfg["dx"], cfg["dy"], cfg["dz"])
    return cfl * min(h[d] / (np.abs(v[:, d]) + c).max() for d in range(3))


def test_unit_cfl_advection_is_an_exact_diagonal_shift():
    """Uniform velocity and pressure, dt = dx/u = dy/v = dz/w: every wave crosses exactly one zone, so the scheme must
    move the state by one zone along the diagonal, whatever the density and composition (white noise here: every
    limiter fires).  Every coefficient of the tracing (I+-(1) = the zone average), of the 1/3 and of the 1/2
    transverse corrections enters; a wrong one leaves O(1) errors.  Measured: 1.2e-15."""
    rng = np.random.default_rng(3)
    n = (8, 12, 16)
    cfg = small_cfg(n=n, nspec=2, gamma=1.4)
    dt = 0.05
    W = np.zeros((7, n[2], n[1], n[0]))
    W[0] = np.exp(0.5 * rng.standard_normal(W[0].shape))
    W[1], W[2], W[3] = cfg["dx"] / dt, cfg["dy"] / dt, cfg["dz"] / dt
    W[4] = 1.0
    W[5] = rng.random(W[0].shape)
    W[6] = 1 - W[5]
    Ug = wl.cons_from_prim(cfg, W)
    A = wl.to_global(cfg, orc.advance_ctu(cfg, orc.fill_ghosts(cfg, wl.from_global(cfg, Ug)), dt))
    exact = (np.roll(Ug, (1, 1, 1), axis=(1, 2, 3)) - Ug) / dt
    assert np.abs(A - exact).max() <= 1e-13 * np.abs(exact).max()
    # and against the flow (negative velocities): a shift the other way
    W[1:4] *= -1.0
    Ug = wl.cons_from_prim(cfg, W)
    A = wl.to_global(cfg, orc.advance_ctu(cfg, orc.fill_ghosts(cfg, wl.from_global(cfg, Ug)), dt))
    exact = (np.roll(Ug, (-1, -1, -1), axis=(1, 2, 3)) - Ug) / dt
    assert np.abs(A - exact).max() <= 1e-13 * np.abs(exact).max()


def run_sod(nx, cfl=0.8, t_end=0.2):
    cfg = small_cfg(n=(nx, 4, 4), bc=(1, 0, 0), gamma=1.4, L=(1.0, 4.0 / nx, 4.0 / nx))
    W = uniform_W(cfg, [1, 0, 0, 0, 1])
    x = (np.arange(nx) + 0.5) / nx
    W[0] = np.where(x < 0.5, 1.0, 0.125)[None, None, :]
    W[4] = np.where(x < 0.5, 1.0, 0.1)[None, None, :]
    U = orc.fill_ghosts(cfg, state_from_prims(cfg, W))
    t, steps = 0.0, 0
    while t < t_end - 1e-14:
        dt = min(cfl_dt_ctu(cfg, U, cfl), t_end - t)
        U = orc.ctu_step(cfg, U, dt)
        t += dt
        steps += 1
    rho = wl.to_global(cfg, U, ghosted=True)[0]
    assert np.abs(rho - rho[0:1, 0:1, :]).max() == 0.0
    re, _, _ = orc.exact_riemann_sample(1.4, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, (x - 0.5) / t_end)
    return np.abs(rho[0, 0] - re).mean(), steps


def test_sod_against_the_exact_riemann_solution_at_cfl_08():
    """The acoustic part of the tracing (a+, a-): shock and rarefaction at the right places, one stage per step at CFL 0.8.
    Measured L1(rho): 5.41e-3 (35 steps) / 2.62e-3 (70 steps) at n = 64 / 128; the SDC path gives 5.93e-3 (119 steps) /
    2.78e-3 (241 steps) at its CFL 0.5 (sum form)."""
    (e64, s64), (e128, s128) = run_sod(64), run_sod(128)
    assert e64 < 8e-3 and e128 < 4e-3 and e64 / e128 > 1.7, (e64, e128, s64, s128)


def pulse_error(n, cfl=0.8, t_end=0.05):
    cfg = wl.make_config(2, n=n)
    U = orc.fill_ghosts(cfg, wl.initial_state(cfg))
    t = 0.0
    while t < t_end - 1e-14:
        dt = min(cfl_dt_ctu(cfg, U, cfl), t_end - t)
        U = orc.ctu_step(cfg, U, dt)
        t += dt
    rho = wl.to_global(cfg, U, ghosted=True)[0]
    x = (np.arange(n) + 0.5) / n
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    d = lambda a: (a - 0.5 - t_end + 0.5) % 1.0 - 0.5
    exact = 1 + 0.5 * np.exp(-(d(X) ** 2 + d(Y) ** 2 + d(Z) ** 2) / 0.01)
    return np.abs(rho - exact).mean()


def test_three_dimensional_pulse_converges_at_cfl_08():
    """Second order in space and time from ONE stage per step at CFL 0.8 (where one Euler stage of the method-of-lines
    operator is unstable).  Measured L1(rho): 3.89e-4, 9.24e-5, 2.24e-5 at 16^3, 32^3, 64^3 (ratios 4.2, 4.1)."""
    e = [pulse_error(n) for n in (16, 32, 64)]
    assert e[1] / e[2] > 3.0 and e[0] / e[1] > 2.0, e


def test_invariants():
    cfg = small_cfg(n=(10, 10, 10), nspec=1, gamma=1.4)
    Gs = wl.to_global(cfg, wl.random_state(cfg, 121), ghosted=True)
    U = orc.fill_ghosts(cfg, wl.from_global(cfg, Gs))
    dt = cfl_dt_ctu(cfg, U, 0.8)
    A = wl.to_global(cfg, orc.advance_ctu(cfg, U, dt))
    assert relmax(orc.advance_ctu(cfg, U, dt), orc.advance_A(cfg, U)).max() > 1e-2      # not the method-of-lines operator
    for c in range(wl.nvar(cfg)):
        assert abs(A[c].sum()) <= 1e-12 * np.abs(A[c]).sum()                            # conservation
    Gp = Gs.transpose(0, 3, 2, 1).copy()
    Gp[[1, 3]] = Gp[[3, 1]]
    Ap = wl.to_global(cfg, orc.advance_ctu(cfg, orc.fill_ghosts(cfg, wl.from_global(cfg, Gp)), dt)).transpose(0, 3, 2, 1).copy()
    Ap[[1, 3]] = Ap[[3, 1]]
    assert np.abs(A - Ap).max() <= 1e-13 * np.abs(A).max()                              # x <-> z
    Gm = Gs[:, :, :, ::-1].copy()
    Gm[1] *= -1.0
    Am = wl.to_global(cfg, orc.advance_ctu(cfg, orc.fill_ghosts(cfg, wl.from_global(cfg, Gm)), dt))[:, :, :, ::-1].copy()
    Am[1] *= -1.0
    assert np.abs(A - Am).max() <= 1e-13 * np.abs(A).max()                              # mirror in x
    Uu = orc.fill_ghosts(cfg, state_from_prims(cfg, uniform_W(cfg, [1.3, 0.4, -0.2, 0.1, 0.7, 0.6])))
    assert np.abs(orc.advance_ctu(cfg, Uu, dt)).max() <= 1e-13                           # uniform state (tracing adds roundoff)
    # dt -> 0: for rho (and the species, which ride on the mass flux) the traced states become the parabola edges of the
    # SDC path's operator; the passively traced velocities do not (a wave that moves away leaves the zone average, C3)
    e0 = relmax(orc.advance_ctu(cfg, U, 0.0), orc.advance_A(cfg, U))
    assert e0[0] <= 1e-13 and e0[5] <= 1e-13 and e0[1:5].max() > 1e-3


def test_box_lattice_and_gravity():
    one = small_cfg(n=(16, 8, 8), nspec=1, gamma=1.4, bc=(1, 0, 2), grav=(0.0, 0.0, -0.3))
    cut = small_cfg(n=(8, 4, 8), nb=(2, 2, 1), nspec=1, gamma=1.4, bc=(1, 0, 2), grav=(0.0, 0.0, -0.3))
    Gs = wl.to_global(one, wl.random_state(one, 122), ghosted=True)
    A1 = orc.advance_ctu(one, orc.fill_ghosts(one, wl.from_global(one, Gs)), 0.01)
    A2 = orc.advance_ctu(cut, orc.fill_ghosts(cut, wl.from_global(cut, Gs)), 0.01)
    assert np.array_equal(wl.to_global(one, A1), wl.to_global(cut, A2))
