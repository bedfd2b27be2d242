"""Pins of the oracle's explicit diffusion term (oracle/orc_diffuse.c; SURVEY 8(f) NEXT-4;
DESIGN.md readings D1-D3).  No test here calls the CUDA path."""
import numpy as np

from oracle import orc
from paper_1910_12578_b200 import workloads as wl
from test_oracle_pins import small_cfg

CV, KTH = 1.5, 0.37


def state_with_temperature(cfg, T, rho=None, v=(0.3, -0.2, 0.1)):
    """Global temperature field [Dz, Dy, Dx] -> ghosted box state with that T (gamma-law, c_v = CV)."""
    Dx, Dy, Dz = wl.domain(cfg)
    W = np.zeros((wl.nvar(cfg), Dz, Dy, Dx))
    W[0] = 1.0 if rho is None else rho
    for d in range(3):
        W[1 + d] = v[d]
    W[4] = (cfg["gamma"] - 1.0) * W[0] * CV * T
    return orc.fill_ghosts(cfg, wl.from_global(cfg, wl.cons_from_prim(cfg, W)))


def test_uniform_temperature_gives_exactly_zero_whatever_rho_and_v():
    cfg = small_cfg(n=(6, 5, 4), nb=(2, 1, 1), gamma=5 / 3)
    rng = np.random.default_rng(3)
    Dx, Dy, Dz = wl.domain(cfg)
    # powers of two keep p / ((gamma-1) rho cv) free of rounding, so that T is bitwise uniform
    rho = 2.0 ** rng.integers(-2, 3, size=(Dz, Dy, Dx))
    g = small_cfg(n=(6, 5, 4), nb=(2, 1, 1), gamma=2.0)
    U = state_with_temperature(g, np.full((Dz, Dy, Dx), 2.0), rho=rho, v=(0.0, 0.0, 0.0))
    assert np.all(orc.diffusion(g, KTH, 1.0, U) == 0.0)


def test_periodic_sum_vanishes_and_only_the_energy_component_changes():
    cfg = small_cfg(n=(8, 6, 5), nb=(1, 2, 1), nspec=2, gamma=5 / 3)
    U = orc.fill_ghosts(cfg, wl.random_state(cfg, 61))
    D = orc.diffusion(cfg, KTH, CV, U)
    assert abs(D.sum()) <= 1e-12 * np.abs(D).sum()
    A0, A1 = orc.advance_A(cfg, U), orc.advance_A_diffuse(cfg, KTH, CV, U)
    assert np.array_equal(np.delete(A0, 4, axis=1), np.delete(A1, 4, axis=1))
    assert np.array_equal(A1[:, 4], A0[:, 4] + D)


def test_sine_mode_discrete_eigenvalue_and_second_order_convergence():
    errs = []
    for n in (16, 32, 64):
        cfg = small_cfg(n=(n, 4, 4), gamma=5 / 3, L=(1.0, 4.0 / n, 4.0 / n))
        x = (np.arange(n) + 0.5) / n
        T = 1.0 + 0.25 * np.sin(2 * np.pi * 2 * x)[None, None, :] * np.ones((4, 4, 1))
        rho = 1.0 + 0.3 * np.cos(2 * np.pi * x)[None, None, :] * np.ones((4, 4, 1))
        D = orc.diffusion(cfg, KTH, CV, state_with_temperature(cfg, T, rho=rho))[0]
        th = 2 * np.pi * 2 / n
        disc = -KTH * (2 - 2 * np.cos(th)) * n * n * (T - 1.0)              # eigenvalue of the 3-point Laplacian
        assert np.abs(D - disc).max() <= 1e-10 * np.abs(disc).max()
        exact = -KTH * (2 * np.pi * 2) ** 2 * (T - 1.0)
        errs.append(np.abs(D - exact).max())
    assert 3.6 < errs[0] / errs[1] < 4.2 and 3.85 < errs[1] / errs[2] < 4.1, errs      # measured 3.71, 3.93


def test_each_direction_uses_its_own_zone_width():
    cfg = small_cfg(n=(4, 4, 16), gamma=1.4, L=(0.5, 0.25, 2.0))
    z = (np.arange(16) + 0.5) / 16 * 2.0
    T = 2.0 + 0.1 * np.cos(2 * np.pi * z / 2.0)[:, None, None] * np.ones((1, 4, 4))
    D = orc.diffusion(cfg, KTH, CV, state_with_temperature(cfg, T))[0]
    th = 2 * np.pi / 16
    disc = -KTH * (2 - 2 * np.cos(th)) / cfg["dz"] ** 2 * (T - 2.0)
    assert np.abs(D - disc).max() <= 1e-10 * np.abs(disc).max()
