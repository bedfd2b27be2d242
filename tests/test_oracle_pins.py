"""Pins of the CPU oracle (oracle/orc.c) against what the paper and the mathematics fix.

No test here calls the CUDA path.  Each pin states which part of the oracle it would catch a
mistake in (SURVEY.md 8(c) pins P1..P15; BASELINE.json north_star's four oracle checks:
exact Sod solution, conservation, A(uniform)=0, permutation/mirror invariance).
"""
import os

import numpy as np
import pytest
from scipy.optimize import brentq

from oracle import orc
from paper_1910_12578_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def small_cfg(n=(8, 8, 8), nb=(1, 1, 1), nspec=0, gamma=1.4, bc=(0, 0, 0), L=None, grav=(0, 0, 0)):
    nx, ny, nz = n
    L = L or (1.0, 1.0, 1.0)
    return dict(name="t", index=99, nx=nx, ny=ny, nz=nz, ng=4, nbx=nb[0], nby=nb[1], nbz=nb[2],
                nspec=nspec, dx=L[0] / (nx * nb[0]), dy=L[1] / (ny * nb[1]), dz=L[2] / (nz * nb[2]),
                gamma=gamma, grav=tuple(grav), bc_lo=tuple(bc), bc_hi=tuple(bc),
                small_dens=1e-200, small_pres=1e-200)


def relmax(a, b):
    """max-normalised per-component error (DESIGN.md parity norm), arrays [b][c]..."""
    axes = (0,) + tuple(range(2, a.ndim))
    num = np.abs(a - b).max(axis=axes)
    den = np.abs(b).max(axis=axes)
    return np.where(den > 0, num / np.where(den > 0, den, 1), num)


# ------------------------------------------------------------------ P2: exact Riemann solver ----
def read_golden():
    d = {}
    for line in open(os.path.join(GOLD, "sod_exact_star.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        d[k] = float(v)
    return d


def independent_sod_star(g=1.4, rL=1.0, pL=1.0, rR=0.125, pR=0.1):
    """Pressure function written out here (left rarefaction, right shock), solved by bisection:
    independent of the Newton iteration in oracle/orc.c."""
    cL = np.sqrt(g * pL / rL)

    def f(p):
        fL = 2 * cL / (g - 1) * ((p / pL) ** ((g - 1) / (2 * g)) - 1)
        AR, BR = 2 / ((g + 1) * rR), (g - 1) / (g + 1) * pR
        fR = (p - pR) * np.sqrt(AR / (p + BR))
        return fL + fR
    ps = brentq(f, pR, pL, xtol=1e-15, rtol=1e-15)
    us = -2 * cL / (g - 1) * ((ps / pL) ** ((g - 1) / (2 * g)) - 1)
    rsL = rL * (ps / pL) ** (1 / g)
    gm = (g - 1) / (g + 1)
    rsR = rR * (ps / pR + gm) / (gm * ps / pR + 1)
    cR = np.sqrt(g * pR / rR)
    S = cR * np.sqrt((g + 1) / (2 * g) * ps / pR + (g - 1) / (2 * g))
    tail = us - cL * (ps / pL) ** ((g - 1) / (2 * g))
    return dict(p_star=ps, u_star=us, rho_star_L=rsL, rho_star_R=rsR, shock_speed=S,
                rarefaction_head=-cL, rarefaction_tail=tail)


def test_P2_exact_riemann_star_values():
    gold, ind = read_golden(), independent_sod_star()
    st = orc.exact_riemann_star(1.4, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
    got = dict(p_star=st[0], u_star=st[1], rho_star_L=st[2], rho_star_R=st[3])
    for k, v in gold.items():
        assert abs(ind[k] - v) <= 2e-6 * max(1, abs(v)), (k, ind[k], v)   # fixture is right
    for k, v in got.items():
        assert abs(v - ind[k]) <= 1e-12, (k, v, ind[k])
        assert abs(v - gold[k]) <= 1e-6


def test_P2_exact_riemann_sampling_and_jump_conditions():
    g = 1.4
    gold = read_golden()
    xi = np.array([-2.0, gold["rarefaction_head"] - 1e-5, gold["rarefaction_tail"] + 1e-5,
                   gold["u_star"] - 1e-5, gold["u_star"] + 1e-5, gold["shock_speed"] - 1e-5,
                   gold["shock_speed"] + 1e-5, 3.0])
    rho, u, p = orc.exact_riemann_sample(g, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, xi)
    assert (rho[0], u[0], p[0]) == (1.0, 0.0, 1.0) and (rho[1], u[1], p[1]) == (1.0, 0.0, 1.0)
    assert abs(rho[2] - gold["rho_star_L"]) < 1e-6 and abs(rho[3] - gold["rho_star_L"]) < 1e-6
    assert abs(rho[4] - gold["rho_star_R"]) < 1e-6 and abs(rho[5] - gold["rho_star_R"]) < 1e-6
    assert (rho[6], u[6], p[6]) == (0.125, 0.0, 0.1) and rho[7] == 0.125
    # inside the fan the Riemann invariant u + 2c/(g-1) and the entropy p/rho^g are those of the left state
    xs = np.linspace(gold["rarefaction_head"], gold["rarefaction_tail"], 7)[1:-1]
    r, uu, pp = orc.exact_riemann_sample(g, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, xs)
    c = np.sqrt(g * pp / r)
    assert np.allclose(uu + 2 * c / (g - 1), 2 * np.sqrt(g) / (g - 1), rtol=1e-13)
    assert np.allclose(pp / r ** g, 1.0, rtol=1e-13)
    assert np.allclose(uu - c, xs, rtol=1e-13, atol=1e-14)
    # Rankine-Hugoniot across the right shock: S [rho] = [rho u]
    S, rs, us = gold["shock_speed"], rho[5], u[5]
    assert abs(S * (rs - 0.125) - rs * us) < 1e-5


# ------------------------------------------------------------------ P5/P6: HLLC ------------------
def physical_flux(d, g, W):
    rho, v, p = W[0], W[1:4], W[4]
    E = p / (g - 1) + 0.5 * rho * (v @ v)
    F = np.empty_like(W)
    F[0] = rho * v[d]
    F[1:4] = rho * v[d] * v
    F[1 + d] += p
    F[4] = (E + p) * v[d]
    F[5:] = rho * v[d] * W[5:]
    return F


@pytest.mark.parametrize("d", [0, 1, 2])
def test_P5_hllc_consistency_and_supersonic(d):
    rng = np.random.default_rng(5 + d)
    g = 5.0 / 3.0
    for _ in range(50):
        W = np.concatenate([[np.exp(rng.normal())], rng.normal(size=3), [np.exp(rng.normal())],
                            rng.random(3)])
        F = orc.hllc(d, g, W, W)
        Fp = physical_flux(d, g, W)
        assert np.allclose(F, Fp, rtol=1e-13, atol=1e-13 * np.abs(Fp).max())
    # supersonic to the right: F = F(W_L) exactly; to the left: F = F(W_R) exactly
    WL = np.array([1.0, 0.1, -0.2, 0.3, 1.0, 0.25, 0.75])
    WR = np.array([0.5, 0.2, 0.1, -0.3, 0.7, 0.6, 0.4])
    WL[1 + d], WR[1 + d] = 5.0, 6.0
    assert np.allclose(orc.hllc(d, 1.4, WL, WR), physical_flux(d, 1.4, WL), rtol=1e-15, atol=0)
    WL[1 + d], WR[1 + d] = -6.0, -5.0
    assert np.allclose(orc.hllc(d, 1.4, WL, WR), physical_flux(d, 1.4, WR), rtol=1e-15, atol=0)


@pytest.mark.parametrize("d", [0, 1, 2])
def test_P6_hllc_isolated_contact_is_exact(d):
    """HLLC (unlike HLL) resolves a contact moving with the flow: across a density jump with
    uniform p and velocity, F = F(upwind state) to roundoff; at rest the mass flux is exactly 0."""
    g = 1.4
    for un in (0.0, 0.3, -0.3):
        WL = np.array([1.0, 0.0, 0.0, 0.0, 1.0, 1.0, 0.0]); WR = np.array([0.125, 0.0, 0.0, 0.0, 1.0, 0.0, 1.0])
        WL[1 + d] = WR[1 + d] = un
        F = orc.hllc(d, g, WL, WR)
        Fu = physical_flux(d, g, WL if un >= 0 else WR)
        assert np.allclose(F, Fu, rtol=0, atol=4e-16 * max(1.0, np.abs(Fu).max()))
        if un == 0.0:
            assert F[0] == 0.0 and F[4] == 0.0 and F[1 + d] == 1.0 and F[5] == 0.0


def test_hllc_mirror_symmetry():
    """Mirroring the Riemann problem flips the sign of all fluxes except normal momentum."""
    rng = np.random.default_rng(11)
    for _ in range(100):
        WL = np.concatenate([[np.exp(rng.normal())], rng.normal(size=3), [np.exp(rng.normal())], rng.random(2)])
        WR = np.concatenate([[np.exp(rng.normal())], rng.normal(size=3), [np.exp(rng.normal())], rng.random(2)])
        F = orc.hllc(0, 1.4, WL, WR)
        ML, MR = WR.copy(), WL.copy()
        ML[1] *= -1; MR[1] *= -1
        Fm = orc.hllc(0, 1.4, ML, MR)
        sgn = np.array([-1, 1, -1, -1, -1, -1, -1.0])
        assert np.allclose(Fm, sgn * F, rtol=1e-13, atol=1e-14)


def test_hllc_entropy_satisfying_against_exact_sod_flux():
    """The HLLC flux of the Sod problem at x/t = 0 approximates the exact Godunov flux there
    (x/t = 0 lies in the left star region); a wrong-sign or transposed state misses by O(1)."""
    g = 1.4
    WL = np.array([1.0, 0, 0, 0, 1.0]); WR = np.array([0.125, 0, 0, 0, 0.1])
    F = orc.hllc(0, g, WL, WR)
    r, u, p = orc.exact_riemann_sample(g, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, np.array([0.0]))
    Fe = physical_flux(0, g, np.array([r[0], u[0], 0, 0, p[0]]))
    assert np.allclose(F, Fe, rtol=0.25, atol=0.02)


# ------------------------------------------------------------------ P9/P10: PPM ------------------
def test_P9_ppm_edge_values_exact_for_cubic_cell_averages():
    """CW84 (1.6) on a uniform grid is the 7/12,-1/12 fourth-order interpolant of cell averages:
    for cell averages of a monotone cubic (no limiter active) the edge equals the point value."""
    h = 0.1
    c = np.array([0.3, 2.0, 0.4, 0.5])                # a + b x + c x^2 + d x^3, monotone on [0, 1.6]
    prim = lambda x: c[0] * x + c[1] * x ** 2 / 2 + c[2] * x ** 3 / 3 + c[3] * x ** 4 / 4
    xe = h * np.arange(17)
    qbar = (prim(xe[1:]) - prim(xe[:-1])) / h
    qm, qp = orc.ppm_line(qbar)
    point = c[0] + c[1] * xe + c[2] * xe ** 2 + c[3] * xe ** 3
    for i in range(2, 14):
        assert abs(qm[i] - point[i]) < 1e-13 and abs(qp[i] - point[i + 1]) < 1e-13
    assert np.isnan(qm[1]) and np.isnan(qp[14])       # documented valid range 2..n-3


def test_P10_ppm_limiter_bounds_monotone_extrema():
    rng = np.random.default_rng(10)
    for trial in range(300):
        n = 12
        q = rng.normal(size=n) if trial % 2 else np.cumsum(rng.random(n) ** 3)
        qm, qp = orc.ppm_line(q)
        for i in range(2, n - 2):
            lo, hi = min(q[i - 1:i + 2]), max(q[i - 1:i + 2])
            eps = 1e-14 * max(1.0, abs(hi), abs(lo))
            assert lo - eps <= qm[i] <= hi + eps and lo - eps <= qp[i] <= hi + eps
            if (q[i + 1] - q[i]) * (q[i] - q[i - 1]) <= 0:
                assert qm[i] == q[i] and qp[i] == q[i]
            # parabola a(x) = qm + x (D + q6 (1-x)) monotone on [0,1]  <=>  |q6| <= |D|
            D, q6 = qp[i] - qm[i], 6 * (q[i] - 0.5 * (qm[i] + qp[i]))
            assert abs(q6) <= abs(D) * (1 + 1e-12) + 1e-14


def test_ppm_mirror_and_affine_invariance():
    rng = np.random.default_rng(12)
    q = rng.normal(size=16)
    qm, qp = orc.ppm_line(q)
    rm, rp = orc.ppm_line(q[::-1].copy())
    assert np.array_equal(rm[::-1][2:-2], qp[2:-2]) and np.array_equal(rp[::-1][2:-2], qm[2:-2])
    sm, sp = orc.ppm_line(-2.0 * q)
    assert np.array_equal(sm[2:-2], -2.0 * qm[2:-2]) and np.array_equal(sp[2:-2], -2.0 * qp[2:-2])


# ------------------------------------------------------------------ S1 ---------------------------
def test_S1_cons_to_prim_roundtrip_and_floor():
    rng = np.random.default_rng(1)
    g = 5.0 / 3.0
    W = np.concatenate([[0.7], rng.normal(size=3), [1.3], [0.2, 0.8]])
    U = np.concatenate([[W[0]], W[0] * W[1:4], [W[4] / (g - 1) + 0.5 * W[0] * (W[1:4] @ W[1:4])], W[0] * W[5:]])
    assert np.allclose(orc.cons_to_prim(g, 1e-200, U), W, rtol=1e-14)
    U[4] = 0.0                                   # negative pressure -> floored
    assert orc.cons_to_prim(g, 1e-5, U)[4] == 1e-5
