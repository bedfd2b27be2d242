"""Round-2 pins of the CPU oracle: the two parts round 1 left unpinned (What's weak 1).

(a) The SHOCK branch of the HLLC wave-speed estimate (oracle/orc.c orc_wave_speeds, reading Q6:
    q_K = sqrt(1 + (gamma+1)/(2 gamma) (p*/p_K - 1)) for p* > p_K).  With the EXACT star pressure the
    estimate is the exact shock speed (Toro ch. 3/4): the textbook Sod value 1.752156
    (tests/golden/sod_exact_star.txt) and, for random shocks, the speed that the Rankine-Hugoniot mass
    condition rho_K (u_K - S) = rho*_K (u* - S) gives from the exact star state.  A wrong factor
    (e.g. (gamma-1)/(2 gamma)) fails both.
(b) The INTERFACE floors of S2 step 4 (orc.c line_fluxes: rho >= small_dens, p >= small_pres on both
    face states), with floors large enough to bind, against a brute-force restatement written here.
No test here calls the CUDA path.
"""
import os

import numpy as np
import pytest

from oracle import orc
from paper_1910_12578_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def read_golden():
    d = {}
    for line in open(os.path.join(GOLD, "sod_exact_star.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        d[k] = float(v)
    return d


# ---------------------------------------------------------------- (a) wave speeds, shock branch ----
def test_wave_speeds_exact_pstar_gives_textbook_sod_shock_speed():
    gold = read_golden()
    g = 1.4
    st = orc.exact_riemann_star(g, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
    SL, SR = orc.wave_speeds(g, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, st[0])
    assert abs(SR - gold["shock_speed"]) <= 1e-6            # right shock: the branch under test
    assert abs(SL - gold["rarefaction_head"]) <= 1e-6       # left rarefaction: q = 1, S_L = u_L - c_L
    # mirrored problem: the LEFT wave is the shock
    SLm, SRm = orc.wave_speeds(g, 0.125, 0.0, 0.1, 1.0, 0.0, 1.0, st[0])
    assert SLm == -SR and SRm == -SL


def test_wave_speeds_exact_pstar_satisfies_rankine_hugoniot_for_random_shocks():
    rng = np.random.default_rng(21)
    n_shock = 0
    for g in (1.4, 5.0 / 3.0):
        for _ in range(200):
            rL, rR = np.exp(rng.normal(size=2))
            pL, pR = np.exp(1.5 * rng.normal(size=2))
            uL, uR = rng.normal(size=2)
            if uR - uL >= 2.0 / (g - 1) * (np.sqrt(g * pL / rL) + np.sqrt(g * pR / rR)) * 0.8:
                continue                                   # near-vacuum: skip
            ps, us, rsL, rsR, _ = orc.exact_riemann_star(g, rL, uL, pL, rR, uR, pR)
            SL, SR = orc.wave_speeds(g, rL, uL, pL, rR, uR, pR, ps)
            if ps > pR * (1 + 1e-3):                       # right shock
                S = (rsR * us - rR * uR) / (rsR - rR)      # mass jump condition
                assert abs(SR - S) <= 1e-9 * max(1.0, abs(S)), (g, SR, S)
                n_shock += 1
            else:
                assert SR == uR + np.sqrt(g * pR / rR) or ps > pR
            if ps > pL * (1 + 1e-3):                       # left shock
                S = (rsL * us - rL * uL) / (rsL - rL)
                assert abs(SL - S) <= 1e-9 * max(1.0, abs(S)), (g, SL, S)
                n_shock += 1
    assert n_shock > 100


def test_hllc_uses_pvrs_estimate_and_wave_speeds():
    """orc_hllc = textbook HLLC (F*_K = F_K + S_K (U*_K - U_K), Toro (10.71)-(10.73)) on the speeds of
    orc_wave_speeds at the PVRS pressure (Toro (10.67)): a strong-shock face, written out here."""
    g = 1.4
    rng = np.random.default_rng(22)
    for _ in range(100):
        WL = np.array([np.exp(rng.normal()), rng.normal(), rng.normal(), rng.normal(), np.exp(2 * rng.normal())])
        WR = np.array([np.exp(rng.normal()), rng.normal(), rng.normal(), rng.normal(), np.exp(2 * rng.normal())])
        WL[1] += 2.0                                      # converging flow: shocks on both sides are common
        rL, uL, pL, rR, uR, pR = WL[0], WL[1], WL[4], WR[0], WR[1], WR[4]
        cL, cR = np.sqrt(g * pL / rL), np.sqrt(g * pR / rR)
        ppv = max(0.0, 0.5 * (pL + pR) - 0.125 * (uR - uL) * (rL + rR) * (cL + cR))
        assert abs(orc.pvrs_pstar(g, rL, uL, pL, rR, uR, pR) - ppv) <= 1e-14 * max(1.0, ppv)
        SL, SR = orc.wave_speeds(g, rL, uL, pL, rR, uR, pR, ppv)
        Ss = (pR - pL + rL * uL * (SL - uL) - rR * uR * (SR - uR)) / (rL * (SL - uL) - rR * (SR - uR))

        def cons(W):
            return np.array([W[0], W[0] * W[1], W[0] * W[2], W[0] * W[3],
                             W[4] / (g - 1) + 0.5 * W[0] * (W[1] ** 2 + W[2] ** 2 + W[3] ** 2)])

        def flux(W):
            U = cons(W)
            return np.array([U[1], U[1] * W[1] + W[4], U[1] * W[2], U[1] * W[3], W[1] * (U[4] + W[4])])

        def star(W, SK):
            U = cons(W)
            f = W[0] * (SK - W[1]) / (SK - Ss)
            return f * np.array([1.0, Ss, W[2], W[3],
                                 U[4] / W[0] + (Ss - W[1]) * (Ss + W[4] / (W[0] * (SK - W[1])))])
        if SL >= 0:
            Fe = flux(WL)
        elif SR <= 0:
            Fe = flux(WR)
        elif Ss >= 0:
            Fe = flux(WL) + SL * (star(WL, SL) - cons(WL))
        else:
            Fe = flux(WR) + SR * (star(WR, SR) - cons(WR))
        F = orc.hllc(0, g, WL, WR)
        assert np.allclose(F, Fe, rtol=1e-11, atol=1e-11 * np.abs(Fe).max())


def test_hllc_on_mirror_image_states_a_reflecting_wall():
    """The face of a reflecting wall sees W_R = mirror(W_L): the numerator of S* cancels exactly, S* = 0.  Subsonic
    approach: S_L < 0 < S_R, the star flux with NO mass through the wall and the wall pressure p + rho u c q (Rankine-
    Hugoniot across S_L).  Approach faster than the PVRS shock speed: S_L > 0 > S_R, and the textbook's first test
    (0 <= S_L: F = F_L, Toro (10.71)) decides -- the side S* >= 0 picks at S* = 0.  The CUDA path must take the same
    side whatever the compiler fuses (tests/test_next_gpu_walls.py)."""
    g = 5.0 / 3.0
    rng = np.random.default_rng(31)
    seen = [0, 0]
    for _ in range(200):
        rho, p = np.exp(rng.normal()), np.exp(rng.normal())
        c = np.sqrt(g * p / rho)
        u = c * rng.uniform(0.05, 4.0)
        v, w = rng.normal(), rng.normal()
        for d in range(3):
            WL = np.array([rho, v, w, v, p]); WR = WL.copy()
            WL[1 + d], WR[1 + d] = u, -u
            ps = orc.pvrs_pstar(g, rho, u, p, rho, -u, p)
            SL, SR = orc.wave_speeds(g, rho, u, p, rho, -u, p, ps)
            assert SL == -SR
            F = orc.hllc(d, g, WL, WR)
            if SL > 0.0:
                E = p / (g - 1) + 0.5 * rho * (WL[1] ** 2 + WL[2] ** 2 + WL[3] ** 2)
                Fe = rho * u * np.array([1.0, WL[1], WL[2], WL[3], 0.0])
                Fe[1 + d] += p
                Fe[4] = u * (E + p)
                assert np.allclose(F, Fe, rtol=1e-14, atol=0.0)
                seen[1] += 1
            else:
                Fn = F.copy(); Fn[1 + d] = 0.0                     # nothing but the wall pressure crosses the face
                E = p / (g - 1) + 0.5 * rho * (u * u + v * v + w * w)
                scale = np.array([rho * u, p + rho * u * u, p + rho * u * u, p + rho * u * u, u * (E + p)])
                assert np.all(np.abs(Fn) <= 1e-13 * scale * (1.0 + abs(v) + abs(w)))
                assert abs(F[1 + d] - (p + rho * u * (u - SL))) <= 1e-13 * F[1 + d]
                seen[0] += 1
    assert min(seen) > 50


# ---------------------------------------------------------------- (b) interface floors ------------
def line_cfg(nx, small_dens, small_pres, nspec=1):
    return dict(name="t", index=99, nx=nx, ny=4, nz=4, ng=4, nbx=1, nby=1, nbz=1, nspec=nspec,
                dx=1.0 / nx, dy=0.25, dz=0.25, gamma=1.4, grav=(0.0, 0.0, 0.0),
                bc_lo=(0, 0, 0), bc_hi=(0, 0, 0), small_dens=small_dens, small_pres=small_pres)


def brute_force_line_A(cfg, U):
    """A of a state that is uniform in y and z, restated zone by zone in Python: cons->prim (orc),
    PPM edges (orc.ppm_line), FLOORS WRITTEN HERE, HLLC (orc.hllc), flux difference along x."""
    ng, nx, N = 4, cfg["nx"], 5 + cfg["nspec"]
    line = U[0, :, ng, ng, :]                               # [N][ex]
    ex = nx + 2 * ng
    W = np.stack([orc.cons_to_prim(cfg["gamma"], cfg["small_pres"], line[:, i]) for i in range(ex)], axis=1)
    qm = np.empty_like(W); qp = np.empty_like(W)
    for c in range(N):
        qm[c], qp[c] = orc.ppm_line(W[c])
    F = np.empty((N, nx + 1))
    n_active = 0
    for f in range(nx + 1):
        WL = qp[:, f - 1 + ng].copy(); WR = qm[:, f + ng].copy()
        for Wk in (WL, WR):
            if Wk[0] < cfg["small_dens"]:
                Wk[0] = cfg["small_dens"]; n_active += 1
            if Wk[4] < cfg["small_pres"]:
                Wk[4] = cfg["small_pres"]; n_active += 1
        F[:, f] = orc.hllc(0, cfg["gamma"], WL, WR)
    return -((F[:, 1:] - F[:, :-1]) / cfg["dx"]), n_active


def floor_state(cfg, seed):
    """Sawtooth density / pressure whose parabola edges undershoot the zone averages next to the floors."""
    rng = np.random.default_rng(seed)
    nx, ng, N = cfg["nx"], 4, 5 + cfg["nspec"]
    rho = 0.62 + 0.5 * rng.random(nx) ** 2
    p = 0.52 + 0.6 * rng.random(nx) ** 2
    u = 0.3 * rng.normal(size=nx)
    X = rng.random(nx)
    U = np.zeros(orc.u_shape(cfg))
    sl = slice(ng, ng + nx)
    U[0, 0, :, :, sl] = rho
    U[0, 1, :, :, sl] = rho * u
    U[0, 4, :, :, sl] = p / (cfg["gamma"] - 1) + 0.5 * rho * u * u
    if cfg["nspec"]:
        U[0, 5, :, :, sl] = rho * X
    return orc.fill_ghosts(cfg, U)


@pytest.mark.parametrize("seed", [1, 2, 3])
def test_interface_floors_match_brute_force(seed):
    cfg = line_cfg(24, small_dens=0.66, small_pres=0.58)
    U = floor_state(cfg, seed)
    A = orc.advance_A(cfg, U)
    Ab, n_active = brute_force_line_A(cfg, U)
    assert n_active >= 4, "the floors must bind for this pin to mean anything"
    for c in range(6):
        assert np.array_equal(A[0, c, 0, 0, :], Ab[c]), c          # same operations in the same order
    # uniform in y and z: every line gives the same A
    assert np.array_equal(A, np.broadcast_to(A[:, :, :1, :1, :], A.shape))
    # and the floors matter: without them the result differs
    cfg0 = line_cfg(24, small_dens=1e-200, small_pres=1e-200)
    A0 = orc.advance_A(cfg0, U)
    assert np.abs(A - A0).max() > 1e-3 * np.abs(A0).max()


def test_density_floor_alone_and_pressure_floor_alone():
    """Density floor only: binds at interfaces and changes A.  Pressure floor only: the zone-centre floor
    of S1 (Q11) already lifts every zone to small_pres and the CW84 edges stay within the range of their
    neighbours (pin P10), so the INTERFACE pressure floor cannot bind beyond roundoff -- it is a guard, and
    the brute-force restatement confirms the oracle's A with it in place."""
    base = line_cfg(24, 1e-200, 1e-200)
    U = floor_state(base, 5)
    A0 = orc.advance_A(base, U)
    cfg = line_cfg(24, 0.66, 1e-200)
    A = orc.advance_A(cfg, U)
    Ab, n_active = brute_force_line_A(cfg, U)
    assert n_active >= 4
    assert np.array_equal(A[0, :, 0, 0, :], Ab)
    assert np.abs(A - A0).max() > 1e-4 * np.abs(A0).max()
    cfg = line_cfg(24, 1e-200, 0.58)
    A = orc.advance_A(cfg, U)
    Ab, n_active = brute_force_line_A(cfg, U)
    assert n_active == 0
    assert np.array_equal(A[0, :, 0, 0, :], Ab)
    assert np.abs(A - A0).max() > 1e-4 * np.abs(A0).max()      # through the zone-centre floor
