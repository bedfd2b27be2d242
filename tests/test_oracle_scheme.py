"""Scheme-level pins of the CPU oracle: ghost fill, <A(U)>, the SDC node update, the CFL step.

BASELINE.json north_star's four oracle checks (exact Sod, conservation, A(uniform) = 0,
permutation/mirror invariance) plus SURVEY.md 8(c) pins P3, P4, P6-P8, P11-P15.
CPU only; the CUDA path is never called here.
"""
import numpy as np
import pytest

from oracle import orc
from paper_1910_12578_b200 import workloads as wl
from test_oracle_pins import small_cfg, relmax


def state_from_prims(cfg, W):
    return wl.from_global(cfg, wl.cons_from_prim(cfg, W))


def uniform_W(cfg, vals):
    Dx, Dy, Dz = wl.domain(cfg)
    W = np.empty((wl.nvar(cfg), Dz, Dy, Dx))
    for c, v in enumerate(vals):
        W[c] = v
    return W


# --------------------------------------------------------------- P13: ghost fill, brute force ---
@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 1, 1), (2, 2, 2), (0, 1, 2)])
def test_P13_ghost_fill_bruteforce(bc):
    cfg = small_cfg(n=(4, 5, 6), nb=(2, 1, 2), nspec=1, bc=bc)
    Dx, Dy, Dz = wl.domain(cfg)
    N = wl.nvar(cfg)
    # value = unique code of (component, global zone): linear index + 1 (so sign flips are visible)
    G = (np.arange(N * Dz * Dy * Dx, dtype=np.float64) + 1.0).reshape(N, Dz, Dy, Dx)
    U = orc.fill_ghosts(cfg, wl.from_global(cfg, G))
    assert not np.isnan(U).any()

    def src(g, D, b):
        if 0 <= g < D:
            return g, 1
        if b == 0:
            return g % D, 1
        if b == 1:
            return min(max(g, 0), D - 1), 1
        return (-1 - g if g < 0 else 2 * D - 1 - g), -1
    ng = 4
    for bk in range(cfg["nbz"]):
        for bi in range(cfg["nbx"]):
            b = bi + cfg["nbx"] * (0 + cfg["nby"] * bk)
            for k in range(cfg["nz"] + 8):
                for j in range(cfg["ny"] + 8):
                    for i in range(cfg["nx"] + 8):
                        sx, fx = src(bi * cfg["nx"] + i - ng, Dx, bc[0])
                        sy, fy = src(j - ng, Dy, bc[1])
                        sz, fz = src(bk * cfg["nz"] + k - ng, Dz, bc[2])
                        exp = G[:, sz, sy, sx].copy()
                        exp[1] *= fx; exp[2] *= fy; exp[3] *= fz
                        assert np.array_equal(U[b, :, k, j, i], exp), (b, k, j, i)


def test_P13_box_lattice_equals_single_box_bitwise():
    c1 = small_cfg(n=(16, 16, 16), nb=(1, 1, 1), nspec=2, gamma=5 / 3, bc=(0, 1, 2), grav=(0, 0, -1.0))
    c8 = small_cfg(n=(8, 8, 8), nb=(2, 2, 2), nspec=2, gamma=5 / 3, bc=(0, 1, 2), grav=(0, 0, -1.0))
    U1 = wl.random_state(c1, 3)
    G = wl.to_global(c1, U1, ghosted=True)
    U8 = wl.from_global(c8, G)
    A1 = orc.advance_A(c1, orc.fill_ghosts(c1, U1))
    A8 = orc.advance_A(c8, orc.fill_ghosts(c8, U8))
    assert np.array_equal(wl.to_global(c1, A1), wl.to_global(c8, A8))
    assert orc.cfl_dt(c1, U1, 0.5) == orc.cfl_dt(c8, U8, 0.5)


# --------------------------------------------------------------- P4 / P6: exact zeros -----------
def test_P4_uniform_state_gives_zero_A_bitwise():
    cfg = small_cfg(n=(8, 6, 5), nspec=2, gamma=5 / 3)
    U = state_from_prims(cfg, uniform_W(cfg, [1.3, 0.7, -0.4, 0.2, 0.9, 0.25, 0.75]))
    A = orc.advance_A(cfg, orc.fill_ghosts(cfg, U))
    assert np.all(A == 0.0)


def test_P6_stationary_contact_gives_zero_A_bitwise():
    cfg = small_cfg(n=(16, 8, 8), bc=(1, 1, 1), nspec=1)
    W = uniform_W(cfg, [1.0, 0, 0, 0, 1.0, 1.0])
    W[0, :, :, 8:] = 0.125
    W[5, :, :, 8:] = 0.3
    A = orc.advance_A(cfg, orc.fill_ghosts(cfg, state_from_prims(cfg, W)))
    assert np.all(A == 0.0)


# --------------------------------------------------------------- P3: conservation ---------------
def test_P3_conservation_periodic():
    cfg = small_cfg(n=(12, 12, 12), nspec=3, gamma=5 / 3)
    U = orc.fill_ghosts(cfg, wl.random_state(cfg, 1))
    A = orc.advance_A(cfg, U)
    for c in range(wl.nvar(cfg)):
        assert abs(A[:, c].sum()) <= 1e-13 * np.abs(A[:, c]).sum()
    # and the total of every conserved component is constant over SDC steps
    tot0 = wl.to_global(cfg, U, ghosted=True).sum(axis=(1, 2, 3))
    for _ in range(3):
        U = orc.sdc_step_2nd(cfg, U, orc.cfl_dt(cfg, U, 0.5))
    tot1 = wl.to_global(cfg, U, ghosted=True).sum(axis=(1, 2, 3))
    absT = np.abs(wl.to_global(cfg, U, ghosted=True)).sum(axis=(1, 2, 3))
    assert np.all(np.abs(tot1 - tot0) <= 1e-13 * absT)


# --------------------------------------------------------------- P7: permutation / mirror -------
def permute_state(G, perm):
    """G[c, z, y, x] -> state seen in axes relabelled so that new axis d = old axis perm[d]."""
    # spatial axes of G are (z,y,x) = array axes (1,2,3); direction d lives on array axis 3-d
    ax = [0] + [3 - perm[2 - a] + 0 for a in range(3)]
    H = np.transpose(G, ax).copy()
    out = H.copy()
    for d in range(3):
        out[1 + d] = H[1 + perm[d]]
    return out


@pytest.mark.parametrize("perm", [(1, 0, 2), (2, 1, 0), (1, 2, 0)])
def test_P7_axis_permutation_invariance(perm):
    n = (6, 8, 10)
    cfg = small_cfg(n=n, nspec=2, gamma=5 / 3, L=(0.6, 0.8, 1.0))
    np_ = tuple(n[perm[d]] for d in range(3))
    Lp = tuple((0.6, 0.8, 1.0)[perm[d]] for d in range(3))
    cfgp = small_cfg(n=np_, nspec=2, gamma=5 / 3, L=Lp)
    U = wl.random_state(cfg, 7)
    G = wl.to_global(cfg, U, ghosted=True)
    A = wl.to_global(cfg, orc.advance_A(cfg, orc.fill_ghosts(cfg, U)))
    Up = wl.from_global(cfgp, permute_state(G, perm))
    Ap = wl.to_global(cfgp, orc.advance_A(cfgp, orc.fill_ghosts(cfgp, Up)))
    ref = permute_state(A, perm)
    err = np.abs(Ap - ref).max(axis=(1, 2, 3)) / np.abs(ref).max(axis=(1, 2, 3))
    assert err.max() <= 1e-14, err


@pytest.mark.parametrize("d", [0, 1, 2])
def test_P7_mirror_invariance(d):
    cfg = small_cfg(n=(8, 8, 8), nspec=1, gamma=1.4)
    U = wl.random_state(cfg, 8)
    G = wl.to_global(cfg, U, ghosted=True)
    A = wl.to_global(cfg, orc.advance_A(cfg, orc.fill_ghosts(cfg, U)))

    def mirror(X):
        M = np.flip(X, axis=3 - d).copy()
        M[1 + d] *= -1
        return M
    Am = wl.to_global(cfg, orc.advance_A(cfg, orc.fill_ghosts(cfg, wl.from_global(cfg, mirror(G)))))
    ref = mirror(A)
    err = np.abs(Am - ref).max(axis=(1, 2, 3)) / np.abs(ref).max(axis=(1, 2, 3))
    assert err.max() <= 1e-14, err


def test_P7_xy_symmetric_state_stays_bitwise_symmetric():
    cfg = wl.make_config(1, n=16)
    U = orc.fill_ghosts(cfg, wl.initial_state(cfg))
    for _ in range(5):
        U = orc.sdc_step_2nd(cfg, U, orc.cfl_dt(cfg, U, 0.5))
    G = wl.to_global(cfg, U, ghosted=True)
    S = np.transpose(G, (0, 1, 3, 2)).copy()
    S[[1, 2]] = S[[2, 1]]
    assert np.array_equal(G, S)


# --------------------------------------------------------------- P8: species --------------------
def test_P8_uniform_species_follow_mass():
    cfg = small_cfg(n=(8, 8, 8), nspec=2, gamma=5 / 3)
    U = wl.random_state(cfg, 9)
    G = wl.to_global(cfg, U, ghosted=True)
    G[5] = 0.3 * G[0]
    G[6] = 0.7 * G[0]
    A = orc.advance_A(cfg, orc.fill_ghosts(cfg, wl.from_global(cfg, G)))
    scale = np.abs(A[:, 0]).max()
    assert np.abs(A[:, 5] - 0.3 * A[:, 0]).max() <= 1e-13 * scale
    assert np.abs(A[:, 6] - 0.7 * A[:, 0]).max() <= 1e-13 * scale


# --------------------------------------------------------------- P11: gravity source ------------
def test_P11_hydrostatic_residual_fourth_order_and_sign():
    H, res = 1.0 / 8.0, []
    for nz in (32, 64, 128):
        cfg = small_cfg(n=(4, 4, nz), bc=(0, 0, 2), gamma=5 / 3, L=(4.0 / nz, 4.0 / nz, 1.0), grav=(0, 0, -1 / H))
        W = uniform_W(cfg, [1, 0, 0, 0, 1])
        z = (np.arange(nz) + 0.5) / nz
        W[0] = np.exp(-z / H)[:, None, None]
        W[4] = W[0]
        U = orc.fill_ghosts(cfg, state_from_prims(cfg, W))
        A = wl.to_global(cfg, orc.advance_A(cfg, U))
        rho = W[0]
        r = np.abs(A[3]) / (rho / H)
        res.append(r[nz // 4: 3 * nz // 4].max())
        assert np.all(A[1] == 0) and np.all(A[2] == 0)
        assert np.abs(A[0][nz // 4: 3 * nz // 4]).max() < 1e-3 * rho.max()
    assert res[0] / res[1] >= 12 and res[1] / res[2] >= 12, res
    assert res[2] < 1e-6, res
    # energy source: S[rho E] = rho v . g (uniform flow, no gradients, periodic => A = S exactly)
    cfg = small_cfg(n=(4, 4, 4), gamma=1.4, grav=(0.5, -0.25, 2.0))
    U = orc.fill_ghosts(cfg, state_from_prims(cfg, uniform_W(cfg, [2.0, 0.3, 0.2, -0.1, 1.0])))
    A = orc.advance_A(cfg, U)
    assert np.allclose(A[0, 1], 2.0 * 0.5, rtol=1e-15) and np.allclose(A[0, 3], 2.0 * 2.0, rtol=1e-15)
    assert np.allclose(A[0, 4], 2.0 * (0.3 * 0.5 - 0.2 * 0.25 - 0.1 * 2.0), rtol=1e-14)
    assert np.all(A[0, 0] == 0)


# --------------------------------------------------------------- P12: SDC update ----------------
def test_P12_sdc_update_formula_and_heun():
    cfg = small_cfg(n=(4, 5, 6), nspec=1)
    rng = np.random.default_rng(12)
    Um = rng.normal(size=orc.u_shape(cfg))
    An, Ao, A1, A2 = (rng.normal(size=orc.a_shape(cfg)) for _ in range(4))
    Un = np.full(orc.u_shape(cfg), 7.0)
    orc.sdc_update(cfg, Un, Um, 0.1, An, Ao, [Ao, A1, A2], [0.01, 0.02, -0.03])
    inner = (slice(None), slice(None), slice(4, -4), slice(4, -4), slice(4, -4))
    exp = Um[inner] + 0.1 * (An - Ao) + (0.01 * Ao + 0.02 * A1 - 0.03 * A2)
    assert np.abs(Un[inner] - exp).max() <= 1e-15
    mask = np.ones(Un.shape, bool); mask[inner] = False
    assert np.all(Un[mask] == 7.0)                           # ghosts untouched (Q28)


def test_P12_two_node_two_iteration_sdc_is_heun():
    """M = 2, K = 2, R = 0 (trapezoid) reduces to Heun's method."""
    cfg = wl.make_config(3, n=8, nspec=2)
    U0 = orc.fill_ghosts(cfg, wl.initial_state(cfg))
    dt = orc.cfl_dt(cfg, U0, 0.5)
    U2 = orc.sdc_step_2nd(cfg, U0, dt)
    inner = (slice(None), slice(None), slice(4, -4), slice(4, -4), slice(4, -4))
    A0 = orc.advance_A(cfg, U0)
    Ue = U0.copy(); Ue[inner] = U0[inner] + dt * A0
    A1 = orc.advance_A(cfg, orc.fill_ghosts(cfg, Ue))
    heun = U0[inner] + 0.5 * dt * (A0 + A1)
    assert np.abs(U2[inner] - heun).max() <= 1e-14 * np.abs(heun).max()


def test_P12_linear_ode_amplification_and_simpson_rows():
    """With A = lambda U the 2-node scheme multiplies by 1 + z + z^2/2; the 3-node weight rows of
    DESIGN.md Q17 integrate quadratics exactly over each sub-interval."""
    cfg = small_cfg(n=(4, 4, 4))
    lam, dt = -0.7, 0.3
    z = lam * dt
    U0 = np.ones(orc.u_shape(cfg)); A0 = lam * U0[:, :, 4:-4, 4:-4, 4:-4].copy()
    U1 = U0.copy(); orc.sdc_update(cfg, U1, U0, dt, A0, A0, [A0, A0], [dt / 2, dt / 2])
    A1 = lam * U1[:, :, 4:-4, 4:-4, 4:-4].copy()
    U2 = U0.copy(); orc.sdc_update(cfg, U2, U0, dt, A0, A0, [A0, A1], [dt / 2, dt / 2])
    assert np.allclose(U2[:, :, 4:-4, 4:-4, 4:-4], 1 + z + z * z / 2, rtol=1e-15)
    w0 = dt * np.array([5, 8, -1]) / 24.0
    w1 = dt * np.array([-1, 8, 5]) / 24.0
    f = lambda t: 2.0 - 3.0 * t + 4.0 * t * t
    F = lambda t: 2.0 * t - 1.5 * t * t + 4.0 * t ** 3 / 3
    nodes = np.array([0, dt / 2, dt])
    Aq = [np.full(orc.a_shape(cfg), f(t)) for t in nodes]
    Z = np.zeros(orc.a_shape(cfg))
    Ua = np.zeros(orc.u_shape(cfg)); orc.sdc_update(cfg, Ua, np.zeros(orc.u_shape(cfg)), dt / 2, Z, Z, Aq, w0)
    Ub = np.zeros(orc.u_shape(cfg)); orc.sdc_update(cfg, Ub, np.zeros(orc.u_shape(cfg)), dt / 2, Z, Z, Aq, w1)
    assert np.allclose(Ua[0, 0, 5, 5, 5], F(dt / 2) - F(0), rtol=1e-14)
    assert np.allclose(Ub[0, 0, 5, 5, 5], F(dt) - F(dt / 2), rtol=1e-14)


# --------------------------------------------------------------- P14: CFL -----------------------
def test_P14_cfl_closed_form():
    cfg = small_cfg(n=(4, 6, 8), gamma=5 / 3, L=(1.0, 3.0, 2.0))
    U = state_from_prims(cfg, uniform_W(cfg, [2.0, 0.3, -0.5, 0.1, 1.5]))
    c = np.sqrt(5 / 3 * 1.5 / 2.0)
    exp = 0.4 / ((0.3 + c) / cfg["dx"] + (0.5 + c) / cfg["dy"] + (0.1 + c) / cfg["dz"])
    assert abs(orc.cfl_dt(cfg, U, 0.4) - exp) <= 1e-15 * exp
    # the max is over interior zones: one fast zone decides; ghosts (NaN here) are ignored
    W = uniform_W(cfg, [2.0, 0.3, -0.5, 0.1, 1.5]); W[3, 5, 2, 1] = -4.0
    exp2 = 0.4 / ((0.3 + c) / cfg["dx"] + (0.5 + c) / cfg["dy"] + (4.0 + c) / cfg["dz"])
    assert abs(orc.cfl_dt(cfg, state_from_prims(cfg, W), 0.4) - exp2) <= 1e-15 * exp2


# --------------------------------------------------------------- P1: exact Sod ------------------
def run_sod_1d(nx, t_end=0.2):
    cfg = small_cfg(n=(nx, 4, 4), bc=(1, 0, 0), gamma=1.4, L=(1.0, 4.0 / nx, 4.0 / nx))
    W = uniform_W(cfg, [1, 0, 0, 0, 1])
    x = (np.arange(nx) + 0.5) / nx
    W[0] = np.where(x < 0.5, 1.0, 0.125)[None, None, :]
    W[4] = np.where(x < 0.5, 1.0, 0.1)[None, None, :]
    U = orc.fill_ghosts(cfg, state_from_prims(cfg, W))
    t = 0.0
    while t < t_end - 1e-14:
        dt = min(orc.cfl_dt(cfg, U, 0.5), t_end - t)
        U = orc.sdc_step_2nd(cfg, U, dt)
        t += dt
    rho = wl.to_global(cfg, U, ghosted=True)[0]
    assert np.abs(rho - rho[0:1, 0:1, :]).max() == 0.0                  # stays 1-D bitwise
    # exact cell averages by 8-point midpoint sampling of each zone
    sub = (np.arange(8) + 0.5) / 8
    xs = ((np.arange(nx)[:, None] + sub[None, :]) / nx - 0.5) / t_end
    re, _, _ = orc.exact_riemann_sample(1.4, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, xs.ravel())
    return np.abs(rho[0, 0] - re.reshape(nx, 8).mean(axis=1)).mean()


def test_P1_sod_L1_error_falls_with_resolution():
    e = [run_sod_1d(n) for n in (32, 64, 128)]
    assert e[0] / e[1] >= 1.7 and e[1] / e[2] >= 1.7, e
    assert e[2] < 4e-3, e


@pytest.mark.slow
def test_P1_sod_L1_error_fine():
    e256 = run_sod_1d(256)
    assert e256 < 2e-3, e256


# --------------------------------------------------------------- P15: second order --------------
def pulse_error(n, t_end=0.05):
    cfg = wl.make_config(2, n=n)
    U = orc.fill_ghosts(cfg, wl.initial_state(cfg))
    t = 0.0
    while t < t_end - 1e-14:
        dt = min(orc.cfl_dt(cfg, U, 0.5), t_end - t)
        U = orc.sdc_step_2nd(cfg, U, dt)
        t += dt
    G = wl.to_global(cfg, U, ghosted=True)
    x = (np.arange(n) + 0.5) / n
    X, Y, Z = np.meshgrid(x, x, x, indexing="ij")   # any labelling: the pulse is symmetric
    r2 = sum((((c - t_end - 0.5 + 0.5) % 1.0) - 0.5) ** 2 for c in (X, Y, Z))
    exact = 1 + 0.5 * np.exp(-r2 / 0.01)
    p = (cfg["gamma"] - 1) * (G[4] - 0.5 * (G[1] ** 2 + G[2] ** 2 + G[3] ** 2) / G[0])
    return np.abs(G[0] - exact).mean(), np.abs(p - 1).max(), np.abs(G[1] / G[0] - 1).max()


def test_P15_smooth_pulse_second_order():
    (e16, _, _), (e32, p32, v32) = pulse_error(16), pulse_error(32)
    assert p32 < 1e-13 and v32 < 1e-13            # p and v stay uniform to roundoff
    assert e16 / e32 >= 2.5, (e16, e32)


@pytest.mark.slow
def test_P15_smooth_pulse_second_order_fine():
    (e32, _, _), (e64, _, _) = pulse_error(32), pulse_error(64)
    assert e32 / e64 >= 3.5, (e32, e64)


# --------------------------------------------------------------- SDC with M nodes, K iterations --
def _linear_ode_error(M, K, dt, lam=-1.3):
    """one step of U' = lam U with the oracle's node driver; returns |U_1 - exp(lam dt)|"""
    cfg = small_cfg(n=(4, 4, 4))
    U0 = np.ones(orc.u_shape(cfg))
    A_fn = lambda V: lam * V[:, :, 4:-4, 4:-4, 4:-4].copy()
    U1 = orc.sdc_step_nodes(cfg, U0, dt, M=M, K=K, A_fn=A_fn)
    return abs(U1[0, 0, 5, 5, 5] - np.exp(lam * dt))


@pytest.mark.parametrize("M,K,order", [(2, 1, 1), (2, 2, 2), (3, 1, 1), (3, 2, 2), (3, 3, 3), (3, 4, 4), (3, 6, 4)])
def test_sdc_iterations_raise_the_order_up_to_the_quadrature(M, K, order):
    """"each iteration ... increases the temporal order by one up to the order of the
    integral"; L44: trapezoid -> 2nd order, Simpson -> 4th.  Local error of one step ~ dt^(order+1)."""
    e1, e2 = _linear_ode_error(M, K, 0.2), _linear_ode_error(M, K, 0.1)
    rate = np.log2(e1 / e2)
    assert abs(rate - (order + 1)) < 0.25, (M, K, rate)


def test_node_driver_with_two_nodes_is_the_second_order_step():
    cfg = small_cfg(n=(8, 6, 5), nspec=1, gamma=5 / 3)
    U = wl.random_state(cfg, 51)
    dt = 0.3 * orc.cfl_dt(cfg, orc.fill_ghosts(cfg, U.copy()), 1.0)
    a, b = orc.sdc_step_2nd(cfg, U, dt), orc.sdc_step_nodes(cfg, U, dt, M=2, K=2)
    inner = (slice(None), slice(None), slice(4, -4), slice(4, -4), slice(4, -4))
    assert np.abs(a[inner] - b[inner]).max() <= 1e-14 * np.abs(a[inner]).max()


def test_lobatto_weights_closed_form():
    c, w = orc.lobatto_nodes_weights(3)
    assert np.allclose(w, np.array([[5, 8, -1], [-1, 8, 5]]) / 24.0, atol=1e-15)
    assert np.allclose(orc.lobatto_nodes_weights(2)[1], [[0.5, 0.5]], atol=1e-15)
