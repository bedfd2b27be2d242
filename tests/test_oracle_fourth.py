"""Pins of the oracle's fourth-order finite-volume <A(U)> (oracle/orc_fourth.c, readings G1-G9; "a
fourth-order method in space and time (using ... the spatial reconstruction of [12])").
No test here calls the CUDA path."""
import numpy as np
import pytest
from numpy.polynomial.legendre import leggauss
from scipy.special import erf

from oracle import orc
from paper_1910_12578_b200 import workloads as wl
from test_oracle_pins import small_cfg, relmax
from test_oracle_scheme import uniform_W, state_from_prims

G = 5.0 / 3.0
GR = np.array([0.1, -0.2, 0.3])
TP = 2 * np.pi


# ------------------------------------------------ an analytic smooth state and its EXACT finite-volume RHS ----
def prim(x, y, z):
    rho = 1 + 0.2 * np.sin(TP * (x + 0.3)) * np.cos(TP * y) + 0.1 * np.sin(TP * z)
    u = 0.3 + 0.1 * np.sin(TP * (y + z))
    v = -0.2 + 0.1 * np.cos(TP * (x - z))
    w = 0.1 + 0.1 * np.sin(TP * (x + y))
    p = 1 + 0.2 * np.cos(TP * (x + y + z))
    X0 = 0.5 + 0.3 * np.sin(TP * x) * np.sin(TP * y)
    return np.stack([rho, u, v, w, p, X0, 1 - X0])


def cons(W):
    rho, u, v, w, p = W[:5]
    return np.stack([rho, rho * u, rho * v, rho * w, p / (G - 1) + 0.5 * rho * (u * u + v * v + w * w), rho * W[5], rho * W[6]])


def flux(W, d):
    U = cons(W)
    F = U * W[1 + d]
    F[1 + d] += W[4]
    F[4] += W[4] * W[1 + d]
    return F


def src(W):
    U = cons(W)
    S = np.zeros_like(U)
    for d in range(3):
        S[1 + d] = U[0] * GR[d]
        S[4] += U[1 + d] * GR[d]
    return S


def exact_fv(n, nq=6):
    """Cell averages of U and the exact cell average of -div F + S on an n^3 grid of the unit cube, by Gauss-Legendre
    quadrature (6 points per direction: error ~1e-12 here) of the analytic fields -- the definition of the
    finite-volume right-hand side, written out."""
    xg, wg = leggauss(nq)
    xg, wg = 0.5 * (xg + 1), 0.5 * wg
    h = 1.0 / n
    c = ((np.arange(n)[:, None] + xg[None, :]) * h).ravel()
    f = np.arange(n + 1) * h
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    W3 = np.einsum("k,j,i->kji", wg, wg, wg)
    W2 = np.einsum("b,a->ba", wg, wg)
    cell = lambda fn: np.einsum("cakbjdi,kji->cabd", fn(prim(X, Y, Z)).reshape(-1, n, nq, n, nq, n, nq), W3)
    Uavg, A = cell(cons), cell(src)
    Zq, Yq, Xq = np.meshgrid(c, c, f, indexing="ij")
    Ff = np.einsum("cakbjf,kj->cabf", flux(prim(Xq, Yq, Zq), 0).reshape(-1, n, nq, n, nq, n + 1), W2)
    A -= (Ff[:, :, :, 1:] - Ff[:, :, :, :-1]) / h
    Zq, Yq, Xq = np.meshgrid(c, f, c, indexing="ij")
    Ff = np.einsum("cakfbi,ki->cafb", flux(prim(Xq, Yq, Zq), 1).reshape(-1, n, nq, n + 1, n, nq), W2)
    A -= (Ff[:, :, 1:, :] - Ff[:, :, :-1, :]) / h
    Zq, Yq, Xq = np.meshgrid(f, c, c, indexing="ij")
    Ff = np.einsum("cfajbi,ji->cfab", flux(prim(Xq, Yq, Zq), 2).reshape(-1, n + 1, n, nq, n, nq), W2)
    A -= (Ff[:, 1:, :, :] - Ff[:, :-1, :, :]) / h
    return Uavg, A


def test_A4_converges_to_the_exact_finite_volume_rhs_at_fourth_order():
    """Measured: max-norm errors 1.1e-2, 1.7e-4, 1.04e-5 at 12^3, 24^3, 48^3 (ratios 69, 15.9); the second-order path
    on the same data: 0.57, 0.28, 0.14."""
    e4, l4, e2 = [], [], []
    for n in (12, 24, 48):
        cfg = small_cfg(n=(n, n, n), nspec=2, gamma=G, grav=tuple(GR))
        Uavg, Aex = exact_fv(n)
        U = orc.fill_ghosts(cfg, wl.from_global(cfg, Uavg))
        A4, A2 = wl.to_global(cfg, orc.advance_A4(cfg, U)), wl.to_global(cfg, orc.advance_A(cfg, U))
        den = np.abs(Aex).max(axis=(1, 2, 3))
        e4.append((np.abs(A4 - Aex).max(axis=(1, 2, 3)) / den).max())
        l4.append((np.abs(A4 - Aex).mean(axis=(1, 2, 3)) / den).max())
        e2.append((np.abs(A2 - Aex).max(axis=(1, 2, 3)) / den).max())
    assert e4[1] / e4[2] > 14.0 and l4[1] / l4[2] > 14.0, (e4, l4)
    assert e4[2] < 2e-5 and e4[2] < 1e-3 * e2[2], (e4, e2)          # and it is a different scheme from the PPM path


# ------------------------------------------------------------------------------ invariants ----
def test_uniform_state_conservation_and_lattice():
    cfg = small_cfg(n=(8, 6, 5), nspec=2, gamma=1.4)
    Uu = orc.fill_ghosts(cfg, state_from_prims(cfg, uniform_W(cfg, [1.3, 0.4, -0.2, 0.1, 0.7, 0.25, 0.75])))
    Au = orc.advance_A4(cfg, Uu)
    assert np.abs(Au).max() <= 1e-13                              # (7/12)(q+q) - (1/12)(q+q) is q only to roundoff
    U = orc.fill_ghosts(cfg, wl.random_state(cfg, 91))
    A = orc.advance_A4(cfg, U)
    for c in range(wl.nvar(cfg)):
        assert abs(A[:, c].sum()) <= 1e-12 * np.abs(A[:, c]).sum()
    one = small_cfg(n=(16, 8, 8), nspec=1, gamma=1.4, bc=(1, 0, 2), grav=(0.0, 0.0, -0.3))
    cut = small_cfg(n=(8, 4, 8), nb=(2, 2, 1), nspec=1, gamma=1.4, bc=(1, 0, 2), grav=(0.0, 0.0, -0.3))
    Gs = wl.to_global(one, wl.random_state(one, 92), ghosted=True)
    A1 = orc.advance_A4(one, orc.fill_ghosts(one, wl.from_global(one, Gs)))
    A2 = orc.advance_A4(cut, orc.fill_ghosts(cut, wl.from_global(cut, Gs)))
    assert np.array_equal(wl.to_global(one, A1), wl.to_global(cut, A2))


def test_permutation_and_mirror_invariance():
    cfg = small_cfg(n=(10, 10, 10), nspec=1, gamma=1.4)
    Gs = wl.to_global(cfg, wl.random_state(cfg, 93), ghosted=True)
    A = wl.to_global(cfg, orc.advance_A4(cfg, orc.fill_ghosts(cfg, wl.from_global(cfg, Gs))))
    Gp = Gs.transpose(0, 3, 2, 1).copy()
    Gp[[1, 3]] = Gp[[3, 1]]
    Ap = wl.to_global(cfg, orc.advance_A4(cfg, orc.fill_ghosts(cfg, wl.from_global(cfg, Gp)))).transpose(0, 3, 2, 1).copy()
    Ap[[1, 3]] = Ap[[3, 1]]
    assert np.abs(A - Ap).max() <= 1e-13 * np.abs(A).max()
    Gm = Gs[:, :, :, ::-1].copy()
    Gm[1] *= -1.0
    Am = wl.to_global(cfg, orc.advance_A4(cfg, orc.fill_ghosts(cfg, wl.from_global(cfg, Gm))))[:, :, :, ::-1].copy()
    Am[1] *= -1.0
    assert np.abs(A - Am).max() <= 1e-13 * np.abs(A).max()


# ------------------------------------------------------------------------------ the limiter (G4-G5) on lines ----
def cell_avg_1d(F, n, a=0.0, b=1.0):
    """cell averages of f = F' on n zones of [a, b], from its antiderivative F"""
    e = np.linspace(a, b, n + 1)
    return (F(e[1:]) - F(e[:-1])) / (e[1] - e[0]), e


def test_limiter_leaves_smooth_data_alone_and_reproduces_cubics():
    # a cubic: the (7/12, -1/12) interpolant of cell averages is the exact point value at the face
    q, e = cell_avg_1d(lambda x: x ** 4 / 4 - 0.3 * x ** 3 + 0.2 * x ** 2 + x, 24, 1.0, 2.0)
    f = lambda x: x ** 3 - 0.9 * x ** 2 + 0.4 * x + 1
    qm, qp = orc.ppm4_line(q)
    assert np.allclose(qp[2:-2], f(e[3:-2]), rtol=1e-13) and np.allclose(qm[2:-2], f(e[2:-3]), rtol=1e-13)
    # smooth monotone data: edges are the unlimited face values, and the parabolas join continuously
    q, e = cell_avg_1d(np.exp, 32)
    qm, qp = orc.ppm4_line(q)
    qf = (7 / 12) * (q[1:-2] + q[2:-1]) - (1 / 12) * (q[:-3] + q[3:])          # faces 3/2 .. n-5/2
    assert np.allclose(qp[2:-3], qf[1:-1], rtol=1e-14) and np.allclose(qm[3:-2], qf[1:-1], rtol=1e-14)
    # a well-resolved smooth extremum keeps its edges (no clipping, unlike CW84): still the unlimited face values
    q, e = cell_avg_1d(lambda x: np.sin(TP * x) / TP, 64)                      # f = cos(2 pi x): maximum at x = 0 / 1, minimum at 1/2
    qm, qp = orc.ppm4_line(q)
    qf = (7 / 12) * (q[1:-2] + q[2:-1]) - (1 / 12) * (q[:-3] + q[3:])
    assert np.allclose(qp[2:-3], qf[1:-1], rtol=1e-12, atol=1e-14)


def test_limiter_keeps_a_step_monotone_and_flattens_a_one_zone_spike():
    q = np.array([1.0] * 8 + [0.0] * 8)
    qm, qp = orc.ppm4_line(q)
    lo, hi = np.minimum(q[1:-3], q[3:-1]), np.maximum(q[1:-3], q[3:-1])        # neighbours of zones 2..n-3
    for edge in (qm[2:-2], qp[2:-2]):
        assert (edge >= np.minimum(lo, q[2:-2]) - 1e-15).all() and (edge <= np.maximum(hi, q[2:-2]) + 1e-15).all()
    assert ((qp[2:-2] - q[2:-2]) * (q[2:-2] - qm[2:-2]) >= -1e-30).all()       # every parabola monotone
    s = np.zeros(16); s[8] = 1.0                                               # an under-resolved extremum is flattened
    qm, qp = orc.ppm4_line(s)
    assert qm[8] == 1.0 and qp[8] == 1.0


# ------------------------------------------------------------------------------ space and time together ----
def pulse_avg(n, t, amp=0.5, s2=0.02):
    """cell averages of rho = 1 + amp exp(-r^2 / s2) advected by v = (1, 1, 1) for a time t (periodic unit cube)"""
    e = np.arange(n + 1) / n
    c = (0.5 + t) % 1.0
    g = np.zeros(n)
    for m in (-1, 0, 1):
        a = (e - c - m) / np.sqrt(s2)
        g += 0.5 * np.sqrt(np.pi * s2) * (erf(a[1:]) - erf(a[:-1])) * n
    return 1 + amp * g[:, None, None] * g[None, :, None] * g[None, None, :]


def run_pulse(n, M, K, A_fn, t_end=0.05):
    cfg = small_cfg(n=(n, n, n), gamma=G)
    rho = pulse_avg(n, 0.0)
    U = orc.fill_ghosts(cfg, wl.from_global(cfg, np.stack([rho, rho, rho, rho, 1.0 / (G - 1) + 1.5 * rho])))
    t = 0.0
    while t < t_end - 1e-14:
        dt = min(orc.cfl_dt(cfg, U, 0.5), t_end - t)
        U = orc.sdc_step_nodes(cfg, U, dt, M=M, K=K, A_fn=lambda V: A_fn(cfg, V))
        t += dt
    return np.abs(wl.to_global(cfg, U, ghosted=True)[0] - pulse_avg(n, t_end)).mean()


def test_fourth_order_in_space_and_time():
    """Simpson's rule + the reconstruction of [12].  Measured: L1(rho) 1.86e-4 -> 1.20e-5 from 16^3 to
    32^3 (ratio 15.5) with 3 nodes / 4 iterations; the second-order method on the same cell averages: 5.2e-4 -> 1.4e-4."""
    e16, e32 = run_pulse(16, 3, 4, orc.advance_A4), run_pulse(32, 3, 4, orc.advance_A4)
    assert e16 / e32 > 13.0, (e16, e32)
    assert e32 < 0.15 * run_pulse(32, 2, 2, orc.advance_A)
