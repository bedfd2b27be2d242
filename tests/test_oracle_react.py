"""Pins of the reactive half of the oracle (oracle/orc_react.c): Eq. (2) of the paper with R != 0
 for the synthetic stiff chain of DESIGN.md readings R1-R4.
No test here calls the CUDA path."""
import numpy as np
import pytest
from scipy.integrate import solve_ivp

from oracle import orc
from paper_1910_12578_b200 import workloads as wl
from test_oracle_pins import small_cfg


def zone_state(ns, seed=1, rho=1.3, T=1.1, cv=1.5, v=(0.2, -0.1, 0.3)):
    rng = np.random.default_rng(seed)
    X = rng.dirichlet(np.ones(ns))
    ke = 0.5 * rho * sum(c * c for c in v)
    y = np.concatenate([rho * X, [rho * cv * T + ke]])
    return rho, ke, y


def rhs_python(react, ns, rho, ke, y):
    """R1-R2 written out again, independently of the C code."""
    T = (y[ns] - ke) / rho / react["cv"]
    lam = np.array(react["rate"][:ns]) * (T / react["T0"]) ** react["nu"]
    lam[ns - 1] = 0.0
    R = np.zeros(ns + 1)
    R[:ns] = -lam * y[:ns]
    R[1:ns] += lam[:ns - 1] * y[:ns - 1]
    R[ns] = np.sum(np.array(react["q"][:ns]) * lam * y[:ns])
    return R


def test_rhs_matches_an_independent_restatement_and_conserves_species():
    ns = 13
    react = wl.react_params(ns)
    rho, ke, y = zone_state(ns)
    R = orc.react_zone(react, rho, ke, y)
    assert np.allclose(R, rhs_python(react, ns, rho, ke, y), rtol=1e-13, atol=1e-15)
    assert abs(R[:ns].sum()) <= 1e-13 * np.abs(R[:ns]).sum()         # the chain only converts species
    assert R[ns] > 0                                                  # exothermic


def test_jacobian_against_finite_differences():
    ns = 6
    react = wl.react_params(ns, nu=4.0)
    rho, ke, y = zone_state(ns, seed=2)
    R0, J = orc.react_zone(react, rho, ke, y, jac=True)
    for j in range(ns + 1):
        h = 1e-6 * max(abs(y[j]), 1e-3)
        yp, ym = y.copy(), y.copy()
        yp[j] += h; ym[j] -= h
        fd = (orc.react_zone(react, rho, ke, yp) - orc.react_zone(react, rho, ke, ym)) / (2 * h)
        assert np.allclose(J[:, j], fd, rtol=2e-6, atol=1e-8 * np.abs(J).max()), j


def test_linear_chain_is_backward_euler_in_closed_form():
    """nu = 0: rates do not depend on T, the implicit equation is linear and Newton lands on
    X_0' = X_0 / (1 + dt l_0), X_k' = (X_k + dt l_{k-1} X_{k-1}') / (1 + dt l_k), E' = E + dt sum q l y'."""
    ns = 5
    react = wl.react_params(ns, nu=0.0, stiff=100.0)            # dt * rate up to 1e3: stiff
    rho, ke, c = zone_state(ns, seed=3)
    dt = 0.1
    y, it = orc.react_solve_zone(react, rho, ke, dt, c)
    lam = np.array(react["rate"][:ns]); lam[-1] = 0.0
    ex = np.zeros(ns + 1)
    prev = 0.0
    for k in range(ns):
        ex[k] = (c[k] + dt * prev) / (1 + dt * lam[k])
        prev = lam[k] * ex[k]
    ex[ns] = c[ns] + dt * np.sum(np.array(react["q"][:ns]) * lam * ex[:ns])
    assert it <= 3
    assert np.allclose(y, ex, rtol=1e-13, atol=1e-16)
    assert abs(y[:ns].sum() - c[:ns].sum()) <= 1e-14 * c[:ns].sum()


@pytest.mark.parametrize("nu,stiff", [(4.0, 1.0), (8.0, 30.0), (-2.0, 300.0)])
def test_converged_solve_satisfies_the_implicit_equation(nu, stiff):
    ns = 13
    react = wl.react_params(ns, nu=nu, stiff=stiff)
    rho, ke, c = zone_state(ns, seed=4)
    dt = 0.02
    y, it = orc.react_solve_zone(react, rho, ke, dt, c)
    assert it <= 12, it                                            # quadratic convergence (a wrong Jacobian crawls)
    res = y - c - dt * rhs_python(react, ns, rho, ke, y)
    assert np.abs(res[:ns]).max() <= 1e-13 * rho and abs(res[ns]) <= 1e-13 * abs(y[ns])
    assert abs(y[:ns].sum() - c[:ns].sum()) <= 1e-13 * c[:ns].sum()
    assert (y[:ns] > -1e-15).all()


def test_array_calls_agree_with_the_zone_calls_and_leave_ghosts_alone():
    cfg = small_cfg(n=(5, 4, 6), nb=(2, 1, 1), nspec=4, gamma=5 / 3)
    react = wl.react_params(4)
    rng = np.random.default_rng(7)
    U = orc.fill_ghosts(cfg, wl.random_state(cfg, 3))
    R = orc.react_R(cfg, react, U)
    assert np.all(R[:, :4] == 0.0)
    b, k, j, i = 1, 2, 3, 4
    z = U[b, :, k + 4, j + 4, i + 4]
    ke = 0.5 * (z[1] ** 2 + z[2] ** 2 + z[3] ** 2) / z[0]
    Rz = orc.react_zone(react, z[0], ke, np.concatenate([z[5:], z[4:5]]))
    assert np.array_equal(R[b, 5:, k, j, i], Rz[:4]) and R[b, 4, k, j, i] == Rz[4]
    # one node update with every term of Eq. (2) present
    A_new, A_old, A_q = (0.1 * rng.standard_normal(R.shape) for _ in range(3))
    R_old = orc.react_R(cfg, react, U * 1.0)
    dt = 0.01
    Un = np.full_like(U, 5.0)
    iters = np.zeros(R[:, 0].shape, dtype=np.int32)
    _, Rn = orc.sdc_update_react(cfg, react, Un, U, dt, A_new, A_old, R_old, [A_q, A_new], [R_old, R], [0.3 * dt, 0.2 * dt],
                                 iters=iters)
    mask = np.ones(Un.shape, bool); mask[:, :, 4:-4, 4:-4, 4:-4] = False
    assert np.all(Un[mask] == 5.0)
    assert iters.min() >= 1 and iters.max() <= 10
    c = U[b, :, k + 4, j + 4, i + 4] + dt * (A_new - A_old)[b, :, k, j, i] - dt * R_old[b, :, k, j, i] \
        + 0.3 * dt * (A_q + R_old)[b, :, k, j, i] + 0.2 * dt * (A_new + R)[b, :, k, j, i]
    un = Un[b, :, k + 4, j + 4, i + 4]
    assert np.allclose(un[:4], c[:4], rtol=1e-15, atol=1e-16)       # rho, rho v: explicit
    assert np.allclose(un - dt * Rn[b, :, k, j, i], c, rtol=1e-12, atol=1e-14)   # U' = c + dt R(U')
    assert np.array_equal(Rn, orc.react_R(cfg, react, Un))          # R_new_out is R of the new state


def reference_ode(react, ns, rho, ke, y0, t):
    sol = solve_ivp(lambda _, y: rhs_python(react, ns, rho, ke, y), (0.0, t), y0, method="Radau", rtol=1e-12, atol=1e-14)
    return sol.y[:, -1]


@pytest.mark.parametrize("M,K,order", [(2, 1, 1), (2, 2, 2), (3, 3, 3), (3, 4, 4)])
def test_sdc_with_reactions_reaches_the_order_of_its_quadrature(M, K, order):
    """Uniform state: <A(U)> = 0 bitwise, so the SDC step integrates dy/dt = R(y) in every zone.  Halving dt must
    divide the error by 2^order, and every iteration must raise the order by one up to the order of the quadrature
    (trapezoid -> 2nd, Simpson -> 4th order).  Measured ratios at the finest pair: 1.97, 3.79, 7.59,
    15.1 for (M, K) = (2, 1), (2, 2), (3, 3), (3, 4)."""
    ns = 3
    cfg = small_cfg(n=(4, 4, 4), nspec=ns, gamma=5 / 3)
    react = wl.react_params(ns, nu=3.0, stiff=0.05)
    rho, ke, y0 = zone_state(ns, seed=5, v=(0.0, 0.0, 0.0))
    U = np.zeros(wl.u_shape(cfg))
    U[0, 0] = rho
    U[0, 4] = y0[ns]
    for s in range(ns):
        U[0, 5 + s] = y0[s]
    T = 0.2
    ref = reference_ode(react, ns, rho, ke, y0, T)
    errs = []
    for nsteps in (4, 8, 16):
        V = U.copy()
        for _ in range(nsteps):
            V = orc.sdc_step_nodes_react(cfg, react, V, T / nsteps, M=M, K=K)
        z = V[0, :, 5, 6, 7]
        errs.append(np.abs(np.concatenate([z[5:], z[4:5]]) - ref).max())
        assert np.array_equal(V[0, :, 4:-4, 4:-4, 4:-4], np.broadcast_to(z[:, None, None, None], (5 + ns, 4, 4, 4)))
    r1, r2 = errs[0] / errs[1], errs[1] / errs[2]
    assert r2 > 0.88 * 2 ** order and r1 > 0.8 * 2 ** order, (errs, r1, r2)
