"""ctypes wrapper of the CPU oracle oracle/liborc.so (TEST INFRASTRUCTURE, not the product).

Argument marshalling only; every formula lives in oracle/orc.c, which cites the
passages of PAPER.md / DESIGN.md it follows.  Arrays are C-contiguous float64 numpy
arrays in the layout U[b][c][k][j][i] (ghosted) and A[b][c][k][j][i] (interior).
"""
import ctypes as C

import numpy as np

from . import build as _build


class OrcParams(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("ng", C.c_int),
                ("nbx", C.c_int), ("nby", C.c_int), ("nbz", C.c_int), ("nspec", C.c_int),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("gamma", C.c_double), ("grav", C.c_double * 3),
                ("bc_lo", C.c_int * 3), ("bc_hi", C.c_int * 3),
                ("small_dens", C.c_double), ("small_pres", C.c_double)]


MAX_REACT = 15


class OrcReact(C.Structure):
    """orc_react of oracle/orc_react.c: the synthetic stiff network (readings R1-R4)."""
    _fields_ = [("cv", C.c_double), ("T0", C.c_double), ("nu", C.c_double),
                ("rate", C.c_double * MAX_REACT), ("q", C.c_double * MAX_REACT),
                ("max_iter", C.c_int), ("tol", C.c_double)]


_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        P = C.POINTER(OrcParams)
        _lib.orc_fill_ghosts.argtypes = [P, _dp]
        _lib.orc_advance_A.argtypes = [P, _dp, _dp]
        _lib.orc_advance_A_flat.argtypes = [P, _dp, _dp]
        _lib.orc_advance_A4.argtypes = [P, _dp, _dp]
        _lib.orc_advance_ctu.argtypes = [P, _dp, C.c_double, _dp]
        _lib.orc_ppm4_line.argtypes = [C.c_int, _dp, _dp, _dp]
        _lib.orc_ppm4_line.restype = None
        _lib.orc_flatten_line.argtypes = [C.c_int, _dp, _dp, C.c_double, _dp]
        _lib.orc_flatten_line.restype = None
        _lib.orc_sdc_update.argtypes = [P, _dp, _dp, C.c_double, _dp, _dp, C.c_int,
                                        C.POINTER(_dp), _dp]
        _lib.orc_cfl_dt.argtypes = [P, _dp, C.c_double, _dp]
        _lib.orc_cons_to_prim.argtypes = [C.c_int, C.c_double, C.c_double, _dp, _dp]
        _lib.orc_cons_to_prim.restype = None
        _lib.orc_ppm_line.argtypes = [C.c_int, _dp, _dp, _dp]
        _lib.orc_ppm_line.restype = None
        _lib.orc_hllc.argtypes = [C.c_int, C.c_int, C.c_double, _dp, _dp, _dp]
        _lib.orc_hllc.restype = None
        _lib.orc_wave_speeds.argtypes = [C.c_double] * 8 + [_dp, _dp]
        _lib.orc_wave_speeds.restype = None
        _lib.orc_pvrs_pstar.argtypes = [C.c_double] * 7
        _lib.orc_pvrs_pstar.restype = C.c_double
        _lib.orc_exact_riemann_star.argtypes = [C.c_double] * 7 + [_dp]
        _lib.orc_exact_riemann_sample.argtypes = [C.c_double] * 7 + [C.c_int, _dp, _dp, _dp, _dp]
        _lib.orc_num_threads.restype = C.c_int
        _lib.orc_diffusion.argtypes = [P, C.c_double, C.c_double, _dp, _dp]
        R = C.POINTER(OrcReact)
        _lib.orc_react_zone.argtypes = [R, C.c_int, C.c_double, C.c_double, _dp, _dp, _dp]
        _lib.orc_react_zone.restype = None
        _lib.orc_react_solve_zone.argtypes = [R, C.c_int, C.c_double, C.c_double, C.c_double, _dp, _dp]
        _lib.orc_react_R.argtypes = [P, R, _dp, _dp]
        _lib.orc_sdc_update_react.argtypes = [P, R, _dp, _dp, C.c_double, _dp, _dp, _dp, C.c_int, C.POINTER(_dp),
                                              C.POINTER(_dp), _dp, _dp, C.POINTER(C.c_int)]
    return _lib


def make_params(cfg: dict) -> OrcParams:
    """cfg: the plain dict produced by paper_1910_12578_b200.workloads (keys = field names)."""
    p = OrcParams()
    for k in ("nx", "ny", "nz", "ng", "nbx", "nby", "nbz", "nspec"):
        setattr(p, k, int(cfg[k]))
    for k in ("dx", "dy", "dz", "gamma", "small_dens", "small_pres"):
        setattr(p, k, float(cfg[k]))
    for d in range(3):
        p.grav[d] = float(cfg["grav"][d])
        p.bc_lo[d] = int(cfg["bc_lo"][d])
        p.bc_hi[d] = int(cfg["bc_hi"][d])
    return p


def _ptr(a):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


def u_shape(cfg):
    ng = cfg["ng"]
    return (cfg["nbx"] * cfg["nby"] * cfg["nbz"], 5 + cfg["nspec"],
            cfg["nz"] + 2 * ng, cfg["ny"] + 2 * ng, cfg["nx"] + 2 * ng)


def a_shape(cfg):
    return (cfg["nbx"] * cfg["nby"] * cfg["nbz"], 5 + cfg["nspec"], cfg["nz"], cfg["ny"], cfg["nx"])


def fill_ghosts(cfg, U):
    assert U.shape == u_shape(cfg)
    _chk(lib().orc_fill_ghosts(C.byref(make_params(cfg)), _ptr(U)), "fill_ghosts")
    return U


def advance_A(cfg, U, A=None):
    assert U.shape == u_shape(cfg)
    if A is None:
        A = np.empty(a_shape(cfg), dtype=np.float64)
    _chk(lib().orc_advance_A(C.byref(make_params(cfg)), _ptr(U), _ptr(A)), "advance_A")
    return A


def advance_A_flat(cfg, U, A=None):
    """<A(U)> with CW84 shock flattening (readings F1-F4); the whole ghost shell of U must be filled."""
    assert U.shape == u_shape(cfg)
    if A is None:
        A = np.empty(a_shape(cfg), dtype=np.float64)
    _chk(lib().orc_advance_A_flat(C.byref(make_params(cfg)), _ptr(U), _ptr(A)), "advance_A_flat")
    return A


def advance_A4(cfg, U, A=None):
    """Fourth-order finite-volume <A(U)> (oracle/orc_fourth.c, readings G1-G9); the whole ghost shell must be filled."""
    assert U.shape == u_shape(cfg)
    if A is None:
        A = np.empty(a_shape(cfg), dtype=np.float64)
    _chk(lib().orc_advance_A4(C.byref(make_params(cfg)), _ptr(U), _ptr(A)), "advance_A4")
    return A


def advance_ctu(cfg, U, dt, A=None):
    """A_ctu(U, dt) = -div F^{n+1/2} + S of the unsplit CTU PPM scheme (oracle/orc_ctu.c, readings C1-C9);
    U^{n+1} = U^n + dt A_ctu.  The whole ghost shell must be filled."""
    assert U.shape == u_shape(cfg)
    if A is None:
        A = np.empty(a_shape(cfg), dtype=np.float64)
    _chk(lib().orc_advance_ctu(C.byref(make_params(cfg)), _ptr(U), float(dt), _ptr(A)), "advance_ctu")
    return A


def ctu_step(cfg, U, dt):
    """One CTU step from library calls of the oracle: ghost fill, A_ctu, U + dt A_ctu.  Returns the new ghosted state."""
    U0 = fill_ghosts(cfg, U.copy())
    A = advance_ctu(cfg, U0, dt)
    Un = U0.copy()
    sdc_update(cfg, Un, U0, dt, A, A, [A], [dt])          # U + dt (A - A) + dt A
    return Un


def ppm4_line(q):
    """Limited fourth-order parabola edges (qm, qp) of one line of cell averages; valid for zones 2..n-3."""
    q = np.ascontiguousarray(q, dtype=np.float64)
    qm, qp = np.full_like(q, np.nan), np.full_like(q, np.nan)
    lib().orc_ppm4_line(len(q), _ptr(q), _ptr(qm), _ptr(qp))
    return qm, qp


def flatten_line(p, u, small_pres=1e-200):
    """chi^d of one line (F1-F2); valid for zones 3..n-4, 1 elsewhere."""
    p = np.ascontiguousarray(p, dtype=np.float64)
    u = np.ascontiguousarray(u, dtype=np.float64)
    chi = np.ones_like(p)
    lib().orc_flatten_line(len(p), _ptr(p), _ptr(u), float(small_pres), _ptr(chi))
    return chi


def sdc_update(cfg, U_next, U_m, dt_m, A_new_m, A_old_m, A_quad, w_quad):
    n = len(A_quad)
    arr = (_dp * max(n, 1))(*[_ptr(a) for a in A_quad])
    w = np.ascontiguousarray(np.asarray(w_quad, dtype=np.float64))
    _chk(lib().orc_sdc_update(C.byref(make_params(cfg)), _ptr(U_next), _ptr(U_m), float(dt_m),
                              _ptr(A_new_m), _ptr(A_old_m), n, arr, _ptr(w) if n else None),
         "sdc_update")
    return U_next


def cfl_dt(cfg, U, cfl):
    out = C.c_double(0.0)
    _chk(lib().orc_cfl_dt(C.byref(make_params(cfg)), _ptr(U), float(cfl), C.byref(out)), "cfl_dt")
    return out.value


def cons_to_prim(gamma, small_pres, Uz):
    Uz = np.ascontiguousarray(Uz, dtype=np.float64)
    Wz = np.empty_like(Uz)
    lib().orc_cons_to_prim(len(Uz), gamma, small_pres, _ptr(Uz), _ptr(Wz))
    return Wz


def ppm_line(q):
    """Returns (qm, qp); valid for zones 2..n-3, NaN elsewhere."""
    q = np.ascontiguousarray(q, dtype=np.float64)
    qm = np.full_like(q, np.nan)
    qp = np.full_like(q, np.nan)
    lib().orc_ppm_line(len(q), _ptr(q), _ptr(qm), _ptr(qp))
    return qm, qp


def hllc(d, gamma, WL, WR):
    WL = np.ascontiguousarray(WL, dtype=np.float64)
    WR = np.ascontiguousarray(WR, dtype=np.float64)
    F = np.empty_like(WL)
    lib().orc_hllc(len(WL), d, gamma, _ptr(WL), _ptr(WR), _ptr(F))
    return F


def wave_speeds(g, rL, uL, pL, rR, uR, pR, ps):
    """(S_L, S_R) of the HLLC wave-speed estimate for a given star-pressure estimate ps."""
    SL, SR = C.c_double(0.0), C.c_double(0.0)
    lib().orc_wave_speeds(g, rL, uL, pL, rR, uR, pR, ps, C.byref(SL), C.byref(SR))
    return SL.value, SR.value


def pvrs_pstar(g, rL, uL, pL, rR, uR, pR):
    return lib().orc_pvrs_pstar(g, rL, uL, pL, rR, uR, pR)


def exact_riemann_star(g, rL, uL, pL, rR, uR, pR):
    out = np.zeros(5)
    lib().orc_exact_riemann_star(g, rL, uL, pL, rR, uR, pR, _ptr(out))
    return out


def exact_riemann_sample(g, rL, uL, pL, rR, uR, pR, xi):
    xi = np.ascontiguousarray(xi, dtype=np.float64).ravel()
    rho, u, p = np.empty_like(xi), np.empty_like(xi), np.empty_like(xi)
    lib().orc_exact_riemann_sample(g, rL, uL, pL, rR, uR, pR, len(xi), _ptr(xi), _ptr(rho), _ptr(u), _ptr(p))
    return rho, u, p


def num_threads():
    return lib().orc_num_threads()


# ---- harness-level SDC driver (SURVEY 8(c) S5 "Driver") ------------------------
def sdc_step_2nd(cfg, U, dt):
    """One 2-node, 2-iteration SDC step (trapezoid) with R = 0, built only from
    oracle calls: ghost fill, A, node update.  U: ghosted state with interior valid; returns new U."""
    U0 = fill_ghosts(cfg, U.copy())
    A0 = advance_A(cfg, U0)
    w = [0.5 * dt, 0.5 * dt]
    # iteration 1: all nodes carry A(U^n)
    U1 = U0.copy()
    sdc_update(cfg, U1, U0, dt, A0, A0, [A0, A0], w)
    fill_ghosts(cfg, U1)
    A1 = advance_A(cfg, U1)
    # iteration 2: node 0 unchanged => A-difference term is zero; integral uses iteration-1 values
    U2 = U0.copy()
    sdc_update(cfg, U2, U0, dt, A0, A0, [A0, A1], w)
    return U2


def lobatto_nodes_weights(M):
    """Gauss-Lobatto nodes c_m on [0, 1] (M = 2: trapezoid, M = 3: Simpson) and the
    node-to-node weights w[m][j] = integral over [c_m, c_{m+1}] of the Lagrange polynomial l_j
    (SURVEY 8(c) Q17), here by integrating the interpolating polynomials numerically exactly."""
    if M == 2:
        c = np.array([0.0, 1.0])
    elif M == 3:
        c = np.array([0.0, 0.5, 1.0])
    else:
        raise ValueError("M must be 2 or 3")
    w = np.zeros((M - 1, M))
    for j in range(M):
        y = np.zeros(M); y[j] = 1.0
        P = np.polyint(np.polyfit(c, y, M - 1))
        for m in range(M - 1):
            w[m, j] = np.polyval(P, c[m + 1]) - np.polyval(P, c[m])
    return c, w


def sdc_step_nodes(cfg, U, dt, M=3, K=4, A_fn=None):
    """One SDC step with M Gauss-Lobatto nodes and K iterations, R = 0 (Eq. (2)):
      U^{m+1,(k+1)} = U^{m,(k+1)} + dt_m (A^{m,(k+1)} - A^{m,(k)}) + sum_j w_{m,j} A^{j,(k)},
    every node starting from U^n.  Built only from oracle calls; A_fn(U_ghosted) -> interior A replaces
    <A(U)> in the pins of the time integrator alone.  Returns the new ghosted state (ghosts stale)."""
    c, wt = lobatto_nodes_weights(M)
    A_of = A_fn if A_fn is not None else (lambda V: advance_A(cfg, V))
    U0 = fill_ghosts(cfg, U.copy())
    A0 = A_of(U0)
    U_old, A_old = [U0] * M, [A0] * M
    for k in range(K):
        U_new, A_new = [U0], [A0]
        for m in range(M - 1):
            dtm = (c[m + 1] - c[m]) * dt
            Un = U_new[m].copy()
            sdc_update(cfg, Un, U_new[m], dtm, A_new[m], A_old[m], A_old, list(wt[m] * dt))
            fill_ghosts(cfg, Un)
            U_new.append(Un)
            last = (k == K - 1) and (m == M - 2)
            A_new.append(None if last else A_of(Un))
        U_old, A_old = U_new, A_new
    return U_old[M - 1]


# ---- reactions: Eq. (2) with R != 0 (oracle/orc_react.c) -------------------------
def make_react(react: dict) -> OrcReact:
    """react: dict(cv, T0, nu, rate=[...], q=[...], max_iter, tol) (paper_1910_12578_b200.workloads.react_params)."""
    r = OrcReact()
    r.cv, r.T0, r.nu = float(react["cv"]), float(react["T0"]), float(react["nu"])
    for k, v in enumerate(react["rate"]):
        r.rate[k] = float(v)
    for k, v in enumerate(react["q"]):
        r.q[k] = float(v)
    r.max_iter, r.tol = int(react["max_iter"]), float(react["tol"])
    return r


def react_zone(react, rho, ke, y, jac=False):
    """R (and dR/dy) of one zone; y = (rho X_0 .., rho E)."""
    y = np.ascontiguousarray(y, dtype=np.float64)
    n = len(y)
    R = np.empty(n)
    J = np.empty((n, n)) if jac else None
    lib().orc_react_zone(C.byref(make_react(react)), n - 1, float(rho), float(ke), _ptr(y), _ptr(R),
                         _ptr(J) if jac else None)
    return (R, J) if jac else R


def react_solve_zone(react, rho, ke, dt, c):
    c = np.ascontiguousarray(c, dtype=np.float64)
    y = np.empty_like(c)
    it = lib().orc_react_solve_zone(C.byref(make_react(react)), len(c) - 1, float(rho), float(ke), float(dt), _ptr(c), _ptr(y))
    return y, it


def react_R(cfg, react, U, R=None):
    if R is None:
        R = np.empty(a_shape(cfg), dtype=np.float64)
    _chk(lib().orc_react_R(C.byref(make_params(cfg)), C.byref(make_react(react)), _ptr(U), _ptr(R)), "react_R")
    return R


def sdc_update_react(cfg, react, U_next, U_m, dt_m, A_new_m, A_old_m, R_old_next, A_quad, R_quad, w_quad, R_new=None,
                     iters=None):
    n = len(A_quad)
    assert n == len(R_quad) == len(w_quad)
    aq = (_dp * max(n, 1))(*[_ptr(a) for a in A_quad])
    rq = (_dp * max(n, 1))(*[_ptr(a) for a in R_quad])
    w = np.ascontiguousarray(np.asarray(w_quad, dtype=np.float64))
    if R_new is None:
        R_new = np.empty(a_shape(cfg), dtype=np.float64)
    ip = iters.ctypes.data_as(C.POINTER(C.c_int)) if iters is not None else None
    _chk(lib().orc_sdc_update_react(C.byref(make_params(cfg)), C.byref(make_react(react)), _ptr(U_next), _ptr(U_m),
                                    float(dt_m), _ptr(A_new_m), _ptr(A_old_m), _ptr(R_old_next), n, aq, rq,
                                    _ptr(w) if n else None, _ptr(R_new), ip), "sdc_update_react")
    return U_next, R_new


def sdc_step_nodes_react(cfg, react, U, dt, M=3, K=4, A_fn=None):
    """One SDC step of Eq. (2) with R != 0: M Gauss-Lobatto nodes, K iterations, every node
    starting from U^n; the node update is implicit in R (oracle sdc_update_react), A is explicit."""
    c, wt = lobatto_nodes_weights(M)
    A_of = A_fn if A_fn is not None else (lambda V: advance_A(cfg, V))
    U0 = fill_ghosts(cfg, U.copy())
    A0, R0 = A_of(U0), react_R(cfg, react, U0)
    A_old, R_old = [A0] * M, [R0] * M
    U_new = [U0]
    for k in range(K):
        U_new, A_new, R_new = [U0], [A0], [R0]
        for m in range(M - 1):
            dtm = (c[m + 1] - c[m]) * dt
            Un = U_new[m].copy()
            _, Rn = sdc_update_react(cfg, react, Un, U_new[m], dtm, A_new[m], A_old[m], R_old[m + 1], A_old, R_old,
                                     list(wt[m] * dt))
            fill_ghosts(cfg, Un)
            U_new.append(Un)
            R_new.append(Rn)
            last = (k == K - 1) and (m == M - 2)
            A_new.append(None if last else A_of(Un))
        A_old, R_old = A_new, R_new
    return U_new[M - 1]


# ---- explicit thermal diffusion as an extra term of A (oracle/orc_diffuse.c) --------
def diffusion(cfg, kth, cv, U):
    """D[b][k][j][i] = k_th lap T on interior zones (ghosts of U filled)."""
    sh = a_shape(cfg)
    D = np.empty((sh[0],) + sh[2:], dtype=np.float64)
    _chk(lib().orc_diffusion(C.byref(make_params(cfg)), float(kth), float(cv), _ptr(U), _ptr(D)), "diffusion")
    return D


def advance_A_diffuse(cfg, kth, cv, U):
    """<A(U)> with the diffusion term added to the energy component."""
    A = advance_A(cfg, U)
    A[:, 4] += diffusion(cfg, kth, cv, U)
    return A
