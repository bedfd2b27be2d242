"""Parity of the reactive node update (Eq. (2) with R != 0; include/cst.h cst_react_R, cst_sdc_update_react; SURVEY
8(f) NEXT-3) with the oracle (oracle/orc_react.c), element by element from bit-identical inputs.  The oracle solves
each zone's Newton system by dense Gaussian elimination with pivoting, the kernel by the O(ns) elimination the
bidiagonal-plus-border structure allows; both iterate to the same fixed point, so the gate is the usual 1e-12."""
import numpy as np
import pytest
import torch

from oracle import orc
from paper_1910_12578_b200 import Context, CstError, sdc_step_nodes_react, workloads as wl
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


@pytest.mark.parametrize("n,nb,ns,nu,stiff,nquad", [
    ((9, 7, 5), (2, 1, 1), 1, 4.0, 1.0, 2),
    ((16, 6, 4), (1, 1, 2), 4, 6.0, 10.0, 3),
    ((8, 8, 8), (1, 1, 1), 13, 4.0, 1.0, 2),            # the paper's network size
    ((5, 4, 6), (1, 2, 1), 15, -2.0, 300.0, 0),         # maximum size, very stiff, no quadrature term
    ((12, 5, 4), (1, 1, 1), 13, 0.0, 1000.0, 4),        # linear (nu = 0), dt * rate up to 1e3
])
def test_react_R_and_node_update_match_oracle(n, nb, ns, nu, stiff, nquad):
    cfg = small_cfg(n=n, nb=nb, nspec=ns, gamma=5 / 3, bc=(0, 1, 2))
    react = wl.react_params(ns, nu=nu, stiff=stiff)
    rng = np.random.default_rng(11)
    U = orc.fill_ghosts(cfg, wl.random_state(cfg, 51))
    ctx = Context(cfg)
    with pytest.raises(CstError):
        ctx.react_R(dev(U), torch.empty(wl.a_shape(cfg), dtype=torch.float64, device=DEV))     # not set yet
    ctx.set_reactions(react)
    Ud = dev(U)
    Rd = torch.full(wl.a_shape(cfg), float("nan"), dtype=torch.float64, device=DEV)
    ctx.react_R(Ud, Rd)
    Ro = orc.react_R(cfg, react, U)
    assert comp_err(Rd.cpu().numpy(), Ro).max() <= TOL
    assert np.all(Rd.cpu().numpy()[:, :4] == 0.0)
    # one node update with every term of Eq. (2) present, sized as in a real SDC sweep: A terms a few per cent of the
    # local state, the weights sum to dt_m and the R arrays are close to one another, so that -dt R_old + sum w R_q
    # nearly cancels (as it does between consecutive iterations) and the explicit part c stays a physical state
    Ui = U[:, :, 4:-4, 4:-4, 4:-4]
    dt = 0.01
    A_new, A_old = (2.0 * np.abs(Ui) * rng.standard_normal(Ro.shape) for _ in range(2))        # dt * A ~ 2 % of U
    Aq = [2.0 * np.abs(Ui) * rng.standard_normal(Ro.shape) for _ in range(nquad)]
    Rq = [Ro * (1.0 + 0.01 * rng.standard_normal()) for _ in range(nquad)]
    w = [float(x) for x in dt * rng.dirichlet(np.ones(nquad))] if nquad else []
    R_old = Ro * (1.01 if nquad else 0.0)
    Uno = np.full_like(U, 3.0)
    iters = np.zeros(Ro[:, 0].shape, dtype=np.int32)
    _, Rno = orc.sdc_update_react(cfg, react, Uno, U, dt, A_new, A_old, R_old, Aq, Rq, w, iters=iters)
    assert iters.max() <= 12 and np.isfinite(Uno).all(), "the oracle itself struggles: bad test parameters"
    Und = torch.full(wl.u_shape(cfg), 3.0, dtype=torch.float64, device=DEV)
    Rnd = torch.full(wl.a_shape(cfg), float("nan"), dtype=torch.float64, device=DEV)
    ctx.sdc_update_react(Und, Ud, dt, dev(A_new), dev(A_old), dev(R_old), [dev(a) for a in Aq], [dev(a) for a in Rq], w, Rnd)
    Ung = Und.cpu().numpy()
    eU, eR = comp_err(Ung, Uno), comp_err(Rnd.cpu().numpy(), Rno)
    assert eU.max() <= TOL, eU
    assert eR.max() <= 100 * TOL, eR                      # R amplifies errors of y by dt-free rates (<= 1e3 here)
    mask = np.ones(Uno.shape, bool); mask[:, :, 4:-4, 4:-4, 4:-4] = False
    assert np.all(Ung[mask] == 3.0), "the update touched ghost zones"
    assert ctx.react_failures() == 0
    print("U_next", eU.max(), "R_new", eR.max(), "oracle Newton iterations <=", iters.max())
    ctx.destroy()


def test_unconverged_zones_are_counted_and_reactions_need_species():
    cfg = small_cfg(n=(6, 5, 4), nspec=3, gamma=5 / 3)
    react = dict(wl.react_params(3, nu=6.0, stiff=50.0), max_iter=1)
    U = dev(orc.fill_ghosts(cfg, wl.random_state(cfg, 52)))
    ctx = Context(cfg)
    ctx.set_reactions(react)
    Z = torch.zeros(wl.a_shape(cfg), dtype=torch.float64, device=DEV)
    Un, Rn = torch.empty_like(U), torch.empty_like(Z)
    ctx.sdc_update_react(Un, U, 0.05, Z, Z, Z, [], [], [], Rn)
    assert ctx.react_failures() == 6 * 5 * 4              # one Newton step never meets tol = 1e-13 here
    assert ctx.react_failures() == 0                      # the counter is reset by the read
    ctx.destroy()
    ctx0 = Context(small_cfg(n=(4, 4, 4), nspec=0))
    with pytest.raises(CstError):
        ctx0.set_reactions(react)
    ctx0.destroy()


@pytest.mark.parametrize("M,K", [(2, 2), (3, 4)])
def test_reactive_sdc_driver_matches_oracle(M, K):
    """A whole SDC step with advection AND reactions (every term of Eq. (2) live), GPU driver against the oracle's."""
    ns = 3
    cfg = small_cfg(n=(8, 6, 5), nb=(2, 1, 1), nspec=ns, gamma=5 / 3)
    react = wl.react_params(ns, nu=4.0, stiff=2.0)
    U0 = wl.random_state(cfg, 53, amp=0.1)
    dt = 0.5 * orc.cfl_dt(cfg, orc.fill_ghosts(cfg, U0.copy()), 0.5)
    Uo = orc.sdc_step_nodes_react(cfg, react, U0, dt, M=M, K=K)
    ctx = Context(cfg)
    ctx.set_reactions(react)
    Ud = dev(np.nan_to_num(U0, nan=0.0))
    sdc_step_nodes_react(ctx, Ud, dt, M=M, K=K)
    I = (slice(None), slice(None), slice(4, -4), slice(4, -4), slice(4, -4))
    e = comp_err(Ud.cpu().numpy()[I], Uo[I])
    assert e.max() <= 10 * TOL, e                          # 2(M-1)K chained calls, each within 1e-12
    assert ctx.react_failures() == 0
    ctx.destroy()
