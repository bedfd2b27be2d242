"""Parity of the optional CW84 shock flattening (include/cst.h cst_set_flattening) with the
oracle's orc_advance_A_flat, from bit-identical inputs, on states whose pressure jumps switch the limiter on."""
import numpy as np
import pytest
import torch

from oracle import orc
from paper_1910_12578_b200 import Context, CstError, workloads as wl
from test_oracle_pins import small_cfg
from test_oracle_flatten import shocked_state

pytestmark = pytest.mark.gpu
TOL = 1e-12
DEV = "cuda:0"


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def comp_err(gpu, ref):
    axes = (0, 2, 3, 4)
    num, den = np.abs(gpu - ref).max(axis=axes), np.abs(ref).max(axis=axes)
    return np.where(den > 0, num / np.where(den > 0, den, 1.0), num)


def flat_ctx(cfg):
    ctx = Context(cfg, workspace=None)
    plain = ctx.workspace_bytes()
    ctx.set_flattening(True)
    assert ctx.workspace_bytes() == plain + 8 * int(np.prod(wl.u_shape(cfg))) // wl.nvar(cfg)
    ctx.set_workspace(torch.empty(ctx.workspace_bytes(), dtype=torch.uint8, device=DEV))
    return ctx


@pytest.mark.parametrize("n,nb,ns,bc", [
    ((16, 16, 16), (1, 1, 1), 3, (0, 0, 0)),          # full tiles (the flattened path still takes the general kernels)
    ((20, 9, 12), (1, 1, 1), 2, (1, 2, 0)),           # ragged tiles, outflow / reflecting shells
    ((8, 6, 5), (2, 2, 1), 1, (2, 0, 1)),             # box lattice: coefficients of face-ghost zones look sideways
    ((32, 4, 4), (1, 1, 1), 0, (1, 0, 0)),            # no species
])
def test_flattened_advance_matches_oracle(n, nb, ns, bc):
    cfg = small_cfg(n=n, nb=nb, nspec=ns, gamma=1.4, bc=bc, grav=(0.0, 0.0, -0.1))
    U = orc.fill_ghosts(cfg, wl.from_global(cfg, wl.cons_from_prim(cfg, shocked_state(cfg, 81))))
    Ao, A_plain = orc.advance_A_flat(cfg, U), orc.advance_A(cfg, U)
    assert comp_err(Ao, A_plain).max() > 1e-2, "flattening must be active in this test"
    ctx = flat_ctx(cfg)
    Ud = dev(U)
    Ad = torch.full(wl.a_shape(cfg), float("nan"), dtype=torch.float64, device=DEV)
    ctx.advance_A(Ud, Ad)
    eA = comp_err(Ad.cpu().numpy(), Ao)
    assert eA.max() <= TOL, eA
    # fused node update
    dt = 0.3 * orc.cfl_dt(cfg, U, 0.5)
    Uno = np.full_like(U, 3.0)
    orc.sdc_update(cfg, Uno, U, dt, Ao, Ao, [Ao, Ao], [0.5 * dt, 0.5 * dt])
    Af = torch.empty_like(Ad)
    Uf = torch.full(wl.u_shape(cfg), 3.0, dtype=torch.float64, device=DEV)
    ctx.advance_A_update(Ud, Af, Uf, dt, Af, [Af, Af], [0.5 * dt, 0.5 * dt])
    assert comp_err(Af.cpu().numpy(), Ao).max() <= TOL
    assert comp_err(Uf.cpu().numpy(), Uno).max() <= TOL
    # switched off: the plain A again (workspace stays large enough)
    ctx.set_flattening(False)
    ctx.advance_A(Ud, Ad)
    assert comp_err(Ad.cpu().numpy(), A_plain).max() <= TOL
    ctx.destroy()


def test_smooth_flow_unchanged_and_workspace_is_checked():
    cfg = wl.make_config(2, n=(24, 16, 20))
    U = orc.fill_ghosts(cfg, wl.initial_state(cfg))
    Ud = dev(U)
    ctx = Context(cfg)                                   # workspace sized without flattening
    A0 = torch.empty(wl.a_shape(cfg), dtype=torch.float64, device=DEV)
    ctx.advance_A(Ud, A0)
    ctx.set_flattening(True)
    with pytest.raises(CstError):
        ctx.advance_A(Ud, A0)                            # the workspace is now too small: CST_ENOWORKSPACE
    ctx.destroy()
    ctx = flat_ctx(cfg)
    A1 = torch.empty_like(A0)
    ctx.advance_A(Ud, A1)
    # chi = 1 everywhere: the flattened (general) kernels give what the plain kernels give, to roundoff
    assert comp_err(A1.cpu().numpy(), orc.advance_A(cfg, U)).max() <= TOL
    ctx.destroy()
