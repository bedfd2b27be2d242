"""Parity of the explicit diffusion term (include/cst.h cst_set_diffusion) with the oracle
(oracle/orc_diffuse.c): A and the fused node update with the term switched on, from bit-identical inputs."""
import numpy as np
import pytest
import torch

from oracle import orc
from paper_1910_12578_b200 import Context, CstError, workloads as wl
from test_oracle_pins import small_cfg

pytestmark = pytest.mark.gpu
TOL = 1e-12
DEV = "cuda:0"
KTH, CV = 0.02, 1.5


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def comp_err(gpu, ref):
    axes = (0, 2, 3, 4)
    num, den = np.abs(gpu - ref).max(axis=axes), np.abs(ref).max(axis=axes)
    return np.where(den > 0, num / np.where(den > 0, den, 1.0), num)


@pytest.mark.parametrize("n,nb,ns,bc", [
    ((32, 16, 16), (1, 1, 1), 2, (0, 0, 0)),          # whole patches, full tiles
    ((40, 9, 37), (1, 1, 1), 0, (1, 2, 0)),           # ragged patches in x and y, two chunks in z
    ((7, 5, 4), (2, 2, 1), 1, (2, 0, 1)),             # boxes smaller than a patch
    ((33, 8, 33), (1, 2, 1), 0, (0, 1, 1)),           # one zone past a patch / chunk edge
])
def test_advance_with_diffusion_matches_oracle(n, nb, ns, bc):
    cfg = small_cfg(n=n, nb=nb, nspec=ns, gamma=5 / 3, bc=bc, grav=(0.0, 0.0, -0.2))
    U = orc.fill_ghosts(cfg, wl.random_state(cfg, 71))
    Ao = orc.advance_A_diffuse(cfg, KTH, CV, U)
    A_plain = orc.advance_A(cfg, U)
    assert np.abs(Ao[:, 4] - A_plain[:, 4]).max() > 1e-3 * np.abs(A_plain[:, 4]).max(), "the term must matter in this test"
    ctx = Context(cfg)
    with pytest.raises(CstError):
        ctx.set_diffusion(-1.0, CV)
    ctx.set_diffusion(KTH, CV)
    Ud = dev(U)
    Ad = torch.full(wl.a_shape(cfg), float("nan"), dtype=torch.float64, device=DEV)
    ctx.advance_A(Ud, Ad)
    eA = comp_err(Ad.cpu().numpy(), Ao)
    assert eA.max() <= TOL, eA
    # fused node update with the complete A
    dt = 0.3 * orc.cfl_dt(cfg, U, 0.5)
    rng = np.random.default_rng(5)
    Aold = Ao + 0.1 * rng.standard_normal(Ao.shape) * np.abs(Ao).max()
    Uno = np.full_like(U, 3.0)
    orc.sdc_update(cfg, Uno, U, dt, Ao, Aold, [Aold, Ao], [0.25 * dt, 0.75 * dt])
    Af = torch.empty_like(Ad)
    Uf = torch.full(wl.u_shape(cfg), 3.0, dtype=torch.float64, device=DEV)
    Aoldd = dev(Aold)
    ctx.advance_A_update(Ud, Af, Uf, dt, Aoldd, [Aoldd, Af], [0.25 * dt, 0.75 * dt])
    assert comp_err(Af.cpu().numpy(), Ao).max() <= TOL
    eU = comp_err(Uf.cpu().numpy(), Uno)
    assert eU.max() <= 10 * TOL, eU
    # switched off again: the plain A
    ctx.set_diffusion(0.0, CV)
    ctx.advance_A(Ud, Ad)
    assert comp_err(Ad.cpu().numpy(), A_plain).max() <= TOL
    ctx.destroy()
