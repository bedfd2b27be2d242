"""GPU parity on the edge cases round 1 never reached: floors that bind
(full and ragged tiles), strong shocks at faces (the shock branch of the HLLC wave speeds), uniformly supersonic
flow in +-x, +-y, +-z (the "pure upwind flux" select), the kernels' own reciprocal / square-root sequences in ulps,
and the blockIdx -> tile map of the advance kernels (brick walk) as a bijection.  Same gate as everywhere:
per component max|gpu - orc| / max|orc| <= 1e-12 from bit-identical inputs.
"""
import numpy as np
import pytest
import torch

from oracle import orc
from paper_1910_12578_b200 import Context, workloads as wl
from test_gpu_parity import check_one_call_set, comp_err, dev, DEV, TOL
from test_oracle_pins import small_cfg

pytestmark = pytest.mark.gpu


# ------------------------------------------------------------------ floors that bind ----------------------------
@pytest.mark.parametrize("n,nb", [((32, 16, 16), (1, 1, 1)),       # full 16^3 tiles: fast paths of both kernels
                                  ((20, 12, 9), (2, 1, 1)),        # ragged tiles: generic paths
                                  ((40, 24, 20), (1, 1, 1))])      # mixed
def test_active_floors(n, nb):
    cfg = small_cfg(n=n, nb=nb, nspec=3, gamma=5 / 3, bc=(0, 1, 2))
    cfg["small_dens"], cfg["small_pres"] = 0.85, 0.8
    U = wl.random_state(cfg, 301)                      # rho, p log-normal(0.3): about a third of the zones sit below
    Uo = orc.fill_ghosts(cfg, U.copy())
    # the floors must change the oracle's answer, else this test gates nothing
    free = dict(cfg, small_dens=1e-200, small_pres=1e-200)
    A_fl, A_fr = orc.advance_A(cfg, Uo), orc.advance_A(free, Uo)
    assert np.abs(A_fl - A_fr).max() > 1e-2 * np.abs(A_fr).max()
    res = check_one_call_set(cfg, U)
    print("active floors", n, nb, res)


def test_density_floor_only_and_tiny_default_floors():
    """interface density floor alone (zone-centre rho is never floored, Q11), then the default 1e-200 floors on a
    state with rho, p ~ 1e-3 .. 1e3: nothing binds and nothing under- or overflows."""
    cfg = small_cfg(n=(32, 16, 16), nspec=1, gamma=1.4)
    cfg["small_dens"] = 0.9
    check_one_call_set(cfg, wl.random_state(cfg, 302))
    cfg = small_cfg(n=(16, 16, 16), nspec=1, gamma=1.4)
    U = wl.random_state(cfg, 303, amp=1.0)
    check_one_call_set(cfg, U)


# ------------------------------------------------------------------ strong shocks ---------------------------------
def blast_state(cfg, axis, seed, pjump=1e4):
    """planar blast along `axis`: p = pjump on one side, 1 on the other, density jump 8, +1% seeded noise; the faces
    at the interface see p* >> p_K (shock branch of the wave-speed estimate) on the first call already."""
    Dx, Dy, Dz = wl.domain(cfg)
    rng = np.random.default_rng([7, seed])
    W = np.zeros((wl.nvar(cfg), Dz, Dy, Dx))
    coord = np.indices((Dz, Dy, Dx))[2 - axis]
    hi = coord < (Dx, Dy, Dz)[axis] // 2
    W[0] = np.where(hi, 8.0, 1.0) * (1 + 0.01 * rng.standard_normal((Dz, Dy, Dx)))
    W[4] = np.where(hi, pjump, 1.0) * (1 + 0.01 * rng.standard_normal((Dz, Dy, Dx)))
    W[1:4] = 0.05 * rng.standard_normal((3, Dz, Dy, Dx))
    if cfg["nspec"]:
        E = rng.standard_exponential((cfg["nspec"], Dz, Dy, Dx))
        W[5:] = E / E.sum(axis=0, keepdims=True)
    return wl.from_global(cfg, wl.cons_from_prim(cfg, W))


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_strong_shock_at_faces_initial_and_evolved(axis):
    cfg = small_cfg(n=(32, 16, 16), nspec=2, gamma=1.4, bc=(1, 1, 1))
    U = blast_state(cfg, axis, 310 + axis)
    # some face of the initial state must take the shock branch (p* > p_K) in the oracle's terms
    Uf = orc.fill_ghosts(cfg, U.copy())
    g = wl.to_global(cfg, Uf, ghosted=True)
    mid = (32, 16, 16)[axis] // 2
    zl = [slice(None)] * 3; zr = [slice(None)] * 3
    zl[2 - axis], zr[2 - axis] = mid - 1, mid
    WL = orc.cons_to_prim(1.4, 1e-200, g[(slice(None),) + tuple(zl)][:, 0, 0])
    WR = orc.cons_to_prim(1.4, 1e-200, g[(slice(None),) + tuple(zr)][:, 0, 0])
    ps = orc.pvrs_pstar(1.4, WL[0], WL[1 + axis], WL[4], WR[0], WR[1 + axis], WR[4])
    assert ps > 100 * WR[4]
    check_one_call_set(cfg, U)
    # evolved: 8 oracle steps produce a real shock / contact / rarefaction structure with Mach > 3 post-shock flow
    Uo = Uf
    for _ in range(8):
        Uo = orc.fill_ghosts(cfg, orc.sdc_step_2nd(cfg, Uo, orc.cfl_dt(cfg, Uo, 0.4)))
    assert np.isfinite(Uo).all()
    res = check_one_call_set(cfg, Uo)
    print("blast axis", axis, res)


# ------------------------------------------------------------------ supersonic everywhere ------------------------
@pytest.mark.parametrize("axis,sign", [(0, 1), (0, -1), (1, 1), (1, -1), (2, 1), (2, -1)])
def test_uniformly_supersonic_flow(axis, sign):
    """Mach ~ 3 bulk flow along one axis in either sense: every face normal to it is supersonic, so the HLLC flux
    must be the pure upwind flux F(W_L) resp. F(W_R) (pin P5) -- on the GPU this is the `pure` select."""
    cfg = small_cfg(n=(32, 16, 16), nspec=2, gamma=5 / 3)
    G = wl.to_global(cfg, wl.random_state(cfg, 320 + axis, amp=0.15), ghosted=True)
    rho = G[0].copy()
    mom = G[1 + axis] + sign * 4.0 * rho                 # c ~ 1.3: Mach ~ 3
    G[4] += 0.5 * (mom ** 2 - G[1 + axis] ** 2) / rho    # keep the pressure
    G[1 + axis] = mom
    res = check_one_call_set(cfg, wl.from_global(cfg, G))
    print("supersonic", axis, sign, res)


# ------------------------------------------------------------------ reciprocal / square root in ulps -------------
def test_rcp_sqrt_sequences_within_one_ulp():
    """hydro.cuh rcp_fast / sqrt_fast (MUFU seed + Newton) against IEEE 1/x and sqrt(x) over [1e-200, 1e200]."""
    ctx = Context(small_cfg(n=(8, 8, 8)), workspace=None)
    rng = np.random.default_rng(330)
    x = np.concatenate([10.0 ** rng.uniform(-200, 200, 400000), rng.uniform(0.5, 2.0, 200000),
                        np.array([1.0, 2.0, 4.0, 0.5, 3.0, 1e-200, 1e200, 1.5, np.nextafter(1.0, 2), np.nextafter(1.0, 0)])])
    xd = dev(x)
    r, s = torch.empty_like(xd), torch.empty_like(xd)
    ctx.debug_rcp_sqrt(xd, r, s)
    torch.cuda.synchronize()
    r, s = r.cpu().numpy(), s.cpu().numpy()
    rr, ss = 1.0 / x, np.sqrt(x)
    ulp_r = np.abs(r - rr) / np.spacing(rr)
    ulp_s = np.abs(s - ss) / np.spacing(ss)
    print("rcp_fast max ulp", ulp_r.max(), "sqrt_fast max ulp", ulp_s.max())
    assert ulp_r.max() <= 1.0 and ulp_s.max() <= 1.0


# ------------------------------------------------------------------ blockIdx -> tile is a bijection --------------
@pytest.mark.parametrize("n,nb", [((128, 128, 64), (1, 1, 1)),      # smallest box the 8 x 8 x 4 brick walk applies to
                                  ((256, 128, 128), (1, 1, 1)),
                                  ((512, 512, 512), (1, 1, 1)),      # configs[3]
                                  ((64, 64, 64), (16, 8, 4)),        # configs[4]
                                  ((40, 24, 20), (2, 1, 3))])        # ragged
def test_tile_map_is_a_bijection(n, nb):
    cfg = small_cfg(n=n, nb=nb)
    ctx = Context(cfg, workspace=None)
    nt = ctx.debug_tile_count()
    out = torch.full((nt, 8), -1, dtype=torch.int32, device=DEV)
    ctx.debug_tile_map(out)
    torch.cuda.synchronize()
    m = out.cpu().numpy().astype(np.int64)
    tx, ty, tz = (-(-v // 16) for v in n)
    assert nt == tx * ty * tz * nb[0] * nb[1] * nb[2]
    key = ((m[:, 0] * tz + m[:, 3] // 16) * ty + m[:, 2] // 16) * tx + m[:, 1] // 16
    assert np.array_equal(np.sort(key), np.arange(nt)), "tiles visited twice / never"
    assert np.array_equal(key, m[:, 7]), "tile id does not address the tile's own workspace slot"
    assert np.all(m[:, 4] == np.minimum(16, n[0] - m[:, 1])) and np.all(m[:, 5] == np.minimum(16, n[1] - m[:, 2])) \
        and np.all(m[:, 6] == np.minimum(16, n[2] - m[:, 3]))


def test_one_brick_walk_box_against_oracle():
    """one parity case on the smallest box that takes the brick walk (128 x 128 x 64), 1 species"""
    cfg = small_cfg(n=(128, 128, 64), nspec=1, gamma=5 / 3)
    ctx = Context(cfg)
    Ud = dev(wl.random_state(cfg, 340)); ctx.fill_ghosts(Ud)
    A = torch.full(wl.a_shape(cfg), float("nan"), dtype=torch.float64, device=DEV)
    ctx.advance_A(Ud, A)
    Ao = orc.advance_A(cfg, Ud.cpu().numpy())
    assert comp_err(A.cpu().numpy(), Ao).max() <= TOL
