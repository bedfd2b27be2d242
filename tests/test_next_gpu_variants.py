"""The kernel variants of the species half of <A(U)> (include/cst.h cst_set_variant, cst_tune_advance): every variant
against the oracle at the usual gate, bitwise against variant 0, for every fused-update arity, and the tuner."""
import numpy as np
import pytest
import torch

from oracle import orc
from paper_1910_12578_b200 import Context, CstError, workloads as wl
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


@pytest.mark.parametrize("n,nb,ns,bc", [
    ((32, 16, 16), (1, 1, 1), 13, (0, 0, 0)),         # two tiles in x, the three-CTAs-per-tile split (5 / 4 / 4 species)
    ((16, 32, 32), (2, 1, 1), 4, (1, 2, 0)),          # boxes, outflow / reflecting shells, gravity
    ((16, 16, 16), (1, 1, 1), 1, (0, 0, 0)),          # one species: one CTA per tile, a single pass
    ((16, 16, 48), (1, 1, 1), 2, (0, 0, 0)),          # split 2, one species per CTA
])
def test_variants_match_oracle_and_each_other(n, nb, ns, bc):
    cfg = small_cfg(n=n, nb=nb, nspec=ns, gamma=5 / 3, bc=bc, grav=(0.0, 0.1, -0.2))
    U = orc.fill_ghosts(cfg, wl.random_state(cfg, 111))
    Ao = orc.advance_A(cfg, U)
    dt = 0.4 * orc.cfl_dt(cfg, U, 0.5)
    rng = np.random.default_rng(7)
    P = [Ao + 0.1 * rng.standard_normal(Ao.shape) * np.abs(Ao).max() for _ in range(3)]
    Ud, Pd = dev(U), [dev(p) for p in P]
    ctx = Context(cfg)
    with pytest.raises(CstError):
        ctx.set_variant(4)
    # update arities: plain A (NR = -1), forward Euler (0 external arrays), 1, 2, 3 external arrays
    cases = {"plain": None, "nr0": ("self", []), "nr1": (0, [0]), "nr2": (0, [0, 1]), "nr3": (0, [1, 2])}
    ref = {}
    for v in (0, 1, 2, 3):
        ctx.set_variant(v)
        assert ctx.get_variant() == v
        for name, case in cases.items():
            A = torch.full(wl.a_shape(cfg), float("nan"), dtype=torch.float64, device=DEV)
            Un = torch.full(wl.u_shape(cfg), 3.0, dtype=torch.float64, device=DEV)
            if case is None:
                ctx.advance_A(Ud, A)
            else:
                old, quad = case
                Aold = A if old == "self" else Pd[old]
                Aq = [Pd[q] for q in quad] + [A]
                w = [0.3 * dt / len(Aq)] * len(Aq)
                ctx.advance_A_update(Ud, A, Un, dt, Aold, Aq, w)
                Uno = np.full_like(U, 3.0)
                orc.sdc_update(cfg, Uno, U, dt, Ao, Ao if old == "self" else P[old], [P[q] for q in quad] + [Ao], w)
                assert comp_err(Un.cpu().numpy(), Uno).max() <= 10 * TOL, (v, name)
            Ah = A.cpu().numpy()
            assert comp_err(Ah, Ao).max() <= TOL, (v, name)
            if v == 0:
                ref[name] = (Ah, Un.cpu().numpy())
            else:
                assert np.array_equal(Ah, ref[name][0]) and np.array_equal(Un.cpu().numpy(), ref[name][1]), (v, name)
    # the number of CTAs that share a tile does not change a bit either
    ctx.set_variant(2)
    for split in (1, 2, 4, 8):
        ctx.set_species_split(split)
        A = torch.full(wl.a_shape(cfg), float("nan"), dtype=torch.float64, device=DEV)
        ctx.advance_A(Ud, A)
        assert np.array_equal(A.cpu().numpy(), ref["plain"][0]), split
    ctx.destroy()


def test_tuner_keeps_a_valid_variant_and_valid_outputs():
    cfg = small_cfg(n=(32, 16, 16), nspec=3, gamma=5 / 3)
    U = orc.fill_ghosts(cfg, wl.random_state(cfg, 112))
    Ao = orc.advance_A(cfg, U)
    ctx = Context(cfg)
    Ud = dev(U)
    A = torch.full(wl.a_shape(cfg), float("nan"), dtype=torch.float64, device=DEV)
    Un = torch.full(wl.u_shape(cfg), 3.0, dtype=torch.float64, device=DEV)
    v, ms = ctx.tune_advance(Ud, A, Un, 1e-3, A, [A, A], [5e-4, 5e-4], repeats=1)
    assert v in (0, 1, 2, 3) and len(ms) == 6 and all(m > 0 for m in ms) and ms[v] == min(ms[:4])
    assert ctx.get_species_split() in (0, 2, 4)
    if ctx.get_species_split():
        assert ms[4 + (ctx.get_species_split() == 4)] == min(ms)
    assert comp_err(A.cpu().numpy(), Ao).max() <= TOL
    Uno = np.full_like(U, 3.0)
    orc.sdc_update(cfg, Uno, U, 1e-3, Ao, Ao, [Ao, Ao], [5e-4, 5e-4])
    assert comp_err(Un.cpu().numpy(), Uno).max() <= TOL
    ctx.destroy()


@pytest.mark.parametrize("n,nb,ns", [
    ((32, 16, 16), (1, 1, 1), 3),          # full tiles: the CFL max is gathered inside the hydro kernel's z sweep
    ((16, 16, 32), (2, 1, 1), 0),          # boxes, no species
    ((20, 12, 9), (1, 1, 1), 2),           # ragged tiles: the two calls run back to back
])
def test_fused_cfl_call_matches_the_separate_calls_and_the_oracle(n, nb, ns):
    cfg = small_cfg(n=n, nb=nb, nspec=ns, gamma=5 / 3, bc=(0, 1, 2), grav=(0.0, 0.0, -0.2))
    U = orc.fill_ghosts(cfg, wl.random_state(cfg, 113))
    dt_o = orc.cfl_dt(cfg, U, 0.4)
    ctx = Context(cfg)
    Ud = dev(U)
    dt = 1e-3
    A0 = torch.full(wl.a_shape(cfg), float("nan"), dtype=torch.float64, device=DEV)
    Un0 = torch.full(wl.u_shape(cfg), 3.0, dtype=torch.float64, device=DEV)
    ctx.advance_A_update(Ud, A0, Un0, dt, A0, [A0, A0], [0.5 * dt, 0.5 * dt])
    A1, Un1 = torch.full_like(A0, float("nan")), torch.full_like(Un0, 3.0)
    dtd = torch.zeros(1, dtype=torch.float64, device=DEV)
    for _ in range(2):                                       # twice: the reduction cell is reset by every call
        ctx.advance_A_update_cfl(Ud, A1, Un1, dt, A1, [A1, A1], [0.5 * dt, 0.5 * dt], 0.4, dtd)
    assert np.array_equal(A1.cpu().numpy(), A0.cpu().numpy()) and np.array_equal(Un1.cpu().numpy(), Un0.cpu().numpy())
    assert abs(float(dtd.cpu()[0]) - dt_o) <= 1e-14 * dt_o
    assert abs(ctx.cfl_dt(Ud, 0.4) - dt_o) <= 1e-14 * dt_o
    ctx.destroy()


# ------------------------------------------------------------ the launch configurations bench.py may time, at full size ----
def checksums(t):
    """two order-independent integer checksums of the BIT PATTERNS of a float64 tensor (wrap-around sums)"""
    a = b = 0
    for box in t:                              # component by component: the shifted copy stays small
        for comp in box:
            v = comp.reshape(-1).view(torch.int64)
            a += int(v.sum())
            b += int((v >> 11).sum())
    return a % (1 << 64), b % (1 << 64)


def variants_agree_bitwise(cfg):
    """Every species-kernel variant, every number of CTAs per tile the tuner tries, and the fused-CFL call produce the
    same bits as variant 0 with separate calls -- whose every zone tests/test_gpu_fullsize.py compares with the oracle."""
    from test_gpu_fullsize import device_state
    ctx = Context(cfg)
    U = device_state(cfg)
    ctx.fill_ghosts(U)
    dt = ctx.cfl_dt(U, 0.5)
    ash = wl.a_shape(cfg)
    A0 = torch.empty(ash, dtype=torch.float64, device=DEV)
    ctx.advance_A(U, A0)
    A1 = A0 * 0.9
    A = torch.empty(ash, dtype=torch.float64, device=DEV)
    Un = torch.empty(wl.u_shape(cfg), dtype=torch.float64, device=DEV)
    w = [0.5 * dt, 0.5 * dt]
    ref = None
    for variant, split, fused in [(0, 0, False), (1, 0, False), (2, 0, False), (3, 0, False), (2, 2, False), (2, 4, False),
                                  (0, 0, True), (2, 0, True)]:
        ctx.set_variant(variant)
        ctx.set_species_split(split)
        A.fill_(float("nan"))
        Un.fill_(3.0)
        if fused:
            dtd = torch.zeros(1, dtype=torch.float64, device=DEV)
            ctx.advance_A_update_cfl(U, A, Un, dt, A0, [A0, A1], w, 0.5, dtd)
            assert float(dtd.cpu()[0]) == dt or abs(float(dtd.cpu()[0]) - dt) <= 1e-14 * dt
        else:
            ctx.advance_A_update(U, A, Un, dt, A0, [A0, A1], w)
        torch.cuda.synchronize()
        got = (checksums(A), checksums(Un))
        if ref is None:
            assert torch.isfinite(A).all()
            ref = got
        assert got == ref, (variant, split, fused)
    ctx.destroy()


def test_variants_agree_bitwise_at_full_size_configs3():
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 112e9:
        pytest.skip(f"needs 112 GB of free device memory, has {free / 1e9:.0f}")
    variants_agree_bitwise(wl.make_config(3))


def test_variants_agree_bitwise_on_a_batch_of_boxes():
    variants_agree_bitwise(wl.make_config(4, nb=(4, 2, 1)))          # 8 of configs[4]'s boxes (64^3, reflecting z, gravity)
