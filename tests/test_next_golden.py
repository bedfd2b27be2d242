"""tests/golden/oracle_next_case.txt (written by tests/golden/make_golden_next.py from the oracle only): the oracle must
reproduce it bit for bit -- the arithmetic of the operators beyond S0-S6 is frozen -- and the CUDA path to <= 1e-12."""
import importlib.util
import os

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
spec = importlib.util.spec_from_file_location("make_golden_next", os.path.join(HERE, "golden", "make_golden_next.py"))
mg = importlib.util.module_from_spec(spec)
spec.loader.exec_module(mg)


def stored():
    out, name = {}, None
    for line in open(os.path.join(HERE, "golden", "oracle_next_case.txt")):
        if line.startswith("#"):
            continue
        if line.startswith("@"):
            name = line[1:].split()[0]
            out[name] = []
        else:
            out[name].append(float(line))
    return {k: np.array(v) for k, v in out.items()}


def test_oracle_reproduces_its_stored_values_bitwise():
    res, U, _ = mg.compute()
    st = stored()
    assert set(st) == set(mg.NAMES)
    for name in mg.NAMES:
        assert np.isfinite(st[name]).all() and np.array_equal(res[name].ravel(), st[name]), name
    assert np.abs(st["A_flat"] - mg.orc.advance_A(mg.CFG, U).ravel()).max() > 1e-3     # flattening is active


def rel(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


@pytest.mark.gpu
def test_cuda_path_matches_the_stored_values():
    import torch
    from paper_1910_12578_b200 import Context, workloads as wl
    cfg, st = mg.CFG, stored()
    _, U, U4 = mg.compute()
    DEV = "cuda:0"
    Ud = torch.from_numpy(U).to(DEV)
    ash = wl.a_shape(cfg)
    new = lambda: torch.empty(ash, dtype=torch.float64, device=DEV)

    def ctx_with(pre=None):
        c = Context(cfg, workspace=None)
        if pre:
            pre(c)
        c.set_workspace(torch.empty(c.workspace_bytes(), dtype=torch.uint8, device=DEV))
        return c
    A = new()
    c = ctx_with(lambda x: x.set_flattening(True))
    c.advance_A(Ud, A)
    assert rel(A.cpu().numpy().ravel(), st["A_flat"]) <= 1e-12
    c.destroy()
    c = ctx_with()
    A0 = new()
    c.advance_A(Ud, A0)
    c.set_diffusion(mg.KTH, mg.CV)
    c.advance_A(Ud, A)
    D = (A - A0)[:, 4].cpu().numpy().ravel()
    assert np.abs(D - st["D"]).max() <= 1e-12 * np.abs(A0[:, 4].cpu().numpy()).max()      # D is the difference of two A's
    c.set_diffusion(0.0, mg.CV)
    ws = torch.empty(c.ctu_workspace_bytes(), dtype=torch.uint8, device=DEV)
    c.advance_ctu(Ud, mg.DT, A, ws)
    assert rel(A.cpu().numpy().ravel(), st["A_ctu"]) <= 1e-12
    react = wl.react_params(2, nu=3.0, stiff=5.0)
    c.set_reactions(react)
    R, Rn, Z = new(), new(), torch.zeros(ash, dtype=torch.float64, device=DEV)
    c.react_R(Ud, R)
    assert rel(R.cpu().numpy().ravel(), st["R"]) <= 1e-12
    Rs = torch.from_numpy(st["R"].reshape(ash)).to(DEV)
    Un = Ud.clone()
    c.sdc_update_react(Un, Ud, mg.DT, Z, Z, Rs, [Z], [Rs], [mg.DT], Rn)
    assert rel(Un.cpu().numpy()[:, :, 4:-4, 4:-4, 4:-4].ravel(), st["U_react"]) <= 1e-12
    assert rel(Rn.cpu().numpy().ravel(), st["R_new"]) <= 1e-10
    c.destroy()
    c = ctx_with(lambda x: x.set_order(4))
    c.advance_A(torch.from_numpy(U4).to(DEV), A)
    assert rel(A.cpu().numpy().ravel(), st["A4"]) <= 1e-12
    c.destroy()
