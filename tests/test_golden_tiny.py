"""tests/golden/oracle_tiny_case.txt (written by tests/golden/make_golden.py from the oracle only):
the oracle must still reproduce it bit for bit (its arithmetic is frozen), the CUDA path to <= 1e-12."""
import importlib.util
import os

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))
spec = importlib.util.spec_from_file_location("make_golden", os.path.join(HERE, "golden", "make_golden.py"))
mg = importlib.util.module_from_spec(spec)
spec.loader.exec_module(mg)


def stored():
    v = np.array([float(x) for x in open(os.path.join(HERE, "golden", "oracle_tiny_case.txt")) if not x.startswith("#")])
    nA = 2 * 7 * 4 * 5 * 6
    return v[0], v[1:1 + nA].reshape(2, 7, 4, 5, 6), v[1 + nA:].reshape(2, 7, 4, 5, 6)


def test_oracle_reproduces_its_stored_values_bitwise():
    dt, A, Un = mg.compute()
    sdt, sA, sUn = stored()
    assert dt == sdt and np.array_equal(A, sA) and np.array_equal(Un, sUn)


@pytest.mark.gpu
def test_cuda_path_matches_the_stored_values():
    import torch
    from paper_1910_12578_b200 import Context, workloads as wl
    cfg = mg.CFG
    sdt, sA, sUn = stored()
    ctx = Context(cfg)
    U = torch.from_numpy(wl.random_state(cfg, mg.SEED)).to("cuda:0")
    ctx.fill_ghosts(U)
    dt = ctx.cfl_dt(U, 0.5)
    assert abs(dt - sdt) <= 1e-14 * sdt
    A = torch.empty(wl.a_shape(cfg), dtype=torch.float64, device="cuda:0")
    ctx.advance_A(U, A)
    Aold = torch.from_numpy(0.5 * sA).to("cuda:0")          # the stored case uses A_old = A/2 (of the ORACLE's A)
    As = torch.from_numpy(sA).to("cuda:0")
    Un = U.clone()
    ctx.sdc_update(Un, U, sdt, As, Aold, [Aold, As], [0.25 * sdt, 0.75 * sdt])
    ax = (0, 2, 3, 4)
    eA = (np.abs(A.cpu().numpy() - sA).max(axis=ax) / np.abs(sA).max(axis=ax)).max()
    eU = (np.abs(Un.cpu().numpy()[:, :, 4:-4, 4:-4, 4:-4] - sUn).max(axis=ax) / np.abs(sUn).max(axis=ax)).max()
    assert eA <= 1e-12 and eU <= 1e-12, (eA, eU)
