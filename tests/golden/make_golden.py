"""Writes tests/golden/oracle_tiny_case.txt: <A(U)>, the node update and dt of a tiny fixed case, computed by
the CPU ORACLE ONLY (this script imports nothing from the CUDA path except the seeded input generator, which holds
no arithmetic of the method).  The stored numbers freeze the oracle's arithmetic: a later change to oracle/orc.c that
moves them must name, in its commit message, the passage or DESIGN.md reading that justifies it.

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import orc                                   # noqa: E402
from paper_1910_12578_b200 import workloads as wl        # noqa: E402

CFG = dict(name="golden", index=99, nx=6, ny=5, nz=4, ng=4, nbx=2, nby=1, nbz=1, nspec=2,
           dx=1.0 / 12, dy=1.0 / 5, dz=1.0 / 4, gamma=5.0 / 3.0, grav=(0.0, 0.1, -0.3),
           bc_lo=(0, 1, 2), bc_hi=(0, 1, 2), small_dens=1e-200, small_pres=1e-200)
SEED = 7


def compute():
    U = orc.fill_ghosts(CFG, wl.random_state(CFG, SEED))
    dt = orc.cfl_dt(CFG, U, 0.5)
    A = orc.advance_A(CFG, U)
    Un = U.copy()
    orc.sdc_update(CFG, Un, U, dt, A, 0.5 * A, [0.5 * A, A], [0.25 * dt, 0.75 * dt])
    return dt, A, Un[:, :, 4:-4, 4:-4, 4:-4]


if __name__ == "__main__":
    dt, A, Un = compute()
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_tiny_case.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/ only; config and seed are in that script\n")
        f.write("# line 1: dt (CFL 0.5); then A (2 boxes x 7 comps x 4 x 5 x 6, C order), then U_next interior\n")
        f.write(repr(float(dt)) + "\n")
        for v in A.ravel():
            f.write(repr(float(v)) + "\n")
        for v in Un.ravel():
            f.write(repr(float(v)) + "\n")
    print("wrote", out, A.size + Un.size + 1, "values")
