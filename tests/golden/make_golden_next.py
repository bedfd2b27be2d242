"""Writes tests/golden/oracle_next_case.txt: the operators beyond S0-S6 (flattened A, diffusion term, fourth-order A,
CTU operator, R and the implicit node update) on a tiny fixed case, computed by the CPU ORACLE ONLY (the seeded input
generator is the only thing shared with the CUDA path).  The stored numbers freeze the arithmetic of oracle/orc.c (S2b),
orc_diffuse.c, orc_fourth.c, orc_ctu.c and orc_react.c: a later change that moves them must name, in its commit message,
the passage or DESIGN.md reading that justifies it.

    python tests/golden/make_golden_next.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import orc                                   # noqa: E402
from paper_1910_12578_b200 import workloads as wl        # noqa: E402

CFG = dict(name="golden_next", index=99, nx=5, ny=4, nz=4, ng=4, nbx=1, nby=1, nbz=1, nspec=2,
           dx=1.0 / 5, dy=1.0 / 4, dz=1.0 / 4, gamma=1.4, grav=(0.0, 0.1, -0.3),
           bc_lo=(0, 1, 2), bc_hi=(0, 1, 2), small_dens=1e-200, small_pres=1e-200)
SEED, KTH, CV, DT = 11, 0.02, 1.5, 2.0e-3
NAMES = ("A_flat", "D", "A4", "A_ctu", "R", "U_react", "R_new")


def compute():
    """-> (dict name -> array, U, U4); U has strong pressure contrasts so that the flattening coefficient is active, the
    fourth-order operator gets a milder state U4 (its cell-centre conversion must stay physical)"""
    rng = np.random.default_rng(SEED)
    W = np.zeros((7, 4, 4, 5))
    W[0] = np.exp(0.3 * rng.standard_normal(W[0].shape))
    W[1:4] = 0.5 * rng.standard_normal((3,) + W[0].shape)
    W[4] = np.exp(0.5 * rng.standard_normal(W[0].shape))
    W[5] = rng.random(W[0].shape)
    W[6] = 1.0 - W[5]
    U = orc.fill_ghosts(CFG, wl.from_global(CFG, wl.cons_from_prim(CFG, W)))
    react = wl.react_params(2, nu=3.0, stiff=5.0)
    R = orc.react_R(CFG, react, U)
    Z = np.zeros_like(R)
    Un = U.copy()
    _, Rn = orc.sdc_update_react(CFG, react, Un, U, DT, Z, Z, R, [Z], [R], [DT])
    U4 = orc.fill_ghosts(CFG, wl.random_state(CFG, SEED, amp=0.1))
    return {"A_flat": orc.advance_A_flat(CFG, U), "D": orc.diffusion(CFG, KTH, CV, U), "A4": orc.advance_A4(CFG, U4),
            "A_ctu": orc.advance_ctu(CFG, U, DT), "R": R, "U_react": Un[:, :, 4:-4, 4:-4, 4:-4].copy(), "R_new": Rn}, U, U4


if __name__ == "__main__":
    res, _, _ = compute()
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_next_case.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_golden_next.py from oracle/ only; config, seed and parameters are in that script\n")
        f.write("# blocks in the order " + ", ".join(NAMES) + "; each: a line '@name count', then the values in C order\n")
        for name in NAMES:
            v = res[name].ravel()
            f.write(f"@{name} {v.size}\n")
            for x in v:
                f.write(repr(float(x)) + "\n")
    print("wrote", out)
