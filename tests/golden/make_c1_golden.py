"""Writes tests/golden/c1_oracle_u_profile_step200.txt from the ORACLE ONLY (never from the CUDA path).

The paper prints no number for the stream-collide path (its printed values belong to workloads whose data
are not available — SURVEY.md §4), so there is no paper-cited fixture.  This file is a regression anchor for
the oracle itself: config 1 (BASELINE.json configs[0]) after 200 steps, the y-averaged u_x at x = 40
(16 cells behind the building) for every level z, and the global min/max of rho.

    python tests/golden/make_c1_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import Oracle  # noqa: E402
from paper_2607_04516_b200 import workloads as W  # noqa: E402


def compute():
    wl = W.config1()
    o = Oracle(wl.nx, wl.ny, wl.nz, wl.nu0, wl.Cs, wl.f_cor, wl.F, wl.faces)
    o.set_flags(wl.height)
    o.set_inlet_profile(*wl.inlet_profile)
    o.set_macros(*wl.init)
    o.step(200)
    rho, ux, uy, uz = o.get_macros()
    return ux[:, :, 40].mean(axis=1), rho.min(), rho.max()


if __name__ == "__main__":
    prof, rmin, rmax = compute()
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "c1_oracle_u_profile_step200.txt")
    with open(out, "w") as fh:
        fh.write("# written by tests/golden/make_c1_golden.py from oracle/ only; config 1, step 200\n")
        fh.write("# line 1: rho_min rho_max ; then one line per level z: y-mean of u_x at x=40\n")
        fh.write(f"{rmin:.15e} {rmax:.15e}\n")
        for v in prof:
            fh.write(f"{v:.15e}\n")
    print("wrote", out)
