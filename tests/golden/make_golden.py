"""Writes tests/golden/oracle_small.txt: H x and H^T y of a small seeded problem,
computed ONLY by the fp64 oracle (oracle/oat_oracle.c, discretisation OAT-DISC v1,
DESIGN.md §3; the passages it follows are cited in that file).  No value here
comes from the CUDA path.  The paper itself prints no value of g, p or alpha'
(SURVEY.md §8(c.3) P10), so there is no paper fixture to store.

    python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import oat_oracle as orc                      # noqa: E402
from paper_1304_2017_b200 import workloads as wl          # noqa: E402


def problem():
    return wl.small(n=10, q=2, nt=37, kband=8, seed=21)   # nt not a multiple of kband: ragged last band


def main():
    w = problem()
    x = w.phantom().astype(np.float64)
    y = w.data_noise(seed=22).astype(np.float64)
    hx = orc.project(w, x)
    hty = orc.backproject(w, y)
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_small.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/ only (OAT-DISC v1; PAPER.md Eq. 12-13, 22-23, 36-39)\n")
        f.write(f"# problem: workloads.small(n=10, q=2, nt=37, kband=8, seed=21); y = data_noise(seed=22)\n")
        f.write(f"# section Hx {hx.size}\n")
        for v in hx.ravel():
            f.write(f"{v:.17e}\n")
        f.write(f"# section HTy {hty.size}\n")
        for v in hty.ravel():
            f.write(f"{v:.17e}\n")
    print("wrote", out)


if __name__ == "__main__":
    main()
