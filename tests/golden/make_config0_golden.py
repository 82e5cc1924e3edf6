"""Writes tests/golden/config0_oracle.txt: the converged lattice temperature of BASELINE.json configs[0]
(gray 20x20 square, 16 directions, walls 301 K / 299 K thermalizing, top/bottom diffuse, tol 1e-10 K)
and the iteration count, from the CPU oracle ONLY (oracle/ref.py; nothing of the CUDA path is imported).

    python tests/golden/make_config0_golden.py

The oracle itself is pinned for this config by the dense global fixed point (P2, tests/test_oracle_pins.py);
the file lets the GPU tests and later rounds detect any drift of either side against a stored value.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle.ref import RefSolver  # noqa: E402
from paper_2607_03226_b200 import workloads as wl  # noqa: E402  (seeded input generators only)


def main():
    pr = wl.config_gray_square()
    r = RefSolver(pr)
    res = r.solve(pr["tol"], pr["max_iter"])
    assert res["converged"]
    T = r.get_T(0)
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config0_oracle.txt")
    with open(path, "w") as f:
        f.write("# BASELINE.json configs[0]; source iteration PAPER.md:62 (Eq. 6), T_L from Eq. 5 (PAPER.md:59);\n")
        f.write("# readings R2-R11 of DESIGN.md.  Written by tests/golden/make_config0_golden.py from oracle/ only.\n")
        f.write(f"# iterations {res['iters']}\n")
        f.write("# T_L [K], cell id = i + 20*j, one row of the grid (fixed j) per line\n")
        for j in range(20):
            f.write(" ".join(f"{v:.15f}" for v in T[20 * j:20 * j + 20]) + "\n")
    print(path, res)


if __name__ == "__main__":
    main()
