"""Writes tests/golden/<config>_<mode>_oracle.npz: the CPU oracle's CONVERGED run of a full-size BASELINE.json config
(configs[2] cube 64^3, configs[3] finfet 128x64x64, configs[4] triangles 320x320) -- lattice temperature T_L of the
active cells, iteration count, max|dT| history and CG iterations per outer iteration -- from oracle/ ONLY (nothing
of the CUDA path is imported; paper_2607_03226_b200.workloads is the shared seeded input generator).

    python tests/golden/make_fullsize_golden.py cube plain
    python tests/golden/make_fullsize_golden.py cube synthetic
    python tests/golden/make_fullsize_golden.py finfet synthetic      # ~15 min on 8 cores, ~9 GB of host memory
    python tests/golden/make_fullsize_golden.py triangles plain

What the stored run is: source iteration PAPER.md:62 (Eq. 6) / synthetic iteration PAPER.md:75-100 (Eq. 8-12) with T_L
from Eq. 5, readings R1-R20 of DESIGN.md, from T_ref to the config's own tolerance (1e-9 K), i.e. exactly
`RefSolver(pr).solve(pr["tol"], pr["max_iter"], mode)`.  The north_star's bar for the GPU is: converged T within 1e-8 K
of this field with an identical iteration count (tests/test_fullsize_gpu.py::test_fullsize_converged_against_golden).
"""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle.ref import RefSolver  # noqa: E402
from paper_2607_03226_b200 import workloads as wl  # noqa: E402  (seeded input generators only)


def active_mask(pr):
    m = pr["mesh"]
    if pr["kind"] == "unstructured" or m["active"] is None:
        n = m["n_cells"] if pr["kind"] == "unstructured" else m["nx"] * m["ny"] * m["nz"]
        return np.ones(n, dtype=bool)
    return np.asarray(m["active"]).reshape(-1) != 0


def main():
    name, mode = sys.argv[1], sys.argv[2]
    pr = wl.CONFIGS[name]()
    t0 = time.time()
    r = RefSolver(pr)
    res = r.solve(pr["tol"], pr["max_iter"], mode)
    assert res["converged"], res
    dT, cg = r.get_history()
    T = r.get_T(0)[active_mask(pr)]
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), f"{name}_{mode}_oracle.npz")
    np.savez(path, T_active=T, iters=np.int64(res["iters"]), hist_dT=dT, hist_cg=cg, tol=np.float64(pr["tol"]),
             T_ref=np.float64(pr["T_ref"]), problem=np.array(pr["name"]), threads=np.int64(r.threads))
    print(path, res, f"{time.time() - t0:.1f} s on {r.threads} threads")


if __name__ == "__main__":
    main()
