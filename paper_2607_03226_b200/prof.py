"""In-kernel timers of the two cooperative/persistent kernels, from the instrumented copy of the library.

    python -m paper_2607_03226_b200.build -DBRICK_PROF -DMG_PROF      # -> libnanobte_prof.so (never loaded by the product)
    python -m paper_2607_03226_b200.prof sweep [--workload finfet|cube]
    python -m paper_2607_03226_b200.prof cg    [--workload finfet|cube]

`sweep`: sweep_brick_kernel (csrc/sweep_brick.cu, BRICK_PROF).  Per plane and CTA the clock64() cycles of the phases of a
plane (thread 0 of every CTA, summed over all tasks), and a timeline of the last sweep from %globaltimer: when each task took
its ticket, had its first plane ready and finished; printed as the number of resident / running tasks over time.
`cg`: cg_mg_kernel (csrc/cg_mg.cu, MG_PROF).  Per CG iteration the time of every part of the V-cycle, per solve the set-up
parts, measured by thread 0 of CTA 0 (waits for other CTAs show up where the exchange happens).

The numbers are for reading the kernels, not bench values: the probes cost a few percent.  DESIGN.md section 10 quotes them.
"""
from __future__ import annotations

import argparse
import ctypes as C
import os

import numpy as np

from . import binding, build, workloads as wl

SM_MHZ = 1965.0  # B200 SM clock under load on this pool (bench.py samples it; the cycle counts are exact, the us derived)


def _solver(workload, mode):
    if not os.path.exists(build.LIB_PROF):
        raise SystemExit(f"{build.LIB_PROF} is missing: python -m paper_2607_03226_b200.build -DBRICK_PROF -DMG_PROF")
    binding.LIB_PATH = build.LIB_PROF
    lib = binding.load()
    pr = wl.config_finfet(mode=mode) if workload == "finfet" else wl.config_cube(mode=mode)
    return lib, binding.Solver(pr)


def sweep(args):
    lib, g = _solver(args.workload, "plain")
    out = (C.c_ulonglong * 16)()
    for _ in range(3):
        g.step(mode=0)
    lib.nanobte_debug_brick_prof(out, 1)
    n_steps = 5
    for _ in range(n_steps):
        g.step(mode=0)
    lib.nanobte_debug_brick_prof(out, 0)
    v = np.array(list(out), dtype=np.float64)
    planes = max(v[6], 1.0)
    names = ["substitution (thread = system)", "barrier 1", "staging of the next plane, face loads, wall faces", "moments",
             "settling the tagged face values", "barrier 2"]
    print(f"{args.workload}: {int(planes / n_steps)} (task, plane) pairs per sweep; cycles per plane and CTA")
    for k, nm in enumerate(names):
        print(f"  {nm:54s} {v[k] / planes:8.0f}")
    print(f"  {'sum':54s} {v[:6].sum() / planes:8.0f}   settle re-loads per plane {v[7] / planes:.2f}")
    # timeline of the last sweep
    n = g.info["n_tasks"]
    buf = np.zeros((n, 4), dtype=np.uint64)
    lib.nanobte_debug_brick_timeline(buf.ctypes.data_as(C.c_void_p), n)
    t0, t1, t2 = (buf[:, k].astype(np.int64) for k in range(3))
    nu = ((buf[:, 3] >> np.uint64(32)) & np.uint64(0xffff)).astype(np.int64)
    base, end = t0.min(), t2.max()
    slots = 3 * 148
    print(f"timeline of one sweep: {n} tasks, {(end - base) / 1e3:.1f} us from the first ticket to the last task's end")
    print(f"  per CTA slot ({slots}): resident {(t2 - t0).sum() / 1e3 / slots:.1f} us, of which before the first plane "
          f"{(t1 - t0).sum() / 1e3 / slots:.1f} us; {(t2 - t1).sum() / nu.sum():.0f} ns per plane in the plane loop")
    edges = np.linspace(base, end, 31)
    print("  time us   resident tasks   tasks in their plane loop")
    for a, b in zip(edges[:-1], edges[1:]):
        res = np.clip(np.minimum(t2, b) - np.maximum(t0, a), 0, None).sum() / (b - a)
        run = np.clip(np.minimum(t2, b) - np.maximum(t1, a), 0, None).sum() / (b - a)
        print(f"  {(a - base) / 1e3:7.1f}   {res:14.1f}   {run:14.1f}")
    g.close()


def cg(args):
    lib, g = _solver(args.workload, "synthetic")
    out = (C.c_ulonglong * 16)()
    for _ in range(4):
        g.step(mode=1)
    lib.nanobte_debug_mg_prof(out, 1)
    for _ in range(5):
        g.step(mode=1)
    lib.nanobte_debug_mg_prof(out, 0)
    v = np.array(list(out), dtype=np.float64)
    its, solves = max(v[10], 1.0), max(v[15], 1.0)
    per_it = [(0, "level 0 down (2 Jacobi steps, exchange, residual, restriction)"), (1, "level 1 down"),
              (2, "level 2 down + gather of the level-3 right-hand side"), (3, "levels 3.. (every CTA, redundantly)"),
              (4, "level 2 up"), (5, "level 1 up"), (6, "level 0 up"), (7, "exchange of u, w = A u, dot products (all-to-all)"),
              (9, "CG vector updates")]
    print(f"{args.workload}: {its / solves:.1f} CG iterations per solve; us per iteration (CTA 0)")
    for k, nm in per_it:
        print(f"  {nm:66s} {v[k] / its / SM_MHZ:6.2f}")
    print(f"  {'sum':66s} {sum(v[k] for k, _ in per_it) / its / SM_MHZ:6.2f}")
    print("per solve, us: tables %.1f, right-hand side %.1f, recycled guess %.1f, kernel from start to end %.1f"
          % (v[11] / solves / SM_MHZ, v[12] / solves / SM_MHZ, v[13] / solves / SM_MHZ, v[14] / solves / SM_MHZ))
    g.close()


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("what", choices=["sweep", "cg"])
    ap.add_argument("--workload", default="finfet", choices=["finfet", "cube"])
    args = ap.parse_args()
    (sweep if args.what == "sweep" else cg)(args)


if __name__ == "__main__":
    main()
