"""Band-sharded data parallelism (Eq. 14): the (direction, band) transport tasks are
distributed over the ranks, the mesh is replicated, and the contributions to the update are merged with ONE all-reduce per
source iteration.

One process per GPU.  Every rank creates a solver on its subset of the band table (round-robin, as in the paper,
PAPER.md:228) with the sums over the whole table handed in (nanobte_options.beta_total / Csum_total / kappa_total), sweeps
its bands, exports its terms of (T_SI, T_energy, q, reflecting-face leak) -- 5 n_active + n_bfaces doubles --, all-reduces
them over NCCL (torch.distributed; NVLink/NVSwitch do the rest), and imports the sums: all ranks then hold the same lattice
temperature, and in synthetic mode solve the same diffusion system redundantly (it is latency-bound and small).  Wall
closures never mix bands, so nothing else crosses ranks.  This module is plumbing (band split, buffers, the collective);
every step of the arithmetic runs in libnanobte's kernels.

Nothing here has run on more than one GPU (the build environment has one); tests/test_sharded_gloo.py exercises the same
driver with two CPU processes over gloo, tests/test_parity_gpu.py two shards on one GPU against the unsharded solver.
"""
from __future__ import annotations

import ctypes as C

import numpy as np


def shard_bands(n_bands: int, rank: int, world: int):
    """Bands of a rank: round-robin over the band index; every rank gets at least one band."""
    if not (0 <= rank < world) or world > n_bands:
        raise ValueError(f"cannot split {n_bands} bands over {world} ranks")
    return list(range(rank, n_bands, world))


def shard_problem(problem, rank: int, world: int):
    """The problem dict of one rank: same mesh, quadrature, walls and source; the rank's rows of the band table."""
    idx = shard_bands(len(problem["bands"]["C"]), rank, world)
    sub = dict(problem)
    sub["bands"] = {k: np.ascontiguousarray(np.asarray(v)[idx]) for k, v in problem["bands"].items()}
    return sub


def band_totals(problem):
    """(beta, sum C, kappa) of the WHOLE band table, computed by the library (nanobte_band_totals)."""
    from . import binding
    lib = binding.load()
    ms = binding._Marshalled(problem)
    out = (C.c_double * 3)()
    rc = lib.nanobte_band_totals(C.byref(ms.bands), C.byref(ms.quad), int(ms.dim), out)
    if rc < 0:
        raise binding.NanoBTEError(rc, lib.nanobte_strerror(rc).decode())
    return float(out[0]), float(out[1]), float(out[2])


def allreduce_sum(buf, dist):
    """One all-reduce (sum) of the update tensor over the ranks; no-op without a process group."""
    if dist is not None:
        dist.all_reduce(buf, op=dist.ReduceOp.SUM)
    return buf


class ShardedSolver:
    """A rank's solver plus the collective.  `make_solver(sub_problem, totals)` builds the local engine; the default is the
    CUDA library.  (The gloo test passes a CPU stand-in with the same four methods.)"""

    def __init__(self, problem, rank: int, world: int, dist=None, make_solver=None, **kw):
        self.rank, self.world, self.dist = rank, world, dist
        self.bands = shard_bands(len(problem["bands"]["C"]), rank, world)
        sub = shard_problem(problem, rank, world)
        if make_solver is None:
            from .binding import Solver
            totals = band_totals(problem)
            self.local = Solver(sub, totals=totals, **kw)
            self.local.set_keep_e(False)
        else:
            self.local = make_solver(sub, problem)
        self.hist_dT, self.hist_cg = [], []

    def local_update(self):
        """Sweep the rank's bands and reduce them: returns the buffer with this rank's terms of the update."""
        self.local.sweep()
        self.local.update_temperature(sync=False)
        return self.local.export_moments()

    def finish(self, summed, mode="plain"):
        """Import the all-reduced terms (T <- T_SI); in synthetic mode the diffusion correction on top.  Returns
        (max|dT|, CG iterations)."""
        dT, it = self.local.import_moments(summed), 0
        if mode in (1, "synthetic"):
            it, dT = self.local.diffusion_correct()
        return dT, it

    def step(self, mode="plain"):
        return self.finish(allreduce_sum(self.local_update(), self.dist), mode)

    def solve(self, tol, max_iter, mode="plain"):
        n, dT = 0, float("inf")
        self.hist_dT, self.hist_cg = [], []
        while n < max_iter:
            dT, it = self.step(mode)
            n += 1
            self.hist_dT.append(dT)
            self.hist_cg.append(it)
            if dT < tol:
                return {"converged": True, "iters": n, "last_dT": dT}
        return {"converged": False, "iters": n, "last_dT": dT}

    def close(self):
        self.local.close()
