"""ctypes binding of the CPU fp64 ORACLE (oracle/nanobte_ref.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  It imports nothing from the CUDA package and takes
plain numpy arrays (a "problem" dict as produced by paper_2607_03226_b200.workloads, or any
dict of the same shape) -- the oracle itself contains no input generation.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nanobte_ref.c")
_HDR = os.path.join(_HERE, "nanobte_ref.h")
_LIB = os.path.join(_HERE, "libnanobte_ref.so")
_lib = None

ERRORS = {0: "OK", 1: "NOT_CONVERGED", -1: "INVALID", -2: "ALLOC", -5: "UNTAGGED", -6: "SPECULAR",
          -7: "CYCLE", -8: "QUADRATURE", -9: "SINGULAR", -10: "NONFINITE"}


class OracleError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"nanobte_ref error {code} ({ERRORS.get(code, '?')}): {msg}")
        self.code = code


def build(force=False):
    """Compile the oracle with gcc (plain -O2, no contraction, OpenMP over direction tasks)."""
    stale = (not os.path.exists(_LIB)) or any(
        os.path.getmtime(p) > os.path.getmtime(_LIB) for p in (_SRC, _HDR))
    if force or stale:
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c11",
               "-Wall", "-Wextra", "-Wno-unused-parameter", _SRC, "-o", _LIB, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_up = C.POINTER(C.c_uint8)


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(build())
    vp = C.c_void_p
    tail = [C.c_int, _dp, _dp, _dp, _dp, C.c_int, _dp, _dp, C.c_int, _ip, _dp, _dp, C.c_double, _dp,
            C.c_double, C.c_int, C.POINTER(vp)]
    lib.nanobte_ref_create_structured.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _up, C.c_int, _ip, _up,
                                                  _ip, _dp] + tail
    lib.nanobte_ref_create_unstructured.argtypes = [C.c_int, _dp, C.c_int, _ip, _ip, C.c_int, _ip, _ip, _dp] + tail
    lib.nanobte_ref_destroy.argtypes = [vp]
    lib.nanobte_ref_destroy.restype = None
    lib.nanobte_ref_set_threads.argtypes = [vp, C.c_int]
    lib.nanobte_ref_sweep.argtypes = [vp]
    lib.nanobte_ref_update_temperature.argtypes = [vp, _dp]
    lib.nanobte_ref_diffusion_correct.argtypes = [vp, _ip, _dp]
    lib.nanobte_ref_init_fourier.argtypes = [vp, _ip]
    lib.nanobte_ref_solve.argtypes = [vp, C.c_double, C.c_int, C.c_int, _ip, _dp]
    lib.nanobte_ref_set_T.argtypes = [vp, _dp]
    lib.nanobte_ref_get_T.argtypes = [vp, C.c_int, _dp]
    lib.nanobte_ref_get_q.argtypes = [vp, _dp]
    lib.nanobte_ref_get_e.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, _dp, C.c_int]
    lib.nanobte_ref_get_G.argtypes = [vp, _dp]
    lib.nanobte_ref_get_boundary_values.argtypes = [vp, _dp]
    lib.nanobte_ref_get_boundary_heat.argtypes = [vp, _dp]
    lib.nanobte_ref_get_history.argtypes = [vp, _dp, _ip, C.c_int]
    lib.nanobte_ref_n_cells.argtypes = [vp]
    lib.nanobte_ref_n_active.argtypes = [vp]
    lib.nanobte_ref_kappa.argtypes = [vp]
    lib.nanobte_ref_kappa.restype = C.c_double
    lib.nanobte_ref_last_error.argtypes = [vp]
    lib.nanobte_ref_last_error.restype = C.c_char_p
    _lib = lib
    return lib


def _d(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _i(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.int32)


def _u(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.uint8)


def _p(a, typ):
    return None if a is None else a.ctypes.data_as(typ)


class RefSolver:
    """One oracle problem instance (same call shapes as the CUDA binding's Solver)."""

    def __init__(self, problem, T_init=None, cg_rtol=1e-12, cg_max_iter=100000, share=None, threads=None):
        lib = _load()
        self._lib = lib
        m, bands, quad = problem["mesh"], problem["bands"], problem["quad"]
        Cb, vb, tb = _d(bands["C"]), _d(bands["v"]), _d(bands["tau"])
        sh = _d(share)
        s, w = _d(quad["s"]), _d(quad["w"])
        tags = m["tags"]
        ttype = _i([t[0] for t in tags])
        tT = _d([t[1] for t in tags])
        Q = _d(problem["Qdot"])
        Ti = _d(T_init)
        self.B, self.D = len(Cb), len(w)
        self.n_tags = len(tags)
        h = C.c_void_p()
        tail = [self.B, _p(Cb, _dp), _p(vb, _dp), _p(tb, _dp), _p(sh, _dp), self.D, _p(s, _dp), _p(w, _dp),
                len(tags), _p(ttype, _ip), _p(tT, _dp), _p(Q, _dp), float(problem["T_ref"]), _p(Ti, _dp),
                float(cg_rtol), int(cg_max_iter), C.byref(h)]
        if problem["kind"] == "structured":
            hx, hy, hz = _d(m["hx"]), _d(m["hy"]), _d(m["hz"])
            act = _u(m["active"])
            bc, bs, bt, bp = _i(m["bf_cell"]), _u(m["bf_side"]), _i(m["bf_tag"]), _d(m["bf_p"])
            rc = lib.nanobte_ref_create_structured(
                m["nx"], m["ny"], m["nz"], _p(hx, _dp), _p(hy, _dp), _p(hz, _dp), _p(act, _up), len(bc),
                _p(bc, _ip), _p(bs, _up), _p(bt, _ip), _p(bp, _dp), *tail)
            self.dim = 3 if m["nz"] > 1 else 2
        else:
            xy = _d(m["xy"])
            cp, cn = _i(m["cell_ptr"]), _i(m["cell_nodes"])
            bn, bt, bp = _i(m["bf_nodes"]), _i(m["bf_tag"]), _d(m["bf_p"])
            rc = lib.nanobte_ref_create_unstructured(
                m["n_nodes"], _p(xy, _dp), m["n_cells"], _p(cp, _ip), _p(cn, _ip), len(bt), _p(bn, _ip),
                _p(bt, _ip), _p(bp, _dp), *tail)
            self.dim = 2
        self._h = h
        self.n_bf = len(bt)
        if rc < 0:
            msg = lib.nanobte_ref_last_error(h).decode() if h else "create failed"
            if h:
                lib.nanobte_ref_destroy(h)
            self._h = None
            raise OracleError(rc, msg)
        self.n_cells = lib.nanobte_ref_n_cells(h)
        self.n_active = lib.nanobte_ref_n_active(h)
        self.kappa = lib.nanobte_ref_kappa(h)
        self.threads = lib.nanobte_ref_set_threads(h, threads if threads else 0)

    def _chk(self, rc):
        if rc < 0:
            raise OracleError(rc, self._lib.nanobte_ref_last_error(self._h).decode())
        return rc

    def close(self):
        if getattr(self, "_h", None):
            self._lib.nanobte_ref_destroy(self._h)
            self._h = None

    __del__ = close

    def set_threads(self, n):
        self.threads = self._lib.nanobte_ref_set_threads(self._h, int(n))
        return self.threads

    def sweep(self):
        self._chk(self._lib.nanobte_ref_sweep(self._h))

    def update_temperature(self):
        d = C.c_double()
        self._chk(self._lib.nanobte_ref_update_temperature(self._h, C.byref(d)))
        return d.value

    def diffusion_correct(self):
        it, d = C.c_int32(), C.c_double()
        self._chk(self._lib.nanobte_ref_diffusion_correct(self._h, C.byref(it), C.byref(d)))
        return it.value, d.value

    def init_fourier(self):
        """O9 / R21: theta <- solution of the steady heat-conduction problem; returns the CG iterations."""
        it = C.c_int32()
        self._chk(self._lib.nanobte_ref_init_fourier(self._h, C.byref(it)))
        return it.value

    def solve(self, tol, max_iter, mode="plain"):
        it, d = C.c_int32(), C.c_double()
        rc = self._chk(self._lib.nanobte_ref_solve(self._h, float(tol), int(max_iter),
                                                   1 if mode in (1, "synthetic") else 0, C.byref(it), C.byref(d)))
        return {"converged": rc == 0, "iters": it.value, "last_dT": d.value}

    def set_T(self, T):
        T = _d(T)
        assert T.size == self.n_cells
        self._chk(self._lib.nanobte_ref_set_T(self._h, _p(T, _dp)))

    def get_T(self, which=0):
        out = np.empty(self.n_cells)
        self._chk(self._lib.nanobte_ref_get_T(self._h, int(which), _p(out, _dp)))
        return out

    def get_q(self):
        out = np.empty((self.n_cells, self.dim))
        self._chk(self._lib.nanobte_ref_get_q(self._h, _p(out, _dp)))
        return out

    def get_e(self, b0=0, nb=None, d0=0, nd=None, deviational=True):
        nb = self.B - b0 if nb is None else nb
        nd = self.D - d0 if nd is None else nd
        out = np.empty((nb, nd, self.n_cells))
        self._chk(self._lib.nanobte_ref_get_e(self._h, b0, nb, d0, nd, _p(out, _dp), 1 if deviational else 0))
        return out

    def get_G(self):
        out = np.empty((self.n_bf, self.B))
        self._chk(self._lib.nanobte_ref_get_G(self._h, _p(out, _dp)))
        return out

    def get_boundary_values(self):
        out = np.empty((self.n_bf, self.B, self.D))
        self._chk(self._lib.nanobte_ref_get_boundary_values(self._h, _p(out, _dp)))
        return out

    def get_boundary_heat(self):
        out = np.empty(self.n_tags)
        self._chk(self._lib.nanobte_ref_get_boundary_heat(self._h, _p(out, _dp)))
        return out

    def get_history(self):
        n = self._lib.nanobte_ref_get_history(self._h, None, None, 0)
        dT, cg = np.empty(n), np.empty(n, dtype=np.int32)
        self._lib.nanobte_ref_get_history(self._h, _p(dT, _dp), _p(cg, _ip), n)
        return dT, cg
