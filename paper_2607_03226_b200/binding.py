"""Thin Python binding of libnanobte (include/nanobte.h): argument marshalling only.

Every step of the hot path (closures, sweep, moments, CG, convergence loop) runs inside the CUDA library; this
module converts numpy problem descriptions into the C structs, lends the library a torch-owned device workspace
and torch's current CUDA stream, and hands results back as numpy arrays or torch tensors.  It never imports
``oracle/`` and has no CPU fallback: without the built library or without a CUDA device it raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnanobte.so")

ERRORS = {0: "OK", 1: "NOT_CONVERGED", -1: "INVALID", -2: "ALLOC", -3: "CUDA", -4: "ARCH", -5: "UNTAGGED",
          -6: "SPECULAR", -7: "CYCLE", -8: "QUADRATURE", -9: "SINGULAR", -10: "NONFINITE", -11: "UNSUPPORTED"}

EXPORTS = [
    "nanobte_workspace_bytes_structured", "nanobte_workspace_bytes_unstructured", "nanobte_create_structured",
    "nanobte_create_unstructured", "nanobte_destroy", "nanobte_sweep", "nanobte_update_temperature",
    "nanobte_diffusion_correct", "nanobte_init_fourier", "nanobte_band_totals", "nanobte_moments_len", "nanobte_export_moments",
    "nanobte_import_moments", "nanobte_step", "nanobte_set_keep_e", "nanobte_solve", "nanobte_set_T", "nanobte_get_T", "nanobte_get_q", "nanobte_get_e",
    "nanobte_get_G", "nanobte_get_boundary_heat", "nanobte_get_boundary_heat_noalloc", "nanobte_get_history", "nanobte_get_info", "nanobte_launch_count",
    "nanobte_kappa", "nanobte_strerror", "nanobte_last_error",
]

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_up = C.POINTER(C.c_uint8)


class Bands(C.Structure):
    _fields_ = [("B", C.c_int32), ("C", _dp), ("v", _dp), ("tau", _dp), ("src_share", _dp)]


class Quadrature(C.Structure):
    _fields_ = [("D", C.c_int32), ("s", _dp), ("w", _dp)]


class Tag(C.Structure):
    _fields_ = [("type", C.c_int32), ("T_wall", C.c_double)]


class StructuredMesh(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("hx", _dp), ("hy", _dp), ("hz", _dp),
                ("active", _up), ("n_bfaces", C.c_int32), ("bf_cell", _ip), ("bf_side", _up), ("bf_tag", _ip),
                ("bf_p", _dp)]


class UnstructuredMesh(C.Structure):
    _fields_ = [("n_nodes", C.c_int32), ("n_cells", C.c_int32), ("xy", _dp), ("cell_ptr", _ip), ("cell_nodes", _ip),
                ("n_bfaces", C.c_int32), ("bf_nodes", _ip), ("bf_tag", _ip), ("bf_p", _dp)]


class Options(C.Structure):
    _fields_ = [("T_ref", C.c_double), ("T_init", _dp), ("stream", C.c_void_p), ("workspace", C.c_void_p),
                ("workspace_bytes", C.c_size_t), ("cg_rtol", C.c_double), ("cg_max_iter", C.c_int32),
                ("sweep_G", C.c_int32), ("sweep_threads", C.c_int32), ("sweep_variant", C.c_int32),
                ("beta_total", C.c_double), ("Csum_total", C.c_double), ("kappa_total", C.c_double)]


class Info(C.Structure):
    _fields_ = [("dim", C.c_int32), ("n_cells", C.c_int32), ("n_active", C.c_int32), ("B", C.c_int32), ("D", C.c_int32),
                ("n_bfaces", C.c_int32), ("n_octants", C.c_int32), ("n_planes", C.c_int32), ("n_tasks", C.c_int32),
                ("sweep_G", C.c_int32), ("sweep_threads", C.c_int32),
                ("sweep_rmax", C.c_int32), ("pencil_axis", C.c_int32), ("n_pos", C.c_int64), ("n_inflow", C.c_int64),
                ("device_bytes", C.c_size_t), ("sweep_smem_bytes", C.c_size_t), ("cg_fused", C.c_int32),
                ("cg_cells_per_thread", C.c_int32), ("cg_ctas", C.c_int32), ("cg_face_uniform", C.c_int32),
                ("cg_recycle", C.c_int32), ("sweep_variant", C.c_int32), ("cg_multigrid", C.c_int32),
                ("cg_mg_levels", C.c_int32)]


class NanoBTEError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"nanobte error {code} ({ERRORS.get(code, '?')}): {msg}")
        self.code = code


_lib = None


def load():
    """dlopen the in-tree CUDA library; raises if it has not been built (no fallback of any kind)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2607_03226_b200.build` (needs nvcc). "
                          "There is no CPU fallback.")
    lib = C.CDLL(LIB_PATH)
    vp, pvp = C.c_void_p, C.POINTER(C.c_void_p)
    pS, pU, pB, pQ, pT, pO = (C.POINTER(StructuredMesh), C.POINTER(UnstructuredMesh), C.POINTER(Bands),
                              C.POINTER(Quadrature), C.POINTER(Tag), C.POINTER(Options))
    lib.nanobte_workspace_bytes_structured.argtypes = [pS, pB, pQ, pT, C.c_int32, pO, C.POINTER(C.c_size_t)]
    lib.nanobte_workspace_bytes_unstructured.argtypes = [pU, pB, pQ, pT, C.c_int32, pO, C.POINTER(C.c_size_t)]
    lib.nanobte_create_structured.argtypes = [pS, pB, pQ, pT, C.c_int32, _dp, pO, pvp]
    lib.nanobte_create_unstructured.argtypes = [pU, pB, pQ, pT, C.c_int32, _dp, pO, pvp]
    lib.nanobte_destroy.argtypes = [vp]
    lib.nanobte_destroy.restype = None
    lib.nanobte_sweep.argtypes = [vp]
    lib.nanobte_update_temperature.argtypes = [vp, _dp]
    lib.nanobte_diffusion_correct.argtypes = [vp, _ip, _dp]
    lib.nanobte_init_fourier.argtypes = [vp, _ip]
    lib.nanobte_moments_len.argtypes = [vp]
    lib.nanobte_moments_len.restype = C.c_int64
    lib.nanobte_export_moments.argtypes = [vp, C.c_void_p, C.c_int32]
    lib.nanobte_import_moments.argtypes = [vp, C.c_void_p, C.c_int32, _dp]
    lib.nanobte_step.argtypes = [vp, C.c_int32, _dp, _ip]
    lib.nanobte_set_keep_e.argtypes = [vp, C.c_int32]
    lib.nanobte_solve.argtypes = [vp, C.c_double, C.c_int32, C.c_int32, _ip, _dp]
    lib.nanobte_set_T.argtypes = [vp, vp, C.c_int32]
    lib.nanobte_get_T.argtypes = [vp, C.c_int32, vp, C.c_int32]
    lib.nanobte_get_q.argtypes = [vp, vp, C.c_int32]
    lib.nanobte_get_e.argtypes = [vp, C.c_int32, C.c_int32, C.c_int32, C.c_int32, vp, C.c_int32, C.c_int32]
    lib.nanobte_get_G.argtypes = [vp, vp, C.c_int32]
    lib.nanobte_get_boundary_heat.argtypes = [vp, _dp]
    lib.nanobte_get_boundary_heat_noalloc.argtypes = [vp, vp, C.c_int32]
    lib.nanobte_get_history.argtypes = [vp, _dp, _ip, C.c_int32]
    lib.nanobte_get_info.argtypes = [vp, C.POINTER(Info)]
    lib.nanobte_launch_count.argtypes = [vp]
    lib.nanobte_launch_count.restype = C.c_int64
    lib.nanobte_kappa.argtypes = [vp]
    lib.nanobte_kappa.restype = C.c_double
    lib.nanobte_strerror.argtypes = [C.c_int]
    lib.nanobte_strerror.restype = C.c_char_p
    lib.nanobte_last_error.argtypes = [vp]
    lib.nanobte_last_error.restype = C.c_char_p
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


class _Marshalled:
    """C structs for one problem dict, keeping the numpy arrays they point at alive."""

    def __init__(self, problem, T_init=None, share=None):
        m, bands, quad = problem["mesh"], problem["bands"], problem["quad"]
        k = self.keep = {}
        k["C"], k["v"], k["tau"], k["share"] = _d(bands["C"]), _d(bands["v"]), _d(bands["tau"]), _d(share)
        k["s"], k["w"] = _d(quad["s"]), _d(quad["w"])
        self.bands = Bands(len(k["C"]), _p(k["C"], _dp), _p(k["v"], _dp), _p(k["tau"], _dp), _p(k["share"], _dp))
        self.quad = Quadrature(len(k["w"]), _p(k["s"], _dp), _p(k["w"], _dp))
        tags = m["tags"]
        self.n_tags = len(tags)
        self.tags = (Tag * max(1, len(tags)))(*[Tag(int(t[0]), float(t[1])) for t in tags])
        k["Q"] = _d(problem.get("Qdot"))
        k["Ti"] = _d(T_init)
        self.kind = problem["kind"]
        if self.kind == "structured":
            k["hx"], k["hy"], k["hz"] = _d(m["hx"]), _d(m["hy"]), _d(m["hz"])
            k["act"] = _u(m["active"])
            k["bc"], k["bs"], k["bt"], k["bp"] = _i(m["bf_cell"]), _u(m["bf_side"]), _i(m["bf_tag"]), _d(m["bf_p"])
            self.mesh = StructuredMesh(m["nx"], m["ny"], m["nz"], _p(k["hx"], _dp), _p(k["hy"], _dp), _p(k["hz"], _dp),
                                       _p(k["act"], _up), len(k["bc"]), _p(k["bc"], _ip), _p(k["bs"], _up),
                                       _p(k["bt"], _ip), _p(k["bp"], _dp))
            self.n_cells = m["nx"] * m["ny"] * m["nz"]
            self.dim = 3 if m["nz"] > 1 else 2
        else:
            k["xy"] = _d(m["xy"])
            k["cp"], k["cn"] = _i(m["cell_ptr"]), _i(m["cell_nodes"])
            k["bn"], k["bt"], k["bp"] = _i(m["bf_nodes"]), _i(m["bf_tag"]), _d(m["bf_p"])
            self.mesh = UnstructuredMesh(m["n_nodes"], m["n_cells"], _p(k["xy"], _dp), _p(k["cp"], _ip),
                                         _p(k["cn"], _ip), len(k["bt"]), _p(k["bn"], _ip), _p(k["bt"], _ip),
                                         _p(k["bp"], _dp))
            self.n_cells = m["n_cells"]
            self.dim = 2
        self.n_bf = len(k["bt"])


def workspace_bytes(problem, sweep_G=0, sweep_threads=0, sweep_variant=0):
    """Device bytes a Solver for this problem needs (host-only call; also validates the problem)."""
    lib = load()
    ms = _Marshalled(problem)
    opt = Options(float(problem["T_ref"]), None, None, None, 0, 0.0, 0, sweep_G, sweep_threads, sweep_variant, 0.0, 0.0, 0.0)
    out = C.c_size_t()
    fn = lib.nanobte_workspace_bytes_structured if ms.kind == "structured" else lib.nanobte_workspace_bytes_unstructured
    rc = fn(C.byref(ms.mesh), C.byref(ms.bands), C.byref(ms.quad), ms.tags, ms.n_tags, C.byref(opt), C.byref(out))
    if rc < 0:
        raise NanoBTEError(rc, lib.nanobte_strerror(rc).decode())
    return out.value


class Solver:
    """One problem instance on the current CUDA device (same call shapes as the C ABI)."""

    def __init__(self, problem, T_init=None, cg_rtol=1e-12, cg_max_iter=100000, share=None, sweep_G=0,
                 sweep_threads=0, sweep_variant=0, own_workspace=True, totals=None):
        """totals = (beta, Csum, kappa) of the whole band table when `problem` carries a band shard (nanobte_options)."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("nanobte needs a CUDA device (sm_100); there is no CPU fallback")
        lib = load()
        self._lib, self._torch = lib, torch
        ms = _Marshalled(problem, T_init, share)
        self.kind, self.dim, self.n_cells, self.n_bf, self.n_tags = ms.kind, ms.dim, ms.n_cells, ms.n_bf, ms.n_tags
        self.B, self.D = ms.bands.B, ms.quad.D
        self.stream = torch.cuda.current_stream()
        opt = Options(float(problem["T_ref"]), _p(ms.keep["Ti"], _dp), C.c_void_p(self.stream.cuda_stream), None, 0,
                      float(cg_rtol), int(cg_max_iter), int(sweep_G), int(sweep_threads), int(sweep_variant),
                      *(tuple(float(x) for x in totals) if totals is not None else (0.0, 0.0, 0.0)))
        structured = ms.kind == "structured"
        self._ws = None
        if own_workspace:  # device memory is a torch tensor (PyTorch: buffers and streams only)
            need = C.c_size_t()
            fn = lib.nanobte_workspace_bytes_structured if structured else lib.nanobte_workspace_bytes_unstructured
            rc = fn(C.byref(ms.mesh), C.byref(ms.bands), C.byref(ms.quad), ms.tags, ms.n_tags, C.byref(opt), C.byref(need))
            if rc < 0:
                raise NanoBTEError(rc, lib.nanobte_strerror(rc).decode())
            self._ws = torch.empty(need.value + 256, dtype=torch.uint8, device="cuda")
            base = (self._ws.data_ptr() + 255) // 256 * 256
            opt.workspace, opt.workspace_bytes = C.c_void_p(base), need.value
        h = C.c_void_p()
        fn = lib.nanobte_create_structured if structured else lib.nanobte_create_unstructured
        rc = fn(C.byref(ms.mesh), C.byref(ms.bands), C.byref(ms.quad), ms.tags, ms.n_tags, _p(ms.keep["Q"], _dp),
                C.byref(opt), C.byref(h))
        self._h = h
        if rc < 0:
            msg = lib.nanobte_last_error(h).decode() if h else "create failed"
            if h:
                lib.nanobte_destroy(h)
            self._h = None
            raise NanoBTEError(rc, msg)
        info = Info()
        lib.nanobte_get_info(h, C.byref(info))
        self.info = {f[0]: getattr(info, f[0]) for f in Info._fields_}
        self.n_active = info.n_active
        self.kappa = lib.nanobte_kappa(h)

    # -- plumbing -----------------------------------------------------------------------------------------------
    def _chk(self, rc):
        if rc < 0:
            raise NanoBTEError(rc, self._lib.nanobte_last_error(self._h).decode())
        return rc

    def close(self):
        if getattr(self, "_h", None):
            self._lib.nanobte_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def launches(self):
        return self._lib.nanobte_launch_count(self._h)

    # -- the hot path ---------------------------------------------------------------------------------------------
    def sweep(self):
        self._chk(self._lib.nanobte_sweep(self._h))

    def set_keep_e(self, keep):
        self._chk(self._lib.nanobte_set_keep_e(self._h, 1 if keep else 0))

    def update_temperature(self, sync=True):
        if not sync:
            self._chk(self._lib.nanobte_update_temperature(self._h, None))
            return None
        d = C.c_double()
        self._chk(self._lib.nanobte_update_temperature(self._h, C.byref(d)))
        return d.value

    def diffusion_correct(self):
        it, d = C.c_int32(), C.c_double()
        self._chk(self._lib.nanobte_diffusion_correct(self._h, C.byref(it), C.byref(d)))
        return it.value, d.value

    def export_moments(self, out=None):
        """nanobte_export_moments into a device tensor (torch, float64, nanobte_moments_len long): this shard's terms."""
        n = int(self._lib.nanobte_moments_len(self._h))
        if out is None:
            out = self._torch.empty(n, dtype=self._torch.float64, device="cuda")
        assert out.is_cuda and out.dtype == self._torch.float64 and out.numel() == n and out.is_contiguous()
        self._chk(self._lib.nanobte_export_moments(self._h, C.c_void_p(out.data_ptr()), 1))
        return out

    def import_moments(self, buf, sync=True):
        """nanobte_import_moments from a device tensor holding the element-wise sum over all shards; returns max|dT|."""
        assert buf.is_cuda and buf.dtype == self._torch.float64 and buf.is_contiguous()
        d = C.c_double()
        self._chk(self._lib.nanobte_import_moments(self._h, C.c_void_p(buf.data_ptr()), 1, C.byref(d) if sync else None))
        return d.value if sync else None

    def init_fourier(self):
        """nanobte_init_fourier: T <- Fourier (steady conduction) solution, PAPER.md:228 / R21; returns the CG iterations."""
        it = C.c_int32()
        self._chk(self._lib.nanobte_init_fourier(self._h, C.byref(it)))
        return it.value

    def step(self, mode="plain"):
        """One source iteration as solve() runs it; returns (max|dT|, CG iterations)."""
        it, d = C.c_int32(), C.c_double()
        self._chk(self._lib.nanobte_step(self._h, 1 if mode in (1, "synthetic") else 0, C.byref(d), C.byref(it)))
        return d.value, it.value

    def solve(self, tol, max_iter, mode="plain"):
        it, d = C.c_int32(), C.c_double()
        rc = self._chk(self._lib.nanobte_solve(self._h, float(tol), int(max_iter),
                                               1 if mode in (1, "synthetic") else 0, C.byref(it), C.byref(d)))
        return {"converged": rc == 0, "iters": it.value, "last_dT": d.value}

    # -- state in / out ---------------------------------------------------------------------------------------------
    def set_T(self, T):
        torch = self._torch
        if isinstance(T, torch.Tensor):
            assert T.is_cuda and T.dtype == torch.float64 and T.numel() == self.n_cells and T.is_contiguous()
            self._chk(self._lib.nanobte_set_T(self._h, C.c_void_p(T.data_ptr()), 1))
        else:
            T = _d(T)
            assert T.size == self.n_cells
            self._chk(self._lib.nanobte_set_T(self._h, T.ctypes.data_as(C.c_void_p), 0))

    def _out(self, shape, device):
        if device:
            t = self._torch.empty(shape, dtype=self._torch.float64, device="cuda")
            return t, C.c_void_p(t.data_ptr())
        a = np.empty(shape)
        return a, a.ctypes.data_as(C.c_void_p)

    def get_T(self, which=0, device=False, out=None):
        """`out`: optional host destination (a contiguous float64 numpy array of n_cells, e.g. the numpy view of a pinned
        torch tensor, which makes the device-to-host copy a true DMA)."""
        if out is not None and not device:
            assert out.dtype == np.float64 and out.size == self.n_cells and out.flags["C_CONTIGUOUS"]
            self._chk(self._lib.nanobte_get_T(self._h, int(which), out.ctypes.data_as(C.c_void_p), 0))
            return out
        out, p = self._out((self.n_cells,), device)
        self._chk(self._lib.nanobte_get_T(self._h, int(which), p, int(device)))
        return out

    def get_q(self, device=False):
        out, p = self._out((self.n_cells, self.dim), device)
        self._chk(self._lib.nanobte_get_q(self._h, p, int(device)))
        return out

    def get_e(self, b0=0, nb=None, d0=0, nd=None, deviational=True, device=False):
        nb = self.B - b0 if nb is None else nb
        nd = self.D - d0 if nd is None else nd
        out, p = self._out((nb, nd, self.n_cells), device)
        self._chk(self._lib.nanobte_get_e(self._h, b0, nb, d0, nd, p, 1 if deviational else 0, int(device)))
        return out

    def get_G(self, device=False):
        out, p = self._out((self.n_bf, self.B), device)
        self._chk(self._lib.nanobte_get_G(self._h, p, int(device)))
        return out

    def get_boundary_heat(self):
        out = np.zeros(max(1, self.n_tags))
        self._chk(self._lib.nanobte_get_boundary_heat(self._h, out.ctypes.data_as(_dp)))
        return out[:self.n_tags]

    def get_boundary_heat_noalloc(self, device=False):
        """nanobte_get_boundary_heat_noalloc: the same per-tag heat through the library's static scratch (no allocation
        below the C-ABI; at most NANOBTE_NOALLOC_MAX_TAGS = 256 tags)."""
        out, p = self._out((max(1, self.n_tags),), device)
        self._chk(self._lib.nanobte_get_boundary_heat_noalloc(self._h, p, int(device)))
        return out[:self.n_tags]

    def get_history(self):
        n = self._lib.nanobte_get_history(self._h, None, None, 0)
        dT, cg = np.empty(n), np.empty(n, dtype=np.int32)
        self._lib.nanobte_get_history(self._h, _p(dT, _dp), _p(cg, _ip), n)
        return dT, cg
