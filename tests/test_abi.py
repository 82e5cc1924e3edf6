"""CPU-side checks of the C-ABI library: it builds, loads without a GPU, exports every symbol include/nanobte.h
declares, its host-side setup (validation, schedules, workspace sizing) runs, and it fails loudly -- never falls
back -- when no CUDA device is present."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2607_03226_b200 import workloads as wl
from paper_2607_03226_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def test_exports_every_declared_symbol(lib):
    hdr = open(os.path.join(ROOT, "include", "nanobte.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(nanobte_[a-z_A-Z0-9]+)\s*\(", hdr))
    assert declared, "no declarations parsed"
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name


def test_struct_layouts_match_header(lib, tmp_path):
    """Sizes and field offsets the C compiler gives the ABI structs of include/nanobte.h (gcc, LP64) against the ctypes
    mirrors in binding.py: a drifted mirror would corrupt every call."""
    import subprocess
    structs = {"nanobte_bands": binding.Bands, "nanobte_quadrature": binding.Quadrature, "nanobte_tag": binding.Tag,
               "nanobte_structured_mesh": binding.StructuredMesh, "nanobte_unstructured_mesh": binding.UnstructuredMesh,
               "nanobte_options": binding.Options, "nanobte_info": binding.Info}
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "nanobte.h"', 'int main(void) {']
    for cname, cls in structs.items():
        lines.append(f'printf("{cname} %zu\\n", sizeof({cname}));')
        for fname, _ in cls._fields_:
            lines.append(f'printf("{cname}.{fname} %zu\\n", offsetof({cname}, {fname}));')
    lines += ['return 0;', '}']
    src = tmp_path / "abi.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "abi"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    got = dict(ln.split() for ln in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.splitlines())
    for cname, cls in structs.items():
        assert int(got[cname]) == C.sizeof(cls), cname
        for fname, _ in cls._fields_:
            assert int(got[f"{cname}.{fname}"]) == getattr(cls, fname).offset, f"{cname}.{fname}"


def test_strerror(lib):
    assert lib.nanobte_strerror(0) == b"OK" and lib.nanobte_strerror(-4) == b"ARCH" and lib.nanobte_strerror(-11) == b"UNSUPPORTED"


@pytest.mark.parametrize("name,kw,nupd", [
    ("gray_square", {}, 6400),
    ("nongray_square", {}, 5242880),
    ("cube", {"n": 16}, 16**3 * 20 * 128),
    ("finfet", {"nx": 32, "ny": 16, "nz": 16}, None),
])
def test_workspace_bytes_and_host_setup(lib, name, kw, nupd):
    pr = wl.CONFIGS[name](**kw)
    nbytes = binding.workspace_bytes(pr)
    n_e = wl.n_updates(pr) * 8
    if nupd is not None:
        assert wl.n_updates(pr) == nupd
    assert nbytes > n_e  # the e array dominates; tables and caches come on top
    # tile-dataflow path: positions padded to 64 per tile plane, tile-face and wall rows at a pitch of 128 systems, partial
    # moments, multigrid tables -- on a grid this small (tiles 4 cells wide) that is up to ~4x the distribution itself
    assert nbytes < 4 * n_e + (64 << 20)


def test_host_validation_errors(lib):
    pr = wl.config_gray_square(n=6)
    bad = dict(pr, quad={"s": pr["quad"]["s"] * 1.1, "w": pr["quad"]["w"], "dim": 2})
    with pytest.raises(binding.NanoBTEError) as e:
        binding.workspace_bytes(bad)
    assert e.value.code == -8
    m = dict(pr["mesh"])
    m["bf_cell"], m["bf_side"], m["bf_tag"] = m["bf_cell"][1:], m["bf_side"][1:], m["bf_tag"][1:]
    with pytest.raises(binding.NanoBTEError) as e:
        binding.workspace_bytes(dict(pr, mesh=m))
    assert e.value.code == -5
    spec = wl.config_gray_square(n=6, wall=wl.SPECULAR)
    q = wl.inplane_quadrature(16)
    q["s"] = q["s"][:-2].copy()
    q["w"] = q["w"][:-2].copy()
    # a quadrature that is not closed under reflection: first failure is sum w s != 0
    with pytest.raises(binding.NanoBTEError):
        binding.workspace_bytes(dict(spec, quad=q))
    b = dict(pr["bands"])
    b["tau"] = np.array([-1.0])
    with pytest.raises(binding.NanoBTEError) as e:
        binding.workspace_bytes(dict(pr, bands=b))
    assert e.value.code == -1


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    with pytest.raises(RuntimeError):
        binding.Solver(wl.config_gray_square(n=4))
    # straight through the C ABI: create must refuse with NANOBTE_E_ARCH
    ms = binding._Marshalled(wl.config_gray_square(n=4))
    opt = binding.Options(300.0, None, None, None, 0, 0.0, 0, 0, 0)
    h = C.c_void_p()
    rc = lib.nanobte_create_structured(C.byref(ms.mesh), C.byref(ms.bands), C.byref(ms.quad), ms.tags, ms.n_tags, None,
                                       C.byref(opt), C.byref(h))
    assert rc == -4
    assert b"no CPU fallback" in lib.nanobte_last_error(h) or b"CUDA" in lib.nanobte_last_error(h)
    lib.nanobte_destroy(h)


def test_band_totals_closed_forms(lib):
    """nanobte_band_totals (host only): beta = sum C/tau (Eq. 5), sum C (R13), kappa = (1/dim) sum C v^2 tau
    (R14d: kinetic-theory value for unit directions spanning the mesh dimension) for the tables of configs 2 and 4."""
    from paper_2607_03226_b200 import sharded
    for pr, dim in ((wl.config_nongray_square(n=8), 2), (wl.config_finfet(nx=8, ny=4, nz=4), 3)):
        beta, Csum, kappa = sharded.band_totals(pr)
        b = pr["bands"]
        assert beta == pytest.approx((b["C"] / b["tau"]).sum(), rel=1e-14)
        assert Csum == pytest.approx(b["C"].sum(), rel=1e-14)
        assert kappa == pytest.approx((b["C"] * b["v"] ** 2 * b["tau"]).sum() / dim, rel=1e-12)
        # a shard's rows are the rank's round-robin share of the table
        sub = sharded.shard_problem(pr, 1, 3)
        assert np.array_equal(sub["bands"]["C"], b["C"][1::3]) and sub["mesh"] is pr["mesh"]
