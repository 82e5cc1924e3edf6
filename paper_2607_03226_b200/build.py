"""Builds libnanobte.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2607_03226_b200.build [--force] [-v]
    python -m paper_2607_03226_b200.build -DBRICK_PROF -DMG_PROF     # instrumented copy, see prof.py

The result, paper_2607_03226_b200/libnanobte.so, is git-ignored but travels to the GPU box with the snapshot.
cudart is linked statically, so the library loads (and its symbols can be checked) on a machine without a GPU.
With -D defines the result is a second library, libnanobte_prof.so, with clock64()/globaltimer probes in the
tile-dataflow sweep (BRICK_PROF) and the multigrid CG (MG_PROF); the product never loads it (prof.py does).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INC = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libnanobte.so")
LIB_PROF = os.path.join(HERE, "libnanobte_prof.so")
SOURCES = ["api.cu", "setup_structured.cu", "sweep_structured.cu", "kernels_common.cu", "cg.cu", "sweep_unstructured.cu",
           "setup_brick.cu", "sweep_brick.cu", "kernels_brick.cu", "cg_mg.cu", "noalloc.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "--fmad=true",
              "-Xcompiler", "-fPIC,-O2,-Wall,-Wno-unused-function", "-cudart", "static"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _deps():
    out = [os.path.join(INC, "nanobte.h")]
    for f in os.listdir(CSRC):
        out.append(os.path.join(CSRC, f))
    return out


def build(force: bool = False, verbose: bool = False, defines=()) -> str:
    lib = LIB_PROF if defines else LIB
    stale = (not os.path.exists(lib)) or any(os.path.getmtime(p) > os.path.getmtime(lib) for p in _deps())
    if not (force or stale):
        return lib
    objdir = os.path.join(HERE, "build", "prof" if defines else "")
    os.makedirs(objdir, exist_ok=True)
    procs, objs = [], []
    for src in SOURCES:
        obj = os.path.join(objdir, src.replace(".cu", ".o"))
        objs.append(obj)
        cmd = [_nvcc(), *NVCC_FLAGS, *[f"-D{d}" for d in defines], "-I", INC, "-c", os.path.join(CSRC, src), "-o", obj]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        procs.append((src, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
    failed = False
    for src, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0 or verbose:
            sys.stderr.write(f"--- nvcc {src} ---\n{out}\n")
        failed |= p.returncode != 0
    if failed:
        raise RuntimeError("nvcc failed (see output above)")
    link = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-cudart", "static", "-o", lib, *objs]
    subprocess.run(link, check=True)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv,
                defines=[a[2:] for a in sys.argv[1:] if a.startswith("-D")]))
