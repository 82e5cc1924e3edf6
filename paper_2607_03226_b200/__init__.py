"""B200-native NanoBTE hot path (arxiv/paper_2607_03226): C-ABI CUDA library + thin binding.

`workloads`  seeded synthetic problem generators (inputs only; shared with the oracle's tests)
`binding`    ctypes binding of libnanobte.so (Solver, workspace_bytes, load)
`build`      nvcc build of the library, in-tree
"""
from . import workloads  # noqa: F401


def __getattr__(name):  # lazy: importing the package must not need the built library
    if name in ("Solver", "NanoBTEError", "workspace_bytes", "load"):
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)
