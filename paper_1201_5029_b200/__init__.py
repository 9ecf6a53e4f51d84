"""B200-native symplectic lattice stepper of PyCOOL (arXiv 1201.5029 §2.1-2.4).

`paper_1201_5029_b200.Lattice` is a thin binding (argument marshalling only) over the C-ABI library
`libpycool.so` declared in include/pycool.h; every step of the hot path runs in its sm_100a kernels.
`paper_1201_5029_b200.inputs` holds the seeded synthetic workloads.  The CUDA library is loaded on
first use and its absence is an error, never a fallback.
"""
from . import inputs  # noqa: F401


def __getattr__(name):  # lazy: importing the package (e.g. for `inputs`) must not need the CUDA library
    import importlib
    if name in ("binding", "build"):
        return importlib.import_module(__name__ + "." + name)
    if name in ("Lattice", "PycoolError", "lib", "stage_weights", "work_bytes", "from_config"):
        return getattr(importlib.import_module(__name__ + ".binding"), name)
    raise AttributeError(name)
