"""paper_1410_4194_b200 — B200-native CTU + PPMC + exact-Riemann hydro step (arXiv:1410.4194).

`Grid` (binding.py) is the thin Python binding over the C-ABI library declared in include/ch.h
and implemented in csrc/ (hand-written CUDA for sm_100a).  `workloads` holds the seeded synthetic
inputs.  Importing the package does not load the CUDA library; constructing a `Grid` does, and
fails loudly if the library is missing or no GPU is present.  There is no CPU fallback.
"""
from . import workloads  # noqa: F401

__all__ = ["workloads", "Grid", "load_library", "build"]


def __getattr__(name):
    if name in ("Grid", "load_library", "build", "PERIODIC", "REFLECTIVE", "OUTFLOW", "NOH"):
        from . import binding
        return getattr(binding, name)
    raise AttributeError(name)
