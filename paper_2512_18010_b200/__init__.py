"""paper_2512_18010_b200 — B200-native analytic molecular scattering form factors (arxiv 2512.18010, SCarFFF's
Cartesian method).  The product is the C-ABI library `libscarf.so` (include/scarf.h) built from `csrc/`;
`binding` is its ctypes front end, `build` the nvcc build step.  (The seeded synthetic input generator shared
with the oracle is the top-level module `workloads`, outside this package.)

`from paper_2512_18010_b200 import Scarf` loads the library and fails loudly if it has not been built.
"""
import importlib

__all__ = ["Scarf", "ScarfError", "build"]


def __getattr__(name):
    if name in ("Scarf", "ScarfError"):
        return getattr(importlib.import_module(__name__ + ".binding"), name)
    raise AttributeError(name)
