"""Build paper_2512_18010_b200/libscarf.so (the C-ABI library of include/scarf.h) for sm_100a with nvcc.

    python -m paper_2512_18010_b200.build [--force] [--verbose]

The library is built IN-TREE so that it travels to the GPU box with the repo snapshot.  nvcc cross-compiles
without a GPU.  cudart is linked statically, so the .so also loads (and its host-only entry points run) on a
machine with no CUDA driver.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libscarf.so")
SOURCES = ["host_setup.cpp", "fold.cu", "ff_v1.cu", "ff_grid.cu", "ff_row.cu", "ff_zrow.cu", "ff_sph.cu", "ff_highl.cu", "angular.cu", "pure.cu", "fft_method.cu", "scarf_api.cu"]
HEADERS = ["host_setup.hpp", "kernels.cuh", "ff_common.cuh", "ff_math.cuh", "math_coeffs.cuh", os.path.join("..", "..", "include", "scarf.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC,-O3,-fopenmp", "--expt-relaxed-constexpr"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.exists(d) and os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, ptxas_verbose: bool = False, debug_checks: bool = False) -> str:
    """debug_checks: compile the device-side invariant checks (SCARF_CHECK, ff_common.cuh) in; the library is written to
    libscarf.so all the same (rebuild without the flag afterwards)."""
    if not force and not debug_checks and not _stale():
        return LIB
    objs = []
    build_dir = os.path.join(HERE, "build")
    os.makedirs(build_dir, exist_ok=True)
    procs = []
    for s in SOURCES:
        src = os.path.join(CSRC, s)
        if not os.path.exists(src):
            continue
        obj = os.path.join(build_dir, os.path.splitext(s)[0] + ".o")
        cmd = ([_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if ptxas_verbose else []) + (["-DSCARF_DEBUG_CHECKS"] if debug_checks else [])
               + ["-c", src, "-o", obj])
        if verbose:
            print(" ".join(cmd), file=sys.stderr)
        procs.append((cmd, subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)))
        objs.append(obj)
    failed = False
    for cmd, p in procs:
        out, _ = p.communicate()
        if p.returncode != 0:
            failed = True
            sys.stderr.write(out)
        elif verbose or ptxas_verbose:
            sys.stderr.write(out)
    if failed:
        raise RuntimeError("nvcc failed")
    cmd = [_nvcc(), "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB] + objs + ["-Xcompiler", "-fopenmp", "-ldl"]
    if verbose:
        print(" ".join(cmd), file=sys.stderr)
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv or "-v" in sys.argv,
                ptxas_verbose="--ptxas" in sys.argv, debug_checks="--debug-checks" in sys.argv))
