"""Builds libphylino.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_2502_15253_b200.build [--force] [--verbose] [--checked]

The library links the CUDA runtime statically and has no Python or torch dependency.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_HERE)
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(_ROOT, "include")
LIB = os.path.join(_HERE, "libphylino.so")
SOURCES = ["api.cu", "spectra.cu", "finalize.cu", "transform.cu", "consumers.cu", "peaks.cu", "static_step.cu"]
HEADERS = ["internal.h", "devmath.cuh", "finalize.cuh", os.path.join(INCLUDE, "phylino.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-fmad=false",              # nothing is contracted behind our back; every fma() is explicit (R8)
    "-Xcompiler", "-fPIC,-O2,-fvisibility=hidden",
    "-shared", "-cudart", "static",
    "-Xptxas", "-v",
]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found: the CUDA path cannot be built (there is no CPU fallback)")
    return exe


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + [h if os.path.isabs(h) else os.path.join(CSRC, h) for h in HEADERS]
    deps.append(os.path.abspath(__file__))
    return any(os.path.getmtime(d) > t for d in deps)


LIB_CHECKED = os.path.join(_HERE, "libphylino_checked.so")


def build(force: bool = False, verbose: bool = False, checked: bool = False) -> str:
    """checked: the same sources with -DPHYLINO_CHECKED (device-side bounds / invariant checks that trap) into
    libphylino_checked.so; load it with PHYLINO_LIBRARY=<path> (binding.py).  Never the shipped library."""
    lib = LIB_CHECKED if checked else LIB
    if not checked and not (force or _stale()):
        return LIB
    tmp = lib + f".tmp{os.getpid()}"
    cmd = [nvcc(), *NVCC_FLAGS, *(["-DPHYLINO_CHECKED"] if checked else []), "-I", INCLUDE, "-I", CSRC,
           *[os.path.join(CSRC, s) for s in SOURCES], "-o", tmp]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed building libphylino.so")
    if verbose:
        sys.stderr.write(res.stderr)
    if not checked:
        with open(os.path.join(_HERE, "ptxas_info.log"), "w") as f:
            f.write(" ".join(cmd) + "\n" + res.stdout + res.stderr)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, checked="--checked" in sys.argv))
