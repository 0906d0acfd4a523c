"""Compile the CETRA CUDA library in-tree for sm_100a (nvcc cross-compiles without a GPU).

    python -m paper_2503_20875_b200.build [--force]

Produces paper_2503_20875_b200/libcetra_b200.so, the C-ABI library declared in include/cetra.h.
"""
from __future__ import annotations

import os
import subprocess
import sys

_PKG = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_PKG)
CSRC = os.path.join(_PKG, "csrc")
INCLUDE = os.path.join(_ROOT, "include")
LIB_PATH = os.environ.get("CETRA_LIB_PATH") or os.path.join(_PKG, "libcetra_b200.so")
SOURCES = ["cetra_api.cu", "linear_search.cu", "periodic_search.cu", "fold_pair.cu", "fold_stream.cu", "setup_steps.cu", "peak_probe.cu", "tc_probe.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-shared", "-Xcompiler", "-fPIC", "--threads", "0",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def stale() -> bool:
    if not os.path.exists(LIB_PATH):
        return True
    built = os.path.getmtime(LIB_PATH)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(INCLUDE, "cetra.h")]
    return any(os.path.getmtime(d) > built for d in deps)


def have_nvcc() -> bool:
    import shutil
    n = _nvcc()
    return os.path.exists(n) if os.path.isabs(n) else shutil.which(n) is not None


def build(force: bool = False, verbose: bool = False) -> str:
    """Build libcetra_b200.so if it is missing or older than its sources; return its path."""
    if not (force or stale()):
        return LIB_PATH
    cmd = [_nvcc(), *NVCC_FLAGS, "-I", INCLUDE, "-I", CSRC] + os.environ.get("CETRA_NVCC_EXTRA", "").split()
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += [os.path.join(CSRC, s) for s in SOURCES] + ["-o", LIB_PATH]
    subprocess.run(cmd, check=True)
    return LIB_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
