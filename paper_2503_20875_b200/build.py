"""Compile the CETRA CUDA library in-tree for sm_100a (nvcc cross-compiles without a GPU).

    python -m paper_2503_20875_b200.build [--force]

Produces paper_2503_20875_b200/libcetra_b200.so, the C-ABI library declared in include/cetra.h, and
libcetra_diag.so, the measurement probes of include/cetra_diag.h that bench.py loads.
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
SOURCES = ["cetra_api.cu", "linear_search.cu", "periodic_search.cu", "fold_pair.cu", "fold_stream.cu", "setup_steps.cu"]
# measurement probes (include/cetra_diag.h): a library of their own that only bench.py loads
DIAG_LIB_PATH = os.path.join(_PKG, "libcetra_diag.so")
DIAG_SOURCES = ["peak_probe.cu", "tc_probe.cu"]
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-shared", "-Xcompiler", "-fPIC", "--threads", "0",
]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def stale(lib_path: str = "") -> bool:
    lib_path = lib_path or LIB_PATH
    if not os.path.exists(lib_path):
        return True
    built = os.path.getmtime(lib_path)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(INCLUDE, f) for f in os.listdir(INCLUDE)]
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


def build_diag(force: bool = False) -> str:
    """Build libcetra_diag.so (the probes of include/cetra_diag.h) if it is missing or older than its sources."""
    if not (force or stale(DIAG_LIB_PATH)):
        return DIAG_LIB_PATH
    cmd = [_nvcc(), *NVCC_FLAGS, "-I", INCLUDE, "-I", CSRC]
    cmd += [os.path.join(CSRC, s) for s in DIAG_SOURCES] + ["-o", DIAG_LIB_PATH]
    subprocess.run(cmd, check=True)
    return DIAG_LIB_PATH


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    print(build_diag(force="--force" in sys.argv))
