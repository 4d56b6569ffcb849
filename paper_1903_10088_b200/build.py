"""Build libosiv.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1903_10088_b200.build [--force]

nvcc cross-compiles without a GPU, so this runs on the CPU box too; the resulting
``paper_1903_10088_b200/libosiv.so`` is git-ignored and travels to the GPU box with the snapshot.
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")
SO = os.path.join(_HERE, "libosiv.so")
SOURCES = [os.path.join(CSRC, "osiv.cu"), os.path.join(CSRC, "osiv_probes.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "osiv_kernels.cuh"), os.path.join(CSRC, "osiv_back_staged.cuh"), os.path.join(INCLUDE, "osiv.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a",
              "-shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v"]


def nvcc_path() -> str:
    p = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(p):
        raise RuntimeError("nvcc not found: libosiv.so cannot be built (there is no CPU fallback)")
    return p


def needs_build() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    return any(os.path.getmtime(d) > t for d in DEPS)


SO_TRACE = os.path.join(_HERE, "libosiv_trace.so")      # the same sources with -DOSIV_TRACE (phase timeline, diagnostics)


def _stale(so: str) -> bool:
    if not os.path.exists(so):
        return True
    t = os.path.getmtime(so)
    return any(os.path.getmtime(d) > t for d in DEPS)


SO_CHECK = os.path.join(_HERE, "libosiv_check.so")      # the same sources with -DOSIV_CHECKED (index checks, diagnostics)


def build(force: bool = False, verbose: bool = False, trace: bool = False, check: bool = False) -> str:
    so = SO_TRACE if trace else SO_CHECK if check else SO
    if force or _stale(so):
        cmd = [nvcc_path()] + NVCC_FLAGS + (["-DOSIV_TRACE"] if trace else ["-DOSIV_CHECKED"] if check else []) + ["-I", INCLUDE, "-o", so] + SOURCES
        res = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or res.returncode != 0:
            sys.stderr.write(res.stdout + res.stderr)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed building " + os.path.basename(so))
    return so


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True, trace="--trace" in sys.argv, check="--check" in sys.argv))
