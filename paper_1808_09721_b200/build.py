"""Build librmhd.so (the C-ABI CUDA library, include/rmhd.h) in-tree for sm_100a.

    python -m paper_1808_09721_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU; the .so travels to the GPU box with the repo snapshot.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.environ.get("RMHD_LIB") or os.path.join(HERE, "librmhd.so")   # RMHD_LIB: build (and, binding.py, load) another copy, e.g. a measurement build
SOURCES = [os.path.join(CSRC, "rmhd.cu")]
HEADERS = [os.path.join(CSRC, f) for f in ("physics.cuh", "stage.cuh", "kernels.cuh", "flux_fused.cuh", "flux_hm.cuh")] + [os.path.join(ROOT, "include", "rmhd.h")]


def _stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in SOURCES + HEADERS if os.path.exists(f))


def build(force=False, verbose=False):
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-std=c++17", "-O3", "-lineinfo", "-gencode", "arch=compute_100a,code=sm_100a",
           "-shared", "-Xcompiler", "-fPIC", "-I", os.path.join(ROOT, "include"), "-o", LIB] + SOURCES
    if verbose:
        cmd += ["-Xptxas", "-v"]
    cmd += os.environ.get("RMHD_NVCC_FLAGS", "").split()
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
