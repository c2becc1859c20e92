"""Build libtpctrk.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo snapshot)."""
from __future__ import annotations

import os
import subprocess

_PKG = os.path.dirname(os.path.abspath(__file__))
_ROOT = os.path.dirname(_PKG)
CSRC = os.path.join(_PKG, "csrc")
LIB = os.path.join(_PKG, "libtpctrk.so")
SOURCES = [os.path.join(CSRC, "tpctrk.cu")]
HEADERS = [os.path.join(CSRC, f) for f in ("device_types.cuh", "kernels_ca.cuh", "kernels_kf.cuh", "kernels_merge.cuh")] + [
    os.path.join(_ROOT, "include", "tpctrk.h")]

# -fmad=false: no FMA contraction, so every fp32 decision value equals the written IEEE expression
# (R-12); division/sqrt stay IEEE (nvcc defaults, never --use_fast_math).
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-fmad=false",
              "--expt-extended-lambda", "-Xcompiler", "-fPIC", "-shared", "-I", os.path.join(_ROOT, "include"),
              "-I", CSRC]


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        extra = os.environ.get("TPCTRK_NVCC_EXTRA", "").split()     # tuning builds, e.g. -DTPC_K5_FUSE_K6A=0
        cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB] + SOURCES
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
