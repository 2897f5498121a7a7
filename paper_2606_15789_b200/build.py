"""Build libanslin.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libanslin.so")
SOURCES = ["kernels.cu", "histogram.cu", "encode_gpu.cu", "host.cpp"]
HEADERS = ["anslin_internal.h", "decode_core.cuh", "fused_tmem.cuh", "decode_lanes.cuh", os.path.join("..", "..", "include", "anslin.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-shared",
              "-Xcompiler", "-fPIC,-O3,-pthread", "--use_fast_math", "-Xptxas", "-v"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        extra = os.environ.get("ANSLIN_NVCC_EXTRA", "").split()      # developer knob: e.g. -DANSLIN_J32=1
        cmd = [nvcc, *NVCC_FLAGS, *extra, *[os.path.join(CSRC, f) for f in SOURCES], "-o", LIB]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode != 0:
            print(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError("nvcc failed building libanslin.so")
    return LIB


if __name__ == "__main__":
    build(force=True, verbose=True)
