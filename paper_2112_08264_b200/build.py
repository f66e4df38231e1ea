"""Build the C-ABI CUDA library in-tree (sm_100a only).

    python -m paper_2112_08264_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so lands in paper_2112_08264_b200/_lib/, is
git-ignored, and travels to the GPU box with the gpurun snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB_DIR = os.path.join(_HERE, "_lib")
LIB_PATH = os.path.join(LIB_DIR, "liblb_b200.so")
SOURCES = [os.path.join(CSRC, "lb_b200.cu"), os.path.join(CSRC, "lb_single.cu")]
NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-shared", "--fmad=true",
]


def _deps():
    out = [os.path.join(_HERE, "..", "include", "lb.h")]
    for name in os.listdir(CSRC):
        if name.endswith((".cu", ".cuh", ".h")):
            out.append(os.path.join(CSRC, name))
    return out


def build_lib(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB_PATH):
        newest = max(os.path.getmtime(p) for p in _deps())
        if os.path.getmtime(LIB_PATH) >= newest:
            return LIB_PATH
    os.makedirs(LIB_DIR, exist_ok=True)
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = LIB_PATH + f".tmp{os.getpid()}"
    cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", tmp, *SOURCES]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB_PATH)
    return LIB_PATH


if __name__ == "__main__":
    print(build_lib(force="--force" in sys.argv, verbose="-v" in sys.argv))
