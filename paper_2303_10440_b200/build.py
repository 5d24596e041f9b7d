"""Build libdeltamic.so (the C-ABI library of include/deltamic.h) in-tree with nvcc for sm_100a.

    python -m paper_2303_10440_b200.build [--force]

nvcc cross-compiles without a GPU.  The CUDA runtime is linked statically; cuFFT (the inverse-FFT stage, a library
call by design) is the toolkit's shared libcufft.so.11 (a static cuFFT would make the library 250 MB).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libdeltamic.so")
SOURCES = ["deltamic.cu"]
HEADERS = ["dm_math.cuh", "dm_kernels.cuh", "dm_fast.cuh", "dm_bwd_fast.cuh", "dm_strips.h", "dm_patches.h", "dm_splits.h", "dm_shape.cuh", os.path.join("..", "..", "include", "deltamic.h")]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
    "-Xcompiler", "-fPIC,-O2,-Wall", "-shared", "--cudart=static",
]
LINK = ["-lcufft", "-Xlinker", "-rpath=/usr/local/cuda/lib64", "-lpthread", "-ldl", "-lrt"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.exists(d) and os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False, extra=()) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + list(extra) + ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES] + \
          ["-L/usr/local/cuda/lib64"] + LINK
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
    r = subprocess.run(cmd, capture_output=True, text=True)
    if verbose:
        sys.stderr.write(r.stdout + r.stderr)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + " ".join(cmd) + "\n" + r.stdout + r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
