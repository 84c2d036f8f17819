"""Build libkharm.so (the CUDA product) in-tree for sm_100a with nvcc.

    python -m paper_2408_01361_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with gpurun.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
SRC = os.path.join(HERE, "csrc", "kharm.cu")
SRC_NOALLOC = os.path.join(HERE, "csrc", "kh_noalloc.cu")      # kh_divB_noalloc: a translation unit of its own (static scratch)
DEPS = [SRC, SRC_NOALLOC] + [os.path.join(HERE, "csrc", f) for f in ("kh_device.cuh", "kh_geometry.cuh", "kh_kernels.cuh")] + \
       [os.path.join(ROOT, "include", "kharm.h")]
OUT = os.path.join(HERE, "libkharm.so")

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared", "-diag-suppress", "68"]


def build(force=False, verbose=False):
    if not force and os.path.exists(OUT) and all(os.path.getmtime(d) <= os.path.getmtime(OUT) for d in DEPS):
        return OUT
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", OUT, SRC, SRC_NOALLOC]
    if verbose:
        print(" ".join(cmd))
    subprocess.check_call(cmd)
    return OUT


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
