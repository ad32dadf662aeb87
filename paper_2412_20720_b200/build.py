"""Builds libfdgs.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfdgs.so")
SOURCES = ["api.cu", "features.cu", "preprocess.cu", "preprocess_bwd.cu", "scan_dup.cu", "radix_sort.cu", "blend.cu", "train.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
              "--use_fast_math=false"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh"))] + [os.path.join(HERE, "..", "include", "fdgs.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    flags = [f for f in NVCC_FLAGS if not f.startswith("--use_fast_math")]
    flags += os.environ.get("FDGS_NVCC_EXTRA", "").split()      # measurement builds only, e.g. -DFDGS_BLEND_ASYNC=0 (profiles/)
    cmd = [nvcc, *flags, "-shared", "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd))
    subprocess.run(cmd, check=True)
    return LIB


CMP_LIB = os.path.join(HERE, "libfdgs_cubcmp.so")


def build_compare(force: bool = False) -> str:
    """The CUB comparison sort (csrc/compare/): a separate library, used only by `sweep --sort-compare`."""
    src = os.path.join(CSRC, "compare", "cub_sort_compare.cu")
    if force or not os.path.exists(CMP_LIB) or os.path.getmtime(CMP_LIB) < os.path.getmtime(src):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        flags = [f for f in NVCC_FLAGS if not f.startswith("--use_fast_math")]
        subprocess.run([nvcc, *flags, "-shared", "-o", CMP_LIB, src], check=True)
    return CMP_LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose="-v" in sys.argv)
    build_compare(force="--force" in sys.argv)
    print(LIB)
