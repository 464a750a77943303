"""Builds paper_2107_08119_b200/libnep_b200.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "csrc", "nep_b200.cu")
# the allocation-free entry point keeps its static scratch, its set-up and its kernel in one translation unit of its own
SRC_NOALLOC = os.path.join(HERE, "csrc", "nep_noalloc.cu")
import glob
DEPS = sorted(glob.glob(os.path.join(HERE, "csrc", "*.cu*")) + glob.glob(os.path.join(HERE, "..", "include", "*.h")))
LIB = os.path.join(HERE, "libnep_b200.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC", "-diag-suppress", "177"]


def build(force: bool = False, verbose: bool = False) -> str:
    stale = (not os.path.exists(LIB)) or any(os.path.getmtime(LIB) < os.path.getmtime(d) for d in DEPS)
    if force or stale:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB, SRC, SRC_NOALLOC]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
