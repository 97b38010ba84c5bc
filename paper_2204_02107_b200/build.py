"""Builds libdnslab.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "csrc", "dnslab.cu")
DEPS = [SRC, os.path.join(HERE, "csrc", "fft.cuh"), os.path.join(HERE, "csrc", "stencil.cuh"), os.path.join(HERE, "csrc", "reduce.cuh"), os.path.join(HERE, "csrc", "particles.cuh"), os.path.join(HERE, "csrc", "tma.cuh"),
        os.path.join(os.path.dirname(HERE), "include", "dnslab.h")]
LIB = os.path.join(HERE, "libdnslab.so")
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-shared", "-Xcompiler", "-fPIC"]


def build(force=False, verbose=False):
    stale = not os.path.exists(LIB) or any(os.path.getmtime(d) > os.path.getmtime(LIB) for d in DEPS)
    if force or stale:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB, SRC]
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
