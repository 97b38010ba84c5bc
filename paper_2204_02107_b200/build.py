"""Builds libdnslab.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "csrc", "dnslab.cu")
DEPS = [SRC, os.path.join(HERE, "csrc", "fft.cuh"), os.path.join(HERE, "csrc", "stencil.cuh"), os.path.join(HERE, "csrc", "reduce.cuh"), os.path.join(HERE, "csrc", "particles.cuh"), os.path.join(HERE, "csrc", "tma.cuh"),
        os.path.join(os.path.dirname(HERE), "include", "dnslab.h")]
LIB = os.path.join(HERE, "libdnslab.so")
# Test-only variant: the same sources with -DDNSLAB_TEST_NO_TMA, in which dnslab_create never obtains the tensor-map
# encoder, so the library runs the paths it falls back to when TMA descriptors cannot be built (cp.async tiles in the RK
# kernel, the five-pass solve, the cp.async z pass).  Loaded only by tests/test_parity_gpu.py; not the product.
LIB_NOTMA = os.path.join(HERE, "libdnslab_notma.so")
NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-shared", "-Xcompiler", "-fPIC"]


def _build(lib, defines, force, verbose):
    stale = not os.path.exists(lib) or any(os.path.getmtime(d) > os.path.getmtime(lib) for d in DEPS)
    if force or stale:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + defines + (["-Xptxas", "-v"] if verbose else []) + ["-o", lib, SRC]
        subprocess.check_call(cmd)
    return lib


def build(force=False, verbose=False):
    return _build(LIB, [], force, verbose)


def build_notma(force=False):
    return _build(LIB_NOTMA, ["-DDNSLAB_TEST_NO_TMA"], force, False)


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
    if "--notma" in sys.argv:
        print(build_notma(force="--force" in sys.argv))
