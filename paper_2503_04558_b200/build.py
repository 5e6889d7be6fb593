"""Build libgrpic.so (hand-written CUDA for sm_100a) in-tree with nvcc.

    python -m paper_2503_04558_b200.build [--force] [--verbose]

The shared library is written next to this file so that it travels with the repository
snapshot to the GPU box; nothing is installed into site-packages and no JIT cache is used.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgrpic.so")
SOURCES = ["api.cu", "push_deposit.cu", "field.cu", "current.cu", "sort.cu", "host_step.cu", "pair.cu", "push_spline3.cu", "diagnostics.cu"]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "--use_fast_math=false"]


def _nvcc():
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    raise RuntimeError("nvcc not found")


def build(force=False, verbose=False):
    srcs = [os.path.join(CSRC, s) for s in SOURCES]
    deps = srcs + [os.path.join(CSRC, "grpic_internal.cuh"), os.path.join(CSRC, "push_math.cuh"), os.path.join(CSRC, "poly_tables.cuh"),
                   os.path.join(HERE, "..", "include", "grpic.h")]
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in deps):
        return LIB
    flags = [f for f in NVCC_FLAGS if f != "--use_fast_math=false"]
    flags += os.environ.get("GRPIC_NVCC_EXTRA", "").split()
    if verbose:
        flags += ["-Xptxas", "-v"]
    cmd = [_nvcc()] + flags + ["-shared", "-o", LIB] + srcs
    if verbose:
        print(" ".join(cmd))
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
