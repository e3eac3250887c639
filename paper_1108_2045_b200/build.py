"""Builds paper_1108_2045_b200/libhomg.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1108_2045_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libhomg.so")
SOURCES = ["homg_layout.cu", "homg_exec.cu", "homg_api.cu", "homg_noalloc.cu"]
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
# -fmad=false: the kernels evaluate exactly the expression trees DESIGN.md states (the same ones the
# oracle is compiled to with -ffp-contract=off), so fp64 AND fp32 results agree with it bit for bit;
# the path is HBM-bound, the extra multiply instructions are free.
FLAGS = ["-O3", "-std=c++17", "-lineinfo", "-fmad=false", "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def _deps():
    out = [os.path.join(CSRC, f) for f in os.listdir(CSRC)]
    out.append(os.path.join(os.path.dirname(HERE), "include", "homg.h"))
    out.append(os.path.abspath(__file__))
    return out


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(p) > t for p in _deps())


def build(force=False, verbose=False):
    if not force and not needs_build():
        return LIB
    cmd = [_nvcc()] + ARCH + FLAGS + (["-Xptxas", "-v"] if verbose else [])
    cmd += ["-shared", "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES] + ["-lcudart"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
