"""Builds the CUDA library in-tree: paper_2512_12466_b200/libnyxrt.so (sm_100a only).

-fmad=false: decision arithmetic (DESIGN.md DEC) must not be contracted; fma() is written where wanted.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "csrc", "nyxrt.cu")
SRC_STATIC = os.path.join(HERE, "csrc", "finalise_static.cu")      # nyxrt_finalise_static: its own translation unit
DEPS = [os.path.join(HERE, "csrc", f) for f in ("nyxrt.cu", "finalise_static.cu", "march.cuh", "sources.cuh", "timestep.cuh", "healpix.cuh", "state.cuh")]
DEPS.append(os.path.join(os.path.dirname(HERE), "include", "nyxrt.h"))
LIB = os.path.join(HERE, "libnyxrt.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-fmad=false",
         "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def stale():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force=False, verbose=False):
    if not force and not stale():
        return LIB
    tmp = LIB + ".%d.tmp" % os.getpid()
    cmd = [NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp, SRC, SRC_STATIC]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
