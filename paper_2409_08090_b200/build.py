"""Build libls_b200.so (the C-ABI library of include/ls.h) for sm_100a, in-tree.

    python -m paper_2409_08090_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with gpurun.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libls_b200.so")
SOURCES = ["ls_api.cu", "ls_pre.cu", "ls_spread.cu", "ls_fft.cu", "ls_fft_f32.cu", "ls_post.cu", "ls_direct.cu"]
HEADERS = [os.path.join(CSRC, "ls_internal.h"), os.path.join(CSRC, "ls_power.cuh"), os.path.join(HERE, "..", "include", "ls.h")]
CUDA_HOME = os.environ.get("CUDA_HOME", "/usr/local/cuda")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC,-Wall,-Wno-unused-function", "--fmad=true"]


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    mt = os.path.getmtime(target)
    return any(os.path.getmtime(d) > mt for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile what is stale.  Serialised across processes by a file lock: under torchrun every rank calls
    this, and concurrent nvcc runs must not write the same objects."""
    import fcntl
    with open(os.path.join(HERE, ".build.lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            return _build_locked(force, verbose)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)


def _build_locked(force: bool, verbose: bool) -> str:
    nvcc = os.path.join(CUDA_HOME, "bin", "nvcc")
    objs = []
    for src in SOURCES:
        sp = os.path.join(CSRC, src)
        op = os.path.join(CSRC, src.replace(".cu", ".o"))
        objs.append(op)
        if force or _stale(op, [sp] + HEADERS):
            cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", sp, "-o", op]
            subprocess.run(cmd, check=True)
    if force or _stale(LIB, objs):
        cmd = [nvcc, "-shared", "-o", LIB + ".tmp"] + objs + [
            "-L" + os.path.join(CUDA_HOME, "lib64"), "-lcufft", "-lcudart",
            "-Xlinker", "-rpath," + os.path.join(CUDA_HOME, "lib64")]
        subprocess.run(cmd, check=True)
        os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
