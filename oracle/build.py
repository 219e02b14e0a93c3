"""Build the CPU oracle shared library (test infrastructure — see ls_oracle.c header).

    python -m oracle.build        # or: from oracle.build import build; build()

gcc only; no CUDA, no torch.  -ffp-contract=off keeps the compensated sums and error-free
transforms exactly as written (FMAs appear only where ls_oracle.c calls fma()).
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ls_oracle.c")
LIB = os.path.join(HERE, "libls_oracle.so")


def build(force: bool = False) -> str:
    import fcntl
    with open(os.path.join(HERE, ".build.lock"), "w") as lock:          # one builder at a time (torchrun ranks)
        fcntl.flock(lock, fcntl.LOCK_EX)
        try:
            return _build_locked(force)
        finally:
            fcntl.flock(lock, fcntl.LOCK_UN)


def _build_locked(force: bool) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-mfma", "-ffp-contract=off", "-fno-fast-math",
           "-Wall", "-Wextra", "-shared", "-fPIC", SRC, "-o", LIB + ".tmp", "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
