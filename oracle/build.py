"""Compile oracle/fe_oracle.c into oracle/libfe_oracle.so (gcc, no CUDA, no fast-math).

TEST INFRASTRUCTURE.  Flags: -O2 -ffp-contract=off (no FMA contraction: every operation
rounds as written), OpenMP for the Delta loop.  Rebuilds only when stale.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "fe_oracle.c")
LIB = os.path.join(HERE, "libfe_oracle.so")


def build(force: bool = False) -> str:
    fresh = lambda: os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC)     # noqa: E731
    if not force and fresh():
        return LIB
    import fcntl
    with open(os.path.join(HERE, ".build.lock"), "w") as lock:       # one builder at a time (parallel test workers, ranks)
        fcntl.flock(lock, fcntl.LOCK_EX)
        if not force and fresh():
            return LIB
        return _build_locked()


def _build_locked() -> str:
    cmd = ["gcc", "-std=c11", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC",
           "-shared", "-Wall", "-Wextra", "-o", LIB + ".tmp", SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
