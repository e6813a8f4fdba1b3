"""Build paper_1412_8754_b200/libfe.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1412_8754_b200.build [--force] [--libdevice-math]

The library is a plain C-ABI shared object (include/fe.h); cudart is linked statically so that it loads
(and its symbols can be checked) on a machine without a GPU or driver.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libfe.so")
SOURCES = [os.path.join(CSRC, "fe_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, "fe_kernels.cuh"), os.path.join(CSRC, "fe_ksum_coop.cuh"), os.path.join(CSRC, "fe_math.cuh"),
                  os.path.join(ROOT, "include", "fe.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--fmad=true", "-Xcompiler", "-fPIC", "-shared", "--cudart", "static",
              "-Xptxas", "-v", "-Wno-deprecated-gpu-targets"]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, extra=(), verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc] + NVCC_FLAGS + list(extra) + ["-o", LIB + ".tmp"] + SOURCES
    r = subprocess.run(cmd, capture_output=True, text=True)
    log = r.stdout + r.stderr
    with open(os.path.join(HERE, "build_ptxas.log"), "w") as f:
        f.write(" ".join(cmd) + "\n" + log)
    if r.returncode != 0:
        errs = [l for l in log.splitlines() if "error" in l.lower()]
        sys.stderr.write("\n".join(errs[:20]) + "\n(full log: paper_1412_8754_b200/build_ptxas.log)\n")
        raise RuntimeError("nvcc failed")
    if verbose:
        print(log)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    extra = ["-DFE_MATH_LIBDEVICE"] if "--libdevice-math" in sys.argv else []
    print(build(force=True, extra=extra, verbose="-v" in sys.argv))
