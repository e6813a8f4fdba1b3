"""Build paper_1412_8754_b200/libfe.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1412_8754_b200.build [--force] [--libdevice-math] [-v]

The library is a plain C-ABI shared object (include/fe.h); cudart is linked statically so that it loads
(and its symbols can be checked) on a machine without a GPU or driver.

The k-sum kernels are template families (tile / block shape x bands x form factor x mode), so they are split
over translation units that compile in parallel: fe_api.cu (C ABI, small kernels), fe_launch_tile.cu once per
register tile of K1 / K1f and fe_launch_coop.cu once per block shape of K1c; objects go to _obj/ (git-ignored).
TILES and COOP_SHAPES must list the same entries, in the same order, as kTiles / kCoopShapes in fe_api.cu.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "_obj")
LIB = os.path.join(HERE, "libfe.so")
LOG = os.path.join(HERE, "build_ptxas.log")

TILES = [(8, 4), (4, 4), (2, 8), (1, 8), (16, 2), (16, 4)]
COOP_SHAPES = [(16, 4, 4, 4, 4, 2), (16, 4, 1, 4, 2, 2), (8, 4, 4, 4, 4, 3), (8, 4, 1, 4, 2, 2), (16, 4, 2, 4, 2, 2), (16, 4, 4, 4, 2, 2)]

HEADERS = [os.path.join(CSRC, f) for f in ("fe_kernels.cuh", "fe_ksum_coop.cuh",  "fe_bands3.cuh", "fe_chi.cuh", "fe_ksum_sp.cuh", "fe_math.cuh",
                                           "fe_launch.h")] + [os.path.join(ROOT, "include", "fe.h"), os.path.join(ROOT, "include", "fe_debug.h")]
SOURCES = [os.path.join(CSRC, f) for f in ("fe_api.cu", "fe_launch_tile.cu", "fe_launch_coop.cu")]
DEPS = SOURCES + HEADERS + [os.path.abspath(__file__)]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--fmad=true", "-Xcompiler", "-fPIC", "-Xptxas", "-v", "-Wno-deprecated-gpu-targets"]


def source_hash() -> str:
    """sha256 (first 16 hex digits) of the kernel sources as compiled: every file of csrc/ and include/, comments and
    white space removed, so that only a change of code changes it.  bench.py compares it with the hash recorded beside
    each committed ncu capture (profiles/COUNTS.md) before it uses that capture's instruction counts, and with the hash
    compiled into libfe.so (fe_build_source_hash) before it trusts the library to be built from these sources."""
    import hashlib
    import re
    files = sorted([os.path.join(CSRC, f) for f in os.listdir(CSRC)] +
                   [os.path.join(ROOT, "include", f) for f in os.listdir(os.path.join(ROOT, "include"))])
    hsh = hashlib.sha256()
    for f in files:
        if not f.endswith((".cu", ".cuh", ".h")):
            continue
        text = open(f).read()
        text = re.sub(r"/\*.*?\*/", " ", text, flags=re.S)
        text = re.sub(r"//[^\n]*", " ", text)
        text = " ".join(text.split())
        hsh.update(os.path.basename(f).encode() + b"\0" + text.encode() + b"\0")
    return hsh.hexdigest()[:16]


def units():
    """[(object name, source, extra -D flags)]"""
    u = [("fe_api.o", "fe_api.cu", [f'-DFE_SOURCE_HASH="{source_hash()}"'])]
    for i, (th, td) in enumerate(TILES):
        u.append((f"fe_tile{i}.o", "fe_launch_tile.cu", [f"-DFE_TILE_ID={i}", f"-DFE_TILE_TH={th}", f"-DFE_TILE_TD={td}"]))
    for i, s in enumerate(COOP_SHAPES):
        u.append((f"fe_coop{i}.o", "fe_launch_coop.cu", [f"-DFE_COOP_ID={i}"] + [f"-DFE_COOP_{n}={v}" for n, v in zip(("TH", "TD", "LH", "NW", "KB", "MINB"), s)]))
    return u


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False, extra=(), verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    # one builder at a time: several ranks of a multi-GPU launch may find the library stale at once
    import fcntl
    with open(os.path.join(HERE, ".build.lock"), "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        if not force and not stale():
            return LIB                       # another process built it while this one waited
        return _build_locked(extra, verbose)


def _build_locked(extra, verbose) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)

    def compile_one(unit):
        obj, src, defs = unit
        cmd = [nvcc] + NVCC_FLAGS + list(extra) + defs + ["-c", "-o", os.path.join(OBJ, obj), os.path.join(CSRC, src)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        return unit, cmd, r

    # heaviest units first so that the pool stays busy
    order = sorted(units(), key=lambda u: (not u[0].startswith("fe_coop"), u[0]))
    with ThreadPoolExecutor(max_workers=min(len(order), os.cpu_count() or 4)) as pool:
        results = list(pool.map(compile_one, order))
    log, failed = [], False
    for (obj, _, _), cmd, r in results:
        log.append(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        failed |= r.returncode != 0
    if not failed:
        cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "--cudart", "static",
               "-Wno-deprecated-gpu-targets", "-o", LIB + ".tmp"] + [os.path.join(OBJ, u[0]) for u in units()]
        r = subprocess.run(cmd, capture_output=True, text=True)
        log.append(" ".join(cmd) + "\n" + r.stdout + r.stderr)
        failed |= r.returncode != 0
    text = "\n".join(log)
    with open(LOG, "w") as f:
        f.write(text)
    if failed:
        errs = [l for l in text.splitlines() if "error" in l.lower()]
        sys.stderr.write("\n".join(errs[:20]) + "\n(full log: paper_1412_8754_b200/build_ptxas.log)\n")
        raise RuntimeError("nvcc failed")
    if verbose:
        print(text)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    extra = ["-DFE_MATH_LIBDEVICE"] if "--libdevice-math" in sys.argv else []
    print(build(force=True, extra=extra, verbose="-v" in sys.argv))
