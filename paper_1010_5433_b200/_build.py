"""Build libstag_b200.so in-tree with nvcc for sm_100a (no JIT cache, no torch extension).

    python -m paper_1010_5433_b200._build [--force]
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libstag_b200.so")
SO_TIMERS = os.path.join(HERE, "libstag_b200_timers.so")     # -DSTAG_PHASE_TIMERS build (STAG_PHASE_TIMERS=1)
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC"]
OBJ = os.path.join(HERE, "build")


def sources() -> list[str]:
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps() -> list[str]:
    inc = os.path.join(os.path.dirname(HERE), "include", "stag.h")
    return sources() + glob.glob(os.path.join(CSRC, "*.cuh")) + [inc]


def stale() -> bool:
    if not os.path.exists(SO):
        return True
    t = os.path.getmtime(SO)
    return any(os.path.getmtime(f) > t for f in _deps())


def build(force: bool = False, verbose: bool = False, timers: bool = False) -> str:
    """timers=True: the per-phase-timer build of the persistent CG (csrc/stag_cg_persist.cuh), a separate .so."""
    if timers:
        return _build(SO_TIMERS, ["-DSTAG_PHASE_TIMERS=" + os.environ.get("STAG_PHASE_TIMERS", "1")], verbose)
    if not force and not stale():
        return SO
    return _build(SO, [], verbose)


def _build(SO: str, defines: list[str], verbose: bool) -> str:
    from concurrent.futures import ThreadPoolExecutor
    nvcc = os.environ.get("NVCC", "nvcc")
    os.makedirs(OBJ, exist_ok=True)
    extra = (["-Xptxas", "-v"] if verbose else []) + defines

    def compile_one(src: str) -> str:          # one translation unit per worker: seconds, not a minute
        obj = os.path.join(OBJ, os.path.basename(src)[:-3] + ".%d.o" % os.getpid())
        subprocess.check_call([nvcc] + NVCC_FLAGS + extra + ["-c", "-o", obj, src])
        return obj

    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 1)) as pool:
        objs = list(pool.map(compile_one, sources()))
    tmp = SO + ".tmp.%d" % os.getpid()
    subprocess.check_call([nvcc] + NVCC_FLAGS[:2] + ["-shared", "-o", tmp] + objs)
    os.replace(tmp, SO)
    for o in objs:
        os.unlink(o)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv,
                timers=os.environ.get("STAG_PHASE_TIMERS") in ("1", "2")))
