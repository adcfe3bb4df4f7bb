"""Build libhigs.so (the C-ABI library of include/higs.h) in-tree with nvcc for sm_100a.

    python -m paper_2606_00352_b200.build [--force] [--verbose]

The library is plain CUDA C++ (no torch headers); it is rebuilt when any source is newer than
the .so.  nvcc cross-compiles without a GPU, so this also runs on the CPU-only box.
"""
from __future__ import annotations

import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "lib" / "libhigs.so"
SOURCES = ["api.cu", "project.cu", "binning.cu", "sort.cu", "raster.cu", "shcodec.cu", "scene.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "--extended-lambda", "-Xcompiler", "-fPIC", "-shared"]


def _deps():
    return [CSRC / s for s in SOURCES] + sorted(CSRC.glob("*.cuh")) + [PKG.parent / "include" / "higs.h"]


def stale() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any(p.stat().st_mtime > t for p in _deps())


def build(force: bool = False, verbose: bool = False, debug_bounds: bool = False) -> Path:
    """debug_bounds: compile with -DHIGS_DEBUG_BOUNDS (device asserts on the frame's indexed writes, higs_internal.cuh)."""
    if not force and not stale() and not debug_bounds:
        return LIB
    LIB.parent.mkdir(parents=True, exist_ok=True)
    cmd = ["nvcc", *NVCC_FLAGS, *(["-DHIGS_DEBUG_BOUNDS"] if debug_bounds else []), *(["-Xptxas", "-v"] if verbose else []), "-o", str(LIB), *[str(CSRC / s) for s in SOURCES]]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libhigs.so")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, debug_bounds="--debug-bounds" in sys.argv))
