"""Build step: compile csrc/greenlantern_b200.cu for sm_100a into csrc/libgreenlantern_b200.so.

``python -m paper_2410_05408_b200.build`` (or ``__graft_entry__.build()``).  nvcc cross-compiles
without a GPU.  The library is kept in-tree so that it travels with the source snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

CSRC = Path(__file__).resolve().parent / "csrc"
LIB = CSRC / "libgreenlantern_b200.so"
SOURCES = [CSRC / "greenlantern_b200.cu"]
DEPENDS = SOURCES + [CSRC / "gl_core.cuh", CSRC / "gl_tables.h", CSRC / "gl_fast32.cuh", CSRC / "gl_hot.cuh", CSRC / "gl_simpson.cuh", CSRC / "gl_frontend.cuh", CSRC / "gl_gp.cuh", CSRC / "gl_gp_scan.cuh",
                     CSRC.parents[1] / "include" / "greenlantern_b200.h"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def up_to_date() -> bool:
    return LIB.exists() and all(LIB.stat().st_mtime >= d.stat().st_mtime for d in DEPENDS)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and up_to_date():
        return LIB
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    cmd = [_nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", str(tmp),
           *map(str, SOURCES)]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
