"""Build the sm_100a C-ABI library in-tree: paper_1503_06203_b200/libcorr_b200.so.

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels with the repo snapshot
to the GPU box.
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
LIB = HERE / "libcorr_b200.so"
SOURCES = [CSRC / "corr_api.cu"]
DEPS = sorted(CSRC.glob("*.cu*")) + [HERE.parent / "include" / "corr.h"]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "-shared", "-Xcompiler", "-fPIC",
    "--cudart", "static",
]


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and LIB.exists() and all(LIB.stat().st_mtime >= d.stat().st_mtime for d in DEPS):
        return LIB
    extra = os.environ.get("CORR_NVCC_EXTRA", "").split()   # e.g. -DT5_PK_N=4 (kernel tuning experiments)
    out = Path(os.environ.get("CORR_LIB_OUT", str(LIB)))
    cmd = ["nvcc", *NVCC_FLAGS, *extra, *(["-Xptxas", "-v"] if verbose else []), *map(str, SOURCES), "-o", str(out)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libcorr_b200.so")
    return LIB


if __name__ == "__main__":
    build(force=True, verbose="-v" in sys.argv)
    print(LIB)
