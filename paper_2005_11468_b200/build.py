"""Build the C-ABI shared library (libpsr_b200.so) in-tree with nvcc for sm_100a.

    python -m paper_2005_11468_b200.build [--force]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels with the gpurun snapshot.
"""
from __future__ import annotations

import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libpsr_b200.so"
SOURCES = [CSRC / "psr_api.cu", CSRC / "psr_kernels.cu", CSRC / "psr_ws.cu", CSRC / "psr_jac.cu", CSRC / "psr_lu.cu", CSRC / "psr_solve.cu"]
HEADERS = [CSRC / "psr_tables.h", CSRC / "psr_math.cuh", CSRC / "psr_ptx.cuh", CSRC / "psr_rx.cuh", PKG.parent / "include" / "psr.h"]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared", "--fmad=true", "-Xptxas", "-v",
]


def needs_build() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any(p.stat().st_mtime > t for p in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> Path:
    if force or needs_build():
        cmd = ["nvcc", *NVCC_FLAGS, "-o", str(LIB), *[str(s) for s in SOURCES]]
        res = subprocess.run(cmd, capture_output=True, text=True)
        log = res.stdout + res.stderr
        (PKG / "build.log").write_text(" ".join(cmd) + "\n" + log)
        if res.returncode != 0:
            raise RuntimeError("nvcc failed:\n" + log[-4000:])
        if verbose:
            print(log)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
    print(LIB)
