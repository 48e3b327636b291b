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
SOURCES = [CSRC / "psr_api.cu", CSRC / "psr_kernels.cu", CSRC / "psr_ws.cu", CSRC / "psr_wsl.cu", CSRC / "psr_jac.cu", CSRC / "psr_lu.cu", CSRC / "psr_solve.cu"]
HEADERS = [CSRC / "psr_tables.h", CSRC / "psr_math.cuh", CSRC / "psr_ptx.cuh", CSRC / "psr_rx.cuh", PKG.parent / "include" / "psr.h"]

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
    "-Xcompiler", "-fPIC", "-shared", "--fmad=true", "-Xptxas", "-v",
]


LIB_CHECK = PKG / "libpsr_b200_check.so"   # the same sources with -DPSR_CHECK (device-side bounds assertions; tests only)


def _stale(lib: Path) -> bool:
    if not lib.exists():
        return True
    t = lib.stat().st_mtime
    return any(p.stat().st_mtime > t for p in SOURCES + HEADERS)


def needs_build() -> bool:
    return _stale(LIB)


def _cmd(lib: Path, extra):
    return ["nvcc", *NVCC_FLAGS, *extra, "-o", str(lib), *[str(s) for s in SOURCES]]


def _finish(proc, cmd, log_name: str):
    out, err = proc.communicate()
    log = (out or "") + (err or "")
    (PKG / log_name).write_text(" ".join(cmd) + "\n" + log)
    if proc.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + log[-4000:])
    return log


def build(force: bool = False, verbose: bool = False, check: bool = False) -> Path:
    """Builds libpsr_b200.so; with check=True also the bounds-checked libpsr_b200_check.so (the two nvcc runs side by side)."""
    jobs = []
    if force or needs_build():
        cmd = _cmd(LIB, [])
        jobs.append((subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True), cmd, "build.log"))
    if check and (force or _stale(LIB_CHECK)):
        cmd = _cmd(LIB_CHECK, ["-DPSR_CHECK"])
        jobs.append((subprocess.Popen(cmd, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True), cmd, "build_check.log"))
    for proc, cmd, name in jobs:
        log = _finish(proc, cmd, name)
        if verbose:
            print(log)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True, check="--check" in sys.argv)
    print(LIB)
