"""Builds librc.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import shutil
import subprocess
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "librc.so"
SOURCES = [CSRC / "rc_api.cu", CSRC / "rc_kernels.cu", CSRC / "rc_static.cu"]
DEPS = SOURCES + [CSRC / "rc_internal.h", PKG.parent / "include" / "rc.h"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not Path(exe).exists():
        raise RuntimeError("nvcc not found: librc.so cannot be built (there is no CPU fallback)")
    return exe


def stale() -> bool:
    return not LIB.exists() or any(LIB.stat().st_mtime < d.stat().st_mtime for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> Path:
    if force or stale():
        tmp = LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = [nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", str(tmp), *map(str, SOURCES)]
        subprocess.check_call(cmd, cwd=str(CSRC))
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
