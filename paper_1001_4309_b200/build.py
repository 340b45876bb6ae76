"""Builds ``libsfd.so`` (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1001_4309_b200.build [--force]

nvcc cross-compiles without a GPU.  The result sits next to this file so that it travels to the
GPU box with the repo snapshot; it is git-ignored."""
from __future__ import annotations

import os
import pathlib
import shutil
import subprocess
import sys

PKG = pathlib.Path(__file__).resolve().parent
ROOT = PKG.parent
CSRC = PKG / "csrc"
LIB = PKG / "libsfd.so"
SOURCES = [CSRC / "sfd_kernels.cu", CSRC / "sfd_asm.cu", CSRC / "sfd_plan.cpp"]
HEADERS = [CSRC / "sfd_fft_core.cuh", CSRC / "sfd_dft32.cuh", CSRC / "sfd_warp1024.cuh", CSRC / "sfd_warp2048.cuh", CSRC / "sfd_warp512.cuh", CSRC / "sfd_asm1024.cuh", CSRC / "sfd_asm2048.cuh", CSRC / "sfd_internal.h", ROOT / "include" / "sfd.h"]

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
    "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden", "-Xlinker", "--exclude-libs,ALL",
]


def _nvcc():
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(exe):
        raise RuntimeError("nvcc not found; libsfd.so cannot be built")
    return exe


def stale():
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any(f.stat().st_mtime > t for f in SOURCES + HEADERS + [pathlib.Path(__file__)])


def build(force=False, verbose=False):
    """Compile libsfd.so if it is missing or older than its sources.  Returns its path."""
    if not force and not stale():
        return LIB
    cmd = [_nvcc(), *NVCC_FLAGS, "-shared", "-I", str(ROOT / "include"), "-I", str(CSRC),
           "-o", str(LIB), *map(str, SOURCES)]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd))
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed:\n" + r.stdout + r.stderr)
    if verbose:
        print(r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
