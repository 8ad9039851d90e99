"""Build step: compile csrc/galario_b200.cu for sm_100a into libgalario_b200.so next to this file.

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU box with the
repo snapshot.  Run as ``python -m paper_1709_06999_b200.build`` or through
``__graft_entry__.build()``.
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

HERE = Path(__file__).resolve().parent
SRC = HERE / "csrc" / "galario_b200.cu"
DEPS = [SRC, HERE / "csrc" / "fft.cuh", HERE / "csrc" / "sample.cuh", HERE.parent / "include" / "galario_b200.h"]
LIB = HERE / "libgalario_b200.so"

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def needs_build() -> bool:
    return not LIB.exists() or any(LIB.stat().st_mtime < d.stat().st_mtime for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    cmd = [nvcc, *NVCC_FLAGS, *( ["-Xptxas", "-v"] if verbose else []), "-o", str(tmp), str(SRC)]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
