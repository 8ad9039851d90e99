"""Build step: compile csrc/*.cu for sm_100a into libgalario_b200.so next to this file.

One object per translation unit (the C ABI and one unit per kernel family and precision), compiled in
parallel, then linked.  nvcc cross-compiles without a GPU.  The .so is git-ignored but travels to the GPU
box with the repo snapshot.  Run as ``python -m paper_1709_06999_b200.build`` or through
``__graft_entry__.build()``.
"""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
OBJ = HERE / "build"
LIB = HERE / "libgalario_b200.so"

NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC"]


def sources():
    return sorted(CSRC.glob("*.cu"))


def headers():
    return sorted(CSRC.glob("*.cuh")) + sorted(CSRC.glob("*.h")) + [HERE.parent / "include" / "galario_b200.h"]


def _stale(target: Path, deps) -> bool:
    return not target.exists() or any(target.stat().st_mtime < d.stat().st_mtime for d in deps)


STAMP = OBJ / "flags.stamp"


def _flags() -> str:
    """The flag set the objects are compiled with.  It is written next to them: objects from a tuning build
    (GAL_NVCC_EXTRA=-D...) must never be mistaken for fresh ones by a later default build, or the other way round."""
    return " ".join(NVCC_FLAGS + os.environ.get("GAL_NVCC_EXTRA", "").split())


def _flags_changed() -> bool:
    return not STAMP.exists() or STAMP.read_text() != _flags()


def needs_build() -> bool:
    return _flags_changed() or _stale(LIB, sources() + headers())


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    extra = os.environ.get("GAL_NVCC_EXTRA", "").split()        # e.g. -DGAL_SAMPLE_U=2 for tuning builds
    OBJ.mkdir(exist_ok=True)
    hdrs = headers()
    jobs = []
    force = force or _flags_changed()                           # other flags than the objects on disk were built with
    if STAMP.exists():
        STAMP.unlink()                                          # (rewritten once every object has been compiled)
    for src in sources():
        obj = OBJ / (src.stem + ".o")
        if force or _stale(obj, [src] + hdrs):
            jobs.append([nvcc, *NVCC_FLAGS, *extra, *(["-Xptxas", "-v"] if verbose else []), "-c", str(src), "-o", str(obj)])
    with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 1) or 1) as ex:
        for r in ex.map(lambda c: subprocess.run(c, capture_output=not verbose, text=True), jobs):
            if r.returncode != 0:
                raise RuntimeError(f"nvcc failed: {' '.join(r.args)}\n{r.stdout or ''}\n{r.stderr or ''}")
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    objs = [str(OBJ / (s.stem + ".o")) for s in sources()]
    subprocess.run([nvcc, "-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a", "-o", str(tmp), *objs],
                   check=True)
    os.replace(tmp, LIB)
    STAMP.write_text(_flags())
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
