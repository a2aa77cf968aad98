"""Compile the CUDA kernels + C ABI into libsplats.so, in-tree, for sm_100a only."""
from __future__ import annotations

import os
import shutil
import subprocess
from pathlib import Path

HERE = Path(__file__).resolve().parent
CSRC = HERE / "csrc"
LIB = HERE / "libsplats.so"
INCLUDE = HERE.parent / "include"

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-lineinfo", "-std=c++17",
    "--shared", "-Xcompiler", "-fPIC", "-Xcompiler", "-ffp-contract=off",
    "-cudart", "static",
]


def sources():
    return sorted(CSRC.glob("*.cu"))


def _newest_source_mtime() -> float:
    files = list(CSRC.glob("*.cu")) + list(CSRC.glob("*.cuh")) + list(INCLUDE.glob("*.h"))
    return max(f.stat().st_mtime for f in files)


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and Path(cand).exists():
            return cand
    raise RuntimeError("nvcc not found: the CUDA extension cannot be built (there is no CPU fallback)")


def build(force: bool = False, verbose: bool = False, extra: list[str] | None = None) -> Path:
    if not force and LIB.exists() and LIB.stat().st_mtime >= _newest_source_mtime():
        return LIB
    extra = list(extra or []) + os.environ.get("SPLATS_NVCC_EXTRA", "").split()   # e.g. -DSPLATS_STATS (debug builds)
    cmd = [nvcc_path(), *NVCC_FLAGS, *extra, f"-I{INCLUDE}", *map(str, sources()), "-o", str(LIB)]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd))
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    import sys
    build(force=True, verbose="-v" in sys.argv)
    print(LIB)
