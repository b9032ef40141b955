"""Build libebic.so (the C-ABI library of include/ebic.h) in-tree with nvcc for sm_100a.

    python -m paper_1807_09932_b200.csrc.build [--force] [--verbose]

Output: paper_1807_09932_b200/libebic.so (git-ignored; travels to the GPU box with the snapshot).
No fast-math, no flush-to-zero: the trend predicate needs exact IEEE float32 comparisons.
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

CSRC = Path(__file__).resolve().parent
PKG = CSRC.parent
LIB = PKG / "libebic.so"
SOURCES = [CSRC / "ebic_api.cu", CSRC / "ebic_debug.cu", CSRC / "ebic_reader.cu"]
HEADERS = (sorted(CSRC.glob("*.cuh")) + sorted(CSRC.glob("*.hpp")) +
           [PKG.parent / "include" / "ebic.h", PKG.parent / "include" / "ebic_debug.h"])

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-ftz=false", "-prec-div=true", "-prec-sqrt=true", "-fmad=false",
    "-Xcompiler", "-fPIC", "-shared",
]


def needs_build() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    return any(p.stat().st_mtime > t for p in SOURCES + HEADERS + [Path(__file__)])


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", str(tmp), *map(str, SOURCES)]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed building libebic.so")
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
