"""Build libsdtw.so (the C-ABI library of include/sdtw.h) in-tree with nvcc for sm_100a.

    python -m paper_2404_12134_b200.build [--force] [--verbose]

nvcc cross-compiles without a GPU.  The .so is git-ignored but travels with the tree.
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
CSRC = PKG / "csrc"
LIB = PKG / "libsdtw.so"
SOURCES = [CSRC / "sdtw.cu", CSRC / "mufu_peak.cu"]
DEPS = SOURCES + sorted(CSRC.glob("*.cuh")) + [ROOT / "include" / "sdtw.h"]


def nvcc_path() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def command(out: Path, verbose: bool = False) -> list[str]:
    cmd = [nvcc_path(), "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
           "-Xcompiler", "-fPIC", "-shared", "-I", str(ROOT / "include"), "-I", str(CSRC), "-o", str(out)]
    if verbose:
        cmd += ["-Xptxas", "-v"]
    return cmd + [str(s) for s in SOURCES]


def up_to_date() -> bool:
    return LIB.exists() and all(LIB.stat().st_mtime >= p.stat().st_mtime for p in DEPS)


def build(force: bool = False, verbose: bool = False) -> Path:
    if force or not up_to_date():
        tmp = LIB.with_suffix(f".tmp{os.getpid()}.so")
        subprocess.run(command(tmp, verbose), check=True)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
