"""Build libmicsa.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_2506_16240_b200.build [--force]
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
INCLUDE = PKG.parent / "include"
LIB = PKG / "libmicsa.so"

NVCC_FLAGS = [
    "-O3", "-std=c++17", "-lineinfo",
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-Xcompiler", "-fPIC", "-shared", "-cudart", "static",
]


def sources():
    return sorted(CSRC.glob("*.cu")), sorted(CSRC.glob("*.cuh")) + sorted(INCLUDE.glob("*.h"))


def needs_build() -> bool:
    if not LIB.exists():
        return True
    cu, deps = sources()
    t = LIB.stat().st_mtime
    return any(p.stat().st_mtime > t for p in cu + deps)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not needs_build():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cu, _ = sources()
    tmp = PKG / f"libmicsa.{os.getpid()}.tmp.so"
    cmd = [nvcc, "--threads", "0"] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
          ["-I", str(INCLUDE), "-o", str(tmp)] + [str(p) for p in cu]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
