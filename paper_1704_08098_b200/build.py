"""Build libpgg.so in-tree with nvcc for sm_100a (cross-compiles without a GPU).

    python -m paper_1704_08098_b200.build [--force]

The shared library lands next to this file so that it travels with the source
tree; it is the only native artefact of the package.
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libpgg.so"
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "-Xcompiler", "-fPIC,-ffp-contract=off",
    "-shared", "-cudart", "static",
]


def sources():
    return sorted(CSRC.glob("*.cu")), sorted(list(CSRC.glob("*.cuh")) + [PKG.parent / "include" / "pgg.h"])


def stale() -> bool:
    if not LIB.exists():
        return True
    cu, hdr = sources()
    t = LIB.stat().st_mtime
    return any(p.stat().st_mtime > t for p in cu + hdr + [Path(__file__)])


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and not stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cu, _ = sources()
    tmp = LIB.with_suffix(f".{os.getpid()}.tmp.so")
    cmd = [nvcc, *NVCC_FLAGS, "-o", str(tmp), *map(str, cu)]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd), file=sys.stderr)
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
