"""Build libsynax.so in-tree with nvcc for sm_100a (B200).  `python -m paper_2410_01136_b200.build`."""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libsynax.so"
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]


def sources():
    return sorted(CSRC.glob("*.cu")), sorted(CSRC.glob("*.cuh")) + [PKG.parent / "include" / "synax.h"]


def up_to_date() -> bool:
    if not LIB.exists():
        return False
    cu, hdr = sources()
    t = LIB.stat().st_mtime
    return all(p.stat().st_mtime <= t for p in cu + hdr)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and up_to_date():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    cu, _ = sources()
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    cmd = [nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), "-o", str(tmp), *map(str, cu)]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
