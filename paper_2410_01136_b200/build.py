"""Build libsynax.so in-tree with nvcc for sm_100a (B200).  `python -m paper_2410_01136_b200.build [--force] [-v]`.

One object file per translation unit of csrc/ (the template kernels are instantiated per model code in their own
files, see csrc/synax_launch.h), compiled in parallel, then linked.  Freshness is decided by a hash of the sources and
flags stored beside the library (`libsynax.so.srchash`) together with the name of the machine that compiled it, not by
modification times: a library built from other sources, or shipped in from another machine (the GPU box receives the
tree with the builder's binary in it), is compiled again where it runs.  SYNAX_TRUST_SHIPPED_LIB=1 accepts a shipped
library whose source hash matches.
"""
from __future__ import annotations

import hashlib
import os
import platform
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libsynax.so"
STAMP = PKG / "libsynax.so.srchash"
OBJ = PKG / "build"
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def sources():
    return sorted(CSRC.glob("*.cu")), sorted(CSRC.glob("*.cuh")) + sorted(CSRC.glob("*.h")) + [PKG.parent / "include" / "synax.h"]


def source_hash() -> str:
    h = hashlib.sha256()
    cu, hdr = sources()
    for p in cu + hdr:
        h.update(p.name.encode())
        h.update(p.read_bytes())
    h.update(" ".join(NVCC_FLAGS).encode())
    h.update(os.environ.get("SYNAX_NVCC_EXTRA", "").encode())
    return h.hexdigest()


def machine_id() -> str:
    """Identifies the machine (and boot) that compiled the library: the kernel's boot id, else the host name."""
    try:
        return Path("/proc/sys/kernel/random/boot_id").read_text().strip()
    except OSError:
        return platform.node()


def _stamp():
    if not (LIB.exists() and STAMP.exists()):
        return None, None
    lines = STAMP.read_text().split()
    return (lines + [None, None])[:2]


def up_to_date() -> bool:
    digest, machine = _stamp()
    if digest != source_hash():
        return False
    return machine == machine_id() or os.environ.get("SYNAX_TRUST_SHIPPED_LIB") == "1"


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and up_to_date():
        return LIB
    nvcc = os.environ.get("NVCC", "nvcc")
    extra = os.environ.get("SYNAX_NVCC_EXTRA", "").split()
    cu, _ = sources()
    OBJ.mkdir(exist_ok=True)
    digest = source_hash()
    jobs = max(1, min(len(cu), os.cpu_count() or 1))

    def compile_one(src: Path) -> Path:
        obj = OBJ / (src.stem + ".o")
        cmd = [nvcc, *NVCC_FLAGS, *extra, *(["-Xptxas", "-v"] if verbose else []), "-c", "-o", str(obj), str(src)]
        r = subprocess.run(cmd, capture_output=True, text=True)
        if verbose or r.returncode != 0:
            sys.stderr.write(r.stdout + r.stderr)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed on {src.name}")
        return obj

    try:
        with ThreadPoolExecutor(jobs) as ex:
            objs = list(ex.map(compile_one, cu))
    except (RuntimeError, OSError) as e:
        if not force and _stamp()[0] == digest:   # the shipped binary matches these sources: use it, but say so
            sys.stderr.write(f"paper_2410_01136_b200.build: recompiling here failed ({e}); using the shipped libsynax.so\n")
            return LIB
        raise
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    subprocess.run([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-o", str(tmp), *map(str, objs)], check=True)
    os.replace(tmp, LIB)
    STAMP.write_text(f"{digest}\n{machine_id()}\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
