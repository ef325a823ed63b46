"""Builds libmg (the sm_100a CUDA library behind include/mg.h) in-tree with nvcc.

The shared object lands in ``paper_2605_30082_b200/_lib/libmg-<hash>.so`` where the hash
covers every source file and the flags, so a stale binary is never loaded.  The built
file travels to the GPU box with the repository snapshot; if it is missing there it is
rebuilt on first import (nvcc is part of the image).
"""
from __future__ import annotations

import hashlib
import os
import shutil
import subprocess
from pathlib import Path

PKG = Path(__file__).resolve().parent
ROOT = PKG.parent
CSRC = PKG / "csrc"
LIBDIR = PKG / "_lib"

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-lineinfo", "-O3", "-std=c++17",
    "-fmad=false",                 # no implicit contraction: all fma are explicit
    "-Xcompiler", "-fPIC", "-shared",
]


def sources():
    return sorted(CSRC.glob("*.cu")) + sorted(CSRC.glob("*.cuh")) + [ROOT / "include" / "mg.h"]


def lib_path() -> Path:
    h = hashlib.sha1()
    for p in sources():
        h.update(p.name.encode())
        h.update(p.read_bytes())
    h.update(" ".join(NVCC_FLAGS).encode())
    return LIBDIR / f"libmg-{h.hexdigest()[:12]}.so"


def nvcc() -> str:
    exe = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not Path(exe).exists():
        raise RuntimeError("nvcc not found: libmg cannot be built (and there is no CPU fallback)")
    return exe


def build(force: bool = False, verbose: bool = False) -> Path:
    out = lib_path()
    if out.exists() and not force:
        return out
    LIBDIR.mkdir(exist_ok=True)
    import fcntl

    # several ranks may import at once (torchrun): one builds, the others wait for the lock and
    # find the library; stale hashes are removed only after the new file is in place
    with open(LIBDIR / ".build.lock", "w") as lock:
        fcntl.flock(lock, fcntl.LOCK_EX)
        if out.exists() and not force:
            return out
        tmp = out.with_suffix(f".tmp{os.getpid()}")
        cmd = [nvcc(), *NVCC_FLAGS, "-o", str(tmp), str(CSRC / "mg.cu")]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
            print(" ".join(cmd))
        subprocess.run(cmd, check=True, cwd=CSRC)
        os.replace(tmp, out)
        for old in LIBDIR.glob("libmg-*.so"):
            if old != out:
                old.unlink()
    return out


if __name__ == "__main__":
    print(build(force=True, verbose=True))
