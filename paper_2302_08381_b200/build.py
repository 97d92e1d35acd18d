"""In-tree build of the CUDA library: ``python -m paper_2302_08381_b200.build``.

One nvcc invocation, sm_100a only, ``-lineinfo`` so ncu's source page maps to the .cuh files.
The result, ``paper_2302_08381_b200/libsphericart_cuda.so``, is git-ignored but travels to the
GPU box with the repository snapshot.
"""
from __future__ import annotations

import os
import subprocess
import sys
from pathlib import Path

PKG = Path(__file__).resolve().parent
CSRC = PKG / "csrc"
LIB = PKG / "libsphericart_cuda.so"
SOURCES = [CSRC / "api.cu", CSRC / "tables.cpp"]
HEADERS = sorted(CSRC.glob("*.cuh")) + sorted(CSRC.glob("*.h")) + [PKG.parent / "include" / "sphericart_cuda.h"]


def nvcc_command(out: Path, extra: list[str] | None = None) -> list[str]:
    nvcc = os.environ.get("NVCC", "nvcc")
    return [nvcc, "-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
            "-Xcompiler", "-fPIC", "-shared", *(extra or []), "-o", str(out),
            *[str(s) for s in SOURCES], "-l:libquadmath.a"]


def up_to_date() -> bool:
    if not LIB.exists():
        return False
    t = LIB.stat().st_mtime
    return all(p.stat().st_mtime <= t for p in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and up_to_date():
        return LIB
    tmp = LIB.with_suffix(f".tmp{os.getpid()}.so")
    cmd = nvcc_command(tmp, ["-Xptxas", "-v"] if verbose else None)
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        tmp.unlink(missing_ok=True)
        raise RuntimeError("nvcc failed: " + " ".join(cmd))
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
