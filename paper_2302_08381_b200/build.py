"""In-tree build of the CUDA library: ``python -m paper_2302_08381_b200.build``.

sm_100a only, ``-lineinfo`` so ncu's source page maps to the .cuh files.  The translation units
(``api.cu``, ``tables.cpp``, ``tpb_inst.cu`` once per element type and derivative order, ``vjpr_inst.cu`` and
``expand_inst.cu`` and ``tq_inst.cu`` once per element type) are
compiled in parallel and linked into one shared library.
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
SOURCES = [CSRC / "api.cu", CSRC / "tables.cpp", CSRC / "tpb_inst.cu", CSRC / "vjpr_inst.cu", CSRC / "expand_inst.cu",
           CSRC / "tq_inst.cu"]
HEADERS = sorted(CSRC.glob("*.cuh")) + sorted(CSRC.glob("*.h")) + [PKG.parent / "include" / "sphericart_cuda.h"]
OBJ_DIR = PKG / "build"

# (object name, source, extra defines)
UNITS = [("api", CSRC / "api.cu", []), ("tables", CSRC / "tables.cpp", [])] + [
    (f"tpb_f{64 if f64 else 32}_{'vgh'[deriv]}", CSRC / "tpb_inst.cu", [f"-DTPB_F64={f64}", f"-DTPB_DERIV={deriv}"])
    for f64 in (0, 1) for deriv in (0, 1, 2)] + [
    (f"vjpr_f{64 if f64 else 32}", CSRC / "vjpr_inst.cu", [f"-DVJPR_F64={f64}"]) for f64 in (0, 1)] + [
    (f"expand_f{64 if f64 else 32}", CSRC / "expand_inst.cu", [f"-DEXPAND_F64={f64}"]) for f64 in (0, 1)] + [
    (f"tq_f{64 if f64 else 32}", CSRC / "tq_inst.cu", [f"-DTQ_F64={f64}"]) for f64 in (0, 1)]

NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC"]


def nvcc() -> str:
    return os.environ.get("NVCC", "nvcc")


def compile_command(name: str, src: Path, defines: list[str], verbose: bool = False) -> list[str]:
    return [nvcc(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), *defines, "-c", str(src),
            "-o", str(OBJ_DIR / f"{name}.o")]


def link_command(out: Path) -> list[str]:
    return [nvcc(), *NVCC_FLAGS, "-shared", "-o", str(out), *[str(OBJ_DIR / f"{u[0]}.o") for u in UNITS],
            "-l:libquadmath.a"]


def up_to_date() -> bool:
    if not LIB.exists():
        return False
    t = LIB.stat().st_mtime
    return all(p.stat().st_mtime <= t for p in SOURCES + HEADERS + [Path(__file__)])


def _run(cmd: list[str], verbose: bool) -> None:
    res = subprocess.run(cmd, capture_output=True, text=True)
    if verbose or res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
    if res.returncode != 0:
        raise RuntimeError("nvcc failed: " + " ".join(cmd))


def build(force: bool = False, verbose: bool = False) -> Path:
    if not force and up_to_date():
        return LIB
    from concurrent.futures import ThreadPoolExecutor

    OBJ_DIR.mkdir(exist_ok=True)
    with ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 1)) as pool:
        list(pool.map(lambda u: _run(compile_command(*u, verbose=verbose), verbose), UNITS))
    tmp = LIB.with_suffix(f".tmp{os.getpid()}.so")
    try:
        _run(link_command(tmp), verbose)
    except RuntimeError:
        tmp.unlink(missing_ok=True)
        raise
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
