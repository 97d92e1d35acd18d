"""CPU ORACLE -- test infrastructure, not the product.

Python face of ``oracle/sph_oracle.c`` (read that file's header first).  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package; the product package
``paper_2302_08381_b200`` never does, and this package never imports it.

Two builds of the same C file:

* ``ld``  -- ``long double`` (x86 80-bit, eps 1.08e-19): the parity reference.
  Needed because the f64 tolerance (1e-12 with a 1e-3 row-scaled floor)
  asks for ~1e-15 of the row scale, which an f64 evaluation of Eq. 7 at l=32 does
  not deliver itself.
* ``f64`` -- ``double`` + OpenMP over points: the timed CPU baseline ("trivially
  parallelized over the sample index using OpenMP").

Paper citations ``P:n`` are lines of PAPER.md (arXiv 2302.08381).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "sph_oracle.c"
_LIBS = {"ld": _HERE / "liboracle_ld.so", "f64": _HERE / "liboracle_f64.so"}
_FLAGS = {"ld": ["-DORACLE_LONG_DOUBLE"], "f64": []}
_DTYPE = {"ld": np.longdouble, "f64": np.float64}
_loaded: dict[str, ctypes.CDLL] = {}


def build(force: bool = False) -> None:
    """Compile both builds with gcc (-O2 -fopenmp, no -ffast-math)."""
    for kind, lib in _LIBS.items():
        if not force and lib.exists() and lib.stat().st_mtime >= _SRC.stat().st_mtime:
            continue
        tmp = lib.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", *_FLAGS[kind],
               "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, lib)


def _lib(kind: str) -> ctypes.CDLL:
    if kind not in _loaded:
        build()
        _loaded[kind] = ctypes.CDLL(str(_LIBS[kind]))
    return _loaded[kind]


def _fn(kind: str, name: str):
    return getattr(_lib(kind), f"{name}_{kind}")


def _ptr(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def n_sph(l_max: int) -> int:
    return (l_max + 1) ** 2


def num_threads(kind: str = "f64") -> int:
    f = _fn(kind, "oracle_num_threads")
    f.restype = ctypes.c_int
    return int(f())


def compute(xyz, l_max: int, normalized: bool, gradients: bool = False, hessians: bool = False,
            kind: str = "ld", out=None):
    """Oracle for ``sphericart_cuda_compute``.

    ``xyz`` [n,3] float32/float64 (the exact values the GPU receives; widened to double, which
    is exact).  Returns ``(sph [n,L], dsph [n,3,L] | None, ddsph [n,3,3,L] | None)`` in
    ``np.longdouble`` (kind="ld") or ``np.float64`` (kind="f64").  ``out`` may hold preallocated
    ``(sph, dsph, ddsph)`` of that dtype.
    """
    if hessians and not gradients:
        raise ValueError("hessians need gradients (SURVEY 8(b))")
    xyz = np.ascontiguousarray(np.asarray(xyz), dtype=np.float64).reshape(-1, 3)
    n, L, dt = xyz.shape[0], n_sph(l_max), _DTYPE[kind]
    if out is None:
        sph = np.empty((n, L), dt)
        dsph = np.empty((n, 3, L), dt) if gradients else None
        ddsph = np.empty((n, 3, 3, L), dt) if hessians else None
    else:
        sph, dsph, ddsph = out
    f = _fn(kind, "oracle_compute")
    f.restype = ctypes.c_int
    f.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_int,
                  ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    rc = f(_ptr(xyz), n, int(l_max), int(bool(normalized)), _ptr(sph), _ptr(dsph), _ptr(ddsph))
    if rc != 0:
        raise RuntimeError("oracle_compute failed")
    return sph, dsph, ddsph


def vjp(dsph, grad_sph, l_max: int, kind: str = "ld"):
    """Oracle for ``sphericart_cuda_vjp``: grad_xyz[n,a] = sum_k dsph[n,a,k] grad_sph[n,k]."""
    dt = _DTYPE[kind]
    dsph = np.ascontiguousarray(np.asarray(dsph), dtype=dt)
    grad_sph = np.ascontiguousarray(np.asarray(grad_sph), dtype=dt)
    n = grad_sph.shape[0]
    out = np.empty((n, 3), dt)
    f = _fn(kind, "oracle_vjp")
    f.restype = ctypes.c_int
    f.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_void_p]
    if f(_ptr(dsph), _ptr(grad_sph), n, int(l_max), _ptr(out)) != 0:
        raise RuntimeError("oracle_vjp failed")
    return out


def vjp_recompute(xyz, grad_sph, l_max: int, normalized: bool, kind: str = "ld"):
    """Oracle for ``sphericart_cuda_vjp_recompute``: the backward pass of P:112
    with the derivatives evaluated again from ``xyz`` instead of stored in the forward pass.  It is
    the composition of the two oracle routines above and nothing else:
    grad_xyz[n,a] = sum_k (d sph[n,k] / d xyz[n,a]) grad_sph[n,k]."""
    _, dsph, _ = compute(xyz, l_max, normalized, gradients=True, kind=kind)
    return vjp(dsph, grad_sph, l_max, kind=kind)


def vjp2(xyz, grad_sph, v, l_max: int, normalized: bool, kind: str = "ld"):
    """Oracle for ``sphericart_cuda_vjp2`` ("second-order VJP for double backward";
    backward pass P:112, derivatives "of any order" P:94).  The backward pass is the map
    ``g(xyz, w)[n,a] = sum_k dsph[n,a,k](xyz) w[n,k]`` with ``w = grad_sph``; given an upstream
    gradient ``v [n,3]`` on its output, its own backward returns

        out_xyz[n,b] = sum_{a,k} ddsph[n,a,b,k] v[n,a] w[n,k]       (gradient w.r.t. xyz)
        out_w[n,k]   = sum_a     dsph[n,a,k]    v[n,a]              (gradient w.r.t. grad_sph)

    Nothing but ``compute(..., hessians=True)`` followed by two plain contractions in the oracle's
    precision."""
    dt = _DTYPE[kind]
    _, dsph, ddsph = compute(xyz, l_max, normalized, gradients=True, hessians=True, kind=kind)
    w = np.asarray(grad_sph).astype(dt)
    v = np.asarray(v).astype(dt)
    n, L = w.shape
    out_xyz = np.zeros((n, 3), dt)
    for a in range(3):
        for b in range(3):
            out_xyz[:, b] += v[:, a] * (ddsph[:, a, b, :] * w).sum(axis=1)
    out_w = np.zeros((n, L), dt)
    for a in range(3):
        out_w += dsph[:, a, :] * v[:, a:a + 1]
    return out_xyz, out_w


# Conventions other than the paper's own (the paper compares with e3nn).
# AXES_E3NN: the harmonics are those of the paper evaluated at the cyclically permuted point
# (x', y', z') = (z, x, y), so that the l = 1 row is proportional to (x, y, z) in that order instead
# of (y, z, x) (reading S1).  SCALE_*: what the per-l row norm sum_m Y_lm^2 is on the
# unit sphere: (2l+1)/4pi ("integral": orthonormal, the paper's), 2l+1 ("component"), 1 ("norm").
AXES_STANDARD, AXES_E3NN = 0, 1
SCALE_INTEGRAL, SCALE_COMPONENT, SCALE_NORM = 0, 1, 2


def compute_convention(xyz, l_max: int, normalized: bool, axes: int, scale: int, gradients: bool = False,
                       hessians: bool = False, kind: str = "ld"):
    """Oracle for ``sphericart_cuda_compute_ex``: ``compute`` at the permuted point, every l-row
    multiplied by its scale, derivative axes mapped back to the caller's (x, y, z)."""
    dt = _DTYPE[kind]
    xyz = np.ascontiguousarray(np.asarray(xyz), dtype=np.float64).reshape(-1, 3)
    perm = [2, 0, 1] if axes == AXES_E3NN else [0, 1, 2]       # ours[i] = caller's[perm[i]]
    sph, dsph, ddsph = compute(xyz[:, perm], l_max, normalized, gradients, hessians, kind=kind)
    l = np.concatenate([[ll] * (2 * ll + 1) for ll in range(l_max + 1)]).astype(dt)
    four_pi = 16 * np.arctan(dt(1))
    sc = {SCALE_INTEGRAL: np.ones_like(l), SCALE_COMPONENT: np.sqrt(four_pi) * np.ones_like(l),
          SCALE_NORM: np.sqrt(four_pi / (2 * l + 1))}[scale]
    sph = sph * sc
    inv = np.argsort(perm)                                     # d/d caller's[j] = d/d ours[inv[j]]
    if dsph is not None:
        dsph = dsph[:, inv, :] * sc
    if ddsph is not None:
        ddsph = ddsph[:, inv][:, :, inv] * sc
    return sph, dsph, ddsph


def expand(xyz, radial, seg_ptr, l_max: int):
    """Oracle for ``sphericart_cuda_expand`` (Eq. 1):

        c[s, n, lm] = sum over the points k of segment s of  R[k, n, l] * Y_l^m(r_k / |r_k|),

    ``xyz`` [N,3] the points r_k, ``radial`` [N, n_rad, l_max+1] the values R_nl(r_k) (the paper
    leaves the radial basis to the application: they are an input), ``seg_ptr`` [S+1] ascending
    offsets: segment s (e.g. the neighbours of centre s) is the points seg_ptr[s] .. seg_ptr[s+1]-1.
    Plain loops over segments, long double throughout; Y from ``compute`` (normalised)."""
    xyz = np.ascontiguousarray(np.asarray(xyz), dtype=np.float64).reshape(-1, 3)
    radial = np.asarray(radial)
    seg_ptr = np.asarray(seg_ptr, dtype=np.int64)
    n, n_rad = xyz.shape[0], radial.shape[1]
    assert radial.shape == (n, n_rad, l_max + 1) and seg_ptr[0] == 0 and seg_ptr[-1] == n
    Y, _, _ = compute(xyz, l_max, True)
    l_of = np.concatenate([[l] * (2 * l + 1) for l in range(l_max + 1)])
    R = radial.astype(np.longdouble)[:, :, l_of]            # [N, n_rad, L]: R_nl repeated over m
    out = np.zeros((len(seg_ptr) - 1, n_rad, n_sph(l_max)), np.longdouble)
    for s in range(len(seg_ptr) - 1):
        for k in range(seg_ptr[s], seg_ptr[s + 1]):
            out[s] += R[k] * Y[k][None, :]
    return out


def F_table(l_max: int, kind: str = "ld"):
    """F_l^m (Eq. C1) as a flat triangle, index l(l+1)/2+m."""
    out = np.empty((l_max + 1) * (l_max + 2) // 2, _DTYPE[kind])
    f = _fn(kind, "oracle_F_table")
    f.restype = None
    f.argtypes = [ctypes.c_int, ctypes.c_void_p]
    f(int(l_max), _ptr(out))
    return out


def Q_triangle(z, r2, l_max: int):
    """Q_l^m(z, r^2) (Eq. 7) in long double, flat triangle index l(l+1)/2+m."""
    out = np.empty((l_max + 1) * (l_max + 2) // 2, np.longdouble)
    zz = np.array([z], np.longdouble)
    rr = np.array([r2], np.longdouble)
    f = _fn("ld", "oracle_Q_p")
    f.restype = None
    f.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p]
    f(_ptr(zz), _ptr(rr), int(l_max), _ptr(out))
    return out


def cs(x, y, l_max: int):
    """c_m, s_m (Eq. 9) in long double."""
    c = np.empty(l_max + 1, np.longdouble)
    s = np.empty(l_max + 1, np.longdouble)
    xx = np.array([x], np.longdouble)
    yy = np.array([y], np.longdouble)
    f = _fn("ld", "oracle_cs_p")
    f.restype = None
    f.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
    f(_ptr(xx), _ptr(yy), int(l_max), _ptr(c), _ptr(s))
    return c, s
