"""B200-native real spherical harmonics (arXiv 2302.08381's Cartesian scheme): Python binding.

A thin ``ctypes`` face of ``libsphericart_cuda.so`` (``include/sphericart_cuda.h``).  The
functions below carry the C names and do argument marshalling only -- every step of the path runs
in the library's sm_100a kernels.  PyTorch supplies device memory and streams, nothing else.
There is no CPU fallback: if the library is missing or the call fails, an exception is raised.

    sphericart_cuda_compute(xyz, n, l_max, normalized, dtype, sph, dsph, ddsph, stream)
    sphericart_cuda_vjp(xyz, dsph, grad_sph, grad_xyz, n, l_max, dtype, stream)
    sphericart_cuda_compute_host(...), sphericart_cuda_vjp_host(...)      host buffers
    compute(xyz, l_max, ...), vjp(dsph, grad_sph)                         torch.Tensor convenience
"""
from __future__ import annotations

import ctypes
from pathlib import Path

_PKG = Path(__file__).resolve().parent
_LIB_PATH = _PKG / "libsphericart_cuda.so"
_lib = None

F32, F64 = 0, 1
MAX_L = 32
AXES_STANDARD, AXES_E3NN = 0, 1
SCALE_INTEGRAL, SCALE_COMPONENT, SCALE_NORM = 0, 1, 2


class SphericartCudaError(RuntimeError):
    pass


def library_path() -> Path:
    return _LIB_PATH


def load():
    """Load the CUDA library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not _LIB_PATH.exists():
        raise SphericartCudaError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_2302_08381_b200.build` "
            "(there is no CPU fallback)")
    lib = ctypes.CDLL(str(_LIB_PATH))
    vp, i64, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int
    lib.sphericart_cuda_compute.restype = ci
    lib.sphericart_cuda_compute.argtypes = [vp, i64, ci, ci, ci, vp, vp, vp, vp]
    lib.sphericart_cuda_vjp.restype = ci
    lib.sphericart_cuda_vjp.argtypes = [vp, vp, vp, vp, i64, ci, ci, vp]
    lib.sphericart_cuda_compute_host.restype = ci
    lib.sphericart_cuda_compute_host.argtypes = [vp, i64, ci, ci, ci, vp, vp, vp]
    lib.sphericart_cuda_vjp_recompute.restype = ci
    lib.sphericart_cuda_vjp_recompute.argtypes = [vp, vp, vp, i64, ci, ci, ci, vp]
    lib.sphericart_cuda_compute_ex.restype = ci
    lib.sphericart_cuda_compute_ex.argtypes = [vp, i64, ci, ci, ci, ci, ci, vp, vp, vp, vp]
    lib.sphericart_cuda_vjp2.restype = ci
    lib.sphericart_cuda_vjp2.argtypes = [vp, vp, vp, vp, vp, i64, ci, ci, ci, vp]
    lib.sphericart_cuda_expand.restype = ci
    lib.sphericart_cuda_expand.argtypes = [vp, vp, vp, i64, ci, ci, ci, vp, vp]
    lib.sphericart_cuda_vjp_noalloc.restype = ci
    lib.sphericart_cuda_vjp_noalloc.argtypes = [vp, vp, vp, i64, ci, ci, vp]
    lib.sphericart_cuda_vjp_host.restype = ci
    lib.sphericart_cuda_vjp_host.argtypes = [vp, vp, vp, vp, i64, ci, ci]
    lib.sphericart_cuda_last_error.restype = ctypes.c_char_p
    lib.sphericart_cuda_last_error.argtypes = []
    lib.sphericart_cuda_launch_count.restype = i64
    lib.sphericart_cuda_launch_count.argtypes = []
    lib.sphericart_cuda_last_kernel.restype = ctypes.c_char_p
    lib.sphericart_cuda_last_kernel.argtypes = []
    lib.sphericart_cuda_set_option.restype = ci
    lib.sphericart_cuda_set_option.argtypes = [ctypes.c_char_p, ctypes.c_char_p]
    _lib = lib
    return lib


def _ptr(a):
    """Address of a torch tensor / numpy array / int / None."""
    if a is None:
        return None
    if isinstance(a, int):
        return a
    if hasattr(a, "data_ptr"):
        return a.data_ptr()
    return a.ctypes.data


def _check(rc: int, what: str):
    if rc != 0:
        msg = load().sphericart_cuda_last_error().decode()
        raise SphericartCudaError(f"{what} failed (code {rc}): {msg}")


# --- the C entry points, same names, same argument order ---------------------------------------
def sphericart_cuda_compute(xyz, n, l_max, normalized, dtype, sph, dsph, ddsph, stream):
    rc = load().sphericart_cuda_compute(_ptr(xyz), n, l_max, int(normalized), dtype, _ptr(sph),
                                        _ptr(dsph), _ptr(ddsph), _ptr(stream))
    _check(rc, "sphericart_cuda_compute")


def sphericart_cuda_vjp(xyz, dsph, grad_sph, grad_xyz, n, l_max, dtype, stream):
    rc = load().sphericart_cuda_vjp(_ptr(xyz), _ptr(dsph), _ptr(grad_sph), _ptr(grad_xyz), n, l_max,
                                    dtype, _ptr(stream))
    _check(rc, "sphericart_cuda_vjp")


def sphericart_cuda_compute_host(xyz, n, l_max, normalized, dtype, sph, dsph, ddsph):
    rc = load().sphericart_cuda_compute_host(_ptr(xyz), n, l_max, int(normalized), dtype, _ptr(sph),
                                             _ptr(dsph), _ptr(ddsph))
    _check(rc, "sphericart_cuda_compute_host")


def sphericart_cuda_vjp_recompute(xyz, grad_sph, grad_xyz, n, l_max, normalized, dtype, stream):
    rc = load().sphericart_cuda_vjp_recompute(_ptr(xyz), _ptr(grad_sph), _ptr(grad_xyz), n, l_max,
                                              int(bool(normalized)), dtype, _ptr(stream))
    _check(rc, "sphericart_cuda_vjp_recompute")


def sphericart_cuda_compute_ex(xyz, n, l_max, normalized, dtype, axes, scale, sph, dsph, ddsph, stream):
    rc = load().sphericart_cuda_compute_ex(_ptr(xyz), n, l_max, int(normalized), dtype, int(axes), int(scale),
                                           _ptr(sph), _ptr(dsph), _ptr(ddsph), _ptr(stream))
    _check(rc, "sphericart_cuda_compute_ex")


def sphericart_cuda_vjp2(xyz, grad_sph, v, grad_grad_xyz, grad_grad_sph, n, l_max, normalized, dtype, stream):
    rc = load().sphericart_cuda_vjp2(_ptr(xyz), _ptr(grad_sph), _ptr(v), _ptr(grad_grad_xyz), _ptr(grad_grad_sph), n,
                                     l_max, int(bool(normalized)), dtype, _ptr(stream))
    _check(rc, "sphericart_cuda_vjp2")


def sphericart_cuda_expand(xyz, radial, seg_ptr, n_seg, l_max, n_rad, dtype, coeff, stream):
    rc = load().sphericart_cuda_expand(_ptr(xyz), _ptr(radial), _ptr(seg_ptr), n_seg, l_max, n_rad, dtype,
                                       _ptr(coeff), _ptr(stream))
    _check(rc, "sphericart_cuda_expand")


NOALLOC_MAX_POINTS = 32768   # SPHERICART_CUDA_NOALLOC_MAX_POINTS (include/sphericart_cuda.h)


def sphericart_cuda_vjp_noalloc(dsph, grad_sph, grad_xyz, n, l_max, dtype, stream):
    rc = load().sphericart_cuda_vjp_noalloc(_ptr(dsph), _ptr(grad_sph), _ptr(grad_xyz), n, l_max, dtype, _ptr(stream))
    _check(rc, "sphericart_cuda_vjp_noalloc")


def sphericart_cuda_vjp_host(xyz, dsph, grad_sph, grad_xyz, n, l_max, dtype):
    rc = load().sphericart_cuda_vjp_host(_ptr(xyz), _ptr(dsph), _ptr(grad_sph), _ptr(grad_xyz), n,
                                         l_max, dtype)
    _check(rc, "sphericart_cuda_vjp_host")


def sphericart_cuda_last_error() -> str:
    return load().sphericart_cuda_last_error().decode()


def sphericart_cuda_launch_count() -> int:
    return int(load().sphericart_cuda_launch_count())


def sphericart_cuda_last_kernel() -> str:
    return load().sphericart_cuda_last_kernel().decode()


def sphericart_cuda_set_option(name: str, value) -> None:
    rc = load().sphericart_cuda_set_option(str(name).encode(), str(value).encode())
    _check(rc, "sphericart_cuda_set_option")


# --- torch.Tensor convenience (allocation + marshalling only) -----------------------------------
def _dtype_code(t):
    import torch

    if t.dtype == torch.float32:
        return F32
    if t.dtype == torch.float64:
        return F64
    raise TypeError(f"unsupported dtype {t.dtype}: float32 or float64")


def _check_out(name, t, shape, like):
    """An output tensor handed in by the caller: right shape, dtype, device, dense."""
    if t is None:
        raise ValueError(f"out: {name} is missing")
    if tuple(t.shape) != tuple(shape) or t.dtype != like.dtype or t.device != like.device or not t.is_contiguous():
        raise ValueError(f"out: {name} must be a contiguous {like.dtype} tensor of shape {tuple(shape)} on {like.device}")
    return t


def compute(xyz, l_max: int, normalized: bool = True, gradients: bool = False, hessians: bool = False,
            out=None, axes: int = AXES_STANDARD, scale: int = SCALE_INTEGRAL):
    """``xyz`` [n,3] CUDA tensor -> ``(sph [n,L], dsph [n,3,L] | None, ddsph [n,3,3,L] | None)``.

    Enqueued on torch's current stream.  ``out`` may hold preallocated ``(sph, dsph, ddsph)``.
    ``axes`` / ``scale``: another convention (``sphericart_cuda_compute_ex``).
    """
    import torch

    if not xyz.is_cuda:
        raise SphericartCudaError("xyz must be a CUDA tensor (no CPU fallback)")
    if hessians and not gradients:
        raise ValueError("hessians need gradients")
    if xyz.dim() != 2 or xyz.shape[1] != 3:
        raise ValueError("xyz must have shape [n, 3]")
    if not 0 <= int(l_max) <= MAX_L:
        raise SphericartCudaError(f"l_max = {l_max} outside [0, {MAX_L}]")
    xyz = xyz.contiguous()
    n, L = xyz.shape[0], (l_max + 1) ** 2
    if out is None:
        sph = torch.empty((n, L), dtype=xyz.dtype, device=xyz.device)
        dsph = torch.empty((n, 3, L), dtype=xyz.dtype, device=xyz.device) if gradients else None
        ddsph = torch.empty((n, 3, 3, L), dtype=xyz.dtype, device=xyz.device) if hessians else None
    else:
        sph, dsph, ddsph = out
        _check_out("sph", sph, (n, L), xyz)
        dsph = _check_out("dsph", dsph, (n, 3, L), xyz) if gradients else None
        ddsph = _check_out("ddsph", ddsph, (n, 3, 3, L), xyz) if hessians else None
    with torch.cuda.device(xyz.device):
        stream = torch.cuda.current_stream().cuda_stream
        sphericart_cuda_compute_ex(xyz, n, l_max, normalized, _dtype_code(xyz), axes, scale, sph, dsph, ddsph, stream)
    return sph, dsph, ddsph


def vjp(dsph, grad_sph, out=None):
    """``grad_xyz[n,a] = sum_k dsph[n,a,k] grad_sph[n,k]`` on torch's current stream."""
    import torch

    if not dsph.is_cuda:
        raise SphericartCudaError("dsph must be a CUDA tensor (no CPU fallback)")
    dsph, grad_sph = dsph.contiguous(), grad_sph.contiguous()
    n, L = grad_sph.shape
    l_max = int(round(L ** 0.5)) - 1
    if (l_max + 1) ** 2 != L or dsph.shape != (n, 3, L) or dsph.dtype != grad_sph.dtype:
        raise ValueError("shapes: dsph [n,3,L], grad_sph [n,L], L a perfect square, same dtype")
    gx = torch.empty((n, 3), dtype=dsph.dtype, device=dsph.device) if out is None else _check_out("grad_xyz", out, (n, 3), dsph)
    with torch.cuda.device(dsph.device):
        stream = torch.cuda.current_stream().cuda_stream
        sphericart_cuda_vjp(None, dsph, grad_sph, gx, n, l_max, _dtype_code(dsph), stream)
    return gx


def vjp_recompute(xyz, grad_sph, normalized: bool, out=None):
    """``grad_xyz[n,a] = sum_k (d sph[n,k] / d xyz[n,a]) grad_sph[n,k]`` evaluated from ``xyz``
    (no stored derivatives), on torch's current stream."""
    import torch

    if not xyz.is_cuda:
        raise SphericartCudaError("xyz must be a CUDA tensor (no CPU fallback)")
    xyz, grad_sph = xyz.contiguous(), grad_sph.contiguous()
    n, L = grad_sph.shape
    l_max = int(round(L ** 0.5)) - 1
    if (l_max + 1) ** 2 != L or xyz.shape != (n, 3) or xyz.dtype != grad_sph.dtype:
        raise ValueError("shapes: xyz [n,3], grad_sph [n,L], L a perfect square, same dtype")
    gx = torch.empty((n, 3), dtype=xyz.dtype, device=xyz.device) if out is None else _check_out("grad_xyz", out, (n, 3), xyz)
    with torch.cuda.device(xyz.device):
        stream = torch.cuda.current_stream().cuda_stream
        sphericart_cuda_vjp_recompute(xyz, grad_sph, gx, n, l_max, normalized, _dtype_code(xyz), stream)
    return gx


def vjp2(xyz, grad_sph, v, normalized: bool, want_grad_grad_sph: bool = True):
    """Double backward from ``xyz``: ``(grad_grad_xyz [n,3], grad_grad_sph [n,L] | None)`` for the upstream
    gradient ``v`` [n,3] on ``vjp_recompute(xyz, grad_sph)`` (``sphericart_cuda_vjp2``)."""
    import torch

    if not xyz.is_cuda:
        raise SphericartCudaError("xyz must be a CUDA tensor (no CPU fallback)")
    xyz, grad_sph, v = xyz.contiguous(), grad_sph.contiguous(), v.contiguous()
    n, L = grad_sph.shape
    l_max = int(round(L ** 0.5)) - 1
    if (l_max + 1) ** 2 != L or xyz.shape != (n, 3) or v.shape != (n, 3) or not (xyz.dtype == grad_sph.dtype == v.dtype):
        raise ValueError("shapes: xyz [n,3], grad_sph [n,L], v [n,3], L a perfect square, same dtype")
    ggx = torch.empty((n, 3), dtype=xyz.dtype, device=xyz.device)
    ggs = torch.empty((n, L), dtype=xyz.dtype, device=xyz.device) if want_grad_grad_sph else None
    with torch.cuda.device(xyz.device):
        stream = torch.cuda.current_stream().cuda_stream
        sphericart_cuda_vjp2(xyz, grad_sph, v, ggx, ggs, n, l_max, normalized, _dtype_code(xyz), stream)
    return ggx, ggs


def expand(xyz, radial, seg_ptr, out=None):
    """``coeff[s,n,lm] = sum_{k in segment s} radial[k,n,l] Y_lm(xyz[k]/|xyz[k]|)`` (Eq. 1 of the paper)
    on torch's current stream; ``seg_ptr`` an int64 CUDA tensor of ascending offsets."""
    import torch

    if not xyz.is_cuda:
        raise SphericartCudaError("xyz must be a CUDA tensor (no CPU fallback)")
    xyz, radial, seg_ptr = xyz.contiguous(), radial.contiguous(), seg_ptr.contiguous()
    n, n_rad, lp1 = radial.shape
    if xyz.shape != (n, 3) or xyz.dtype != radial.dtype or seg_ptr.dtype != torch.int64:
        raise ValueError("shapes: xyz [n,3], radial [n,n_rad,l_max+1] of the same dtype, seg_ptr int64")
    n_seg, L = seg_ptr.numel() - 1, lp1 * lp1
    if n_seg < 0 or (n_seg >= 0 and seg_ptr.numel() and int(seg_ptr[-1]) != n) or (seg_ptr.numel() and int(seg_ptr[0]) != 0):
        raise ValueError("seg_ptr must run from 0 to the number of points")
    c = (torch.empty((n_seg, n_rad, L), dtype=xyz.dtype, device=xyz.device) if out is None
         else _check_out("coeff", out, (n_seg, n_rad, L), xyz))
    with torch.cuda.device(xyz.device):
        stream = torch.cuda.current_stream().cuda_stream
        sphericart_cuda_expand(xyz, radial, seg_ptr, n_seg, lp1 - 1, n_rad, _dtype_code(xyz), c, stream)
    return c
