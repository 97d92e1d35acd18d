"""Parity metric shared by the GPU tests.

north_star: "relative error <= 1e-12 in f64 and <= 5e-6*(l_max+1) in f32 (absolute where
|Y| < 1e-3)".  Reading R1 makes the 1e-3 floor relative to the row scale so that it also means
something for solid harmonics (size r^l) and for derivatives (size l/r, l^2/r^2):

    S_d = sqrt((2l+1)/4pi) * rho * max(l,1)^d / r^d,   rho = 1 (normalised) or r^l (solid)
    e   = |got - oracle| / max(|oracle|, 1e-3 * S_d)          PASS iff max e <= tol

S_0 is exactly the 2-norm of the l-row (addition theorem).  For normalised values S_0 = O(1) and
this IS the literal rule.  ``strict`` counts violations of the literal, unscaled rule for the record.

Underflow (reading U1): solid harmonics of a point with r ~ 1e-5 are ~r^l, below the
smallest normal number of the output type (f32: 1.18e-38) already at l = 8; there the output type
has no relative precision to offer, so the floor never drops below ``finfo(dtype).tiny``.
"""
from __future__ import annotations

import math

import numpy as np

LD = np.longdouble


def tol_for(dtype: str, l_max: int) -> float:
    return 1e-12 if dtype == "f64" else 5e-6 * (l_max + 1)


def l_of_k(l_max: int) -> np.ndarray:
    return np.concatenate([[l] * (2 * l + 1) for l in range(l_max + 1)])


def row_scales(xyz, l_max: int, normalized: bool, order: int) -> np.ndarray:
    """S_order for every (point, k): shape [n, L] (long double)."""
    x = np.asarray(xyz, LD)
    r = np.sqrt((x * x).sum(axis=1))
    l = l_of_k(l_max).astype(LD)
    base = np.sqrt((2 * l + 1) / (4 * LD(math.pi)))[None, :]
    lam = np.maximum(l, 1)[None, :]
    if normalized:
        with np.errstate(divide="ignore"):
            return base * (lam / r[:, None]) ** order
    # solid: r^l / r^order as ONE power so that r = 0 gives 0 or 1, not 0 * inf; a derivative of
    # order > l of a degree-l polynomial is identically zero, hence the clamp of the exponent
    return base * lam ** order * r[:, None] ** np.maximum(l - order, 0)[None, :]


def errors(got, want, xyz, l_max: int, normalized: bool, order: int, tiny: float = 0.0):
    """Return (max scaled-floor error e, number of strict-rule violations at tol=1, max strict e).

    got / want: [n, (3,)*order, L].  Points whose oracle value is non-finite (r = 0, normalised)
    must be non-finite in ``got`` too and are excluded from the maximum.
    """
    got = np.asarray(got).astype(LD)
    want = np.asarray(want).astype(LD)
    S = row_scales(xyz, l_max, normalized, order)
    S = S.reshape((S.shape[0],) + (1,) * order + (S.shape[1],))
    bad = ~np.isfinite(want)
    if bad.any():
        assert np.all(~np.isfinite(got[bad])), "GPU finite where the oracle is not"
    diff = np.abs(np.where(bad, 0, got - want))
    aw = np.abs(np.where(bad, 1, want))
    e = diff / np.maximum(np.maximum(aw, LD(1e-3) * S), LD(tiny))
    e = np.where(np.isfinite(e), e, np.where(diff == 0, 0, np.inf))   # S = 0 (r = 0 solid, l >= 1): exact zeros
    strict = diff / np.maximum(aw, LD(1e-3))
    return float(e.max(initial=0)), strict, e


def check(got, want, xyz, l_max, normalized, order, dtype, what=""):
    tol = tol_for(dtype, l_max)
    tiny = float(np.finfo(np.float32 if dtype == "f32" else np.float64).tiny)
    emax, strict, e = errors(got, want, xyz, l_max, normalized, order, tiny)
    n_strict = int((strict > tol).sum())
    msg = (f"{what}: max scaled error {emax:.3e} (tol {tol:.1e}); strict-rule violations "
           f"{n_strict} of {strict.size}, max {float(strict.max(initial=0)):.3e}")
    assert emax <= tol, msg
    return emax, n_strict, msg


def check_vjp(got, want, dsph, grad_sph, l_max, dtype, what="vjp", point_scale=False):
    """|err| / max(|ref|, 1e-3 * ||dsph[n,a,:]||_2 ||grad_sph[n,:]||_2) <= tol (SURVEY 8(c) VJP).

    ``point_scale``: the floor uses max_a ||dsph[n,a,:]||_2 instead (reading R3, used for
    the recompute route: like R1's row scale S_1 it does not depend on the component a, so a
    component whose derivatives all vanish identically -- d/dz of normalised Y for a point ON the z
    axis -- is held to the size of that point's gradient, not to an exact zero)."""
    tol = tol_for(dtype, l_max)
    got = np.asarray(got).astype(LD)
    want = np.asarray(want).astype(LD)
    d = np.asarray(dsph).astype(LD)
    g = np.asarray(grad_sph).astype(LD)
    dn = np.sqrt((d * d).sum(axis=2))
    if point_scale:
        dn = np.broadcast_to(dn.max(axis=1, keepdims=True), dn.shape)
    scale = dn * np.sqrt((g * g).sum(axis=1))[:, None]
    diff = np.abs(got - want)
    with np.errstate(invalid="ignore", divide="ignore"):
        e = diff / np.maximum(np.abs(want), LD(1e-3) * scale)
    # scale = 0 (every d/dx_a vanishes, e.g. d/dz of normalised Y for a point ON the z axis): the
    # reference is an exact zero and only an exact zero passes
    e = np.where(np.isfinite(e), e, np.where(diff == 0, 0, np.inf))
    emax = float(e.max(initial=0))
    assert emax <= tol, f"{what}: max scaled error {emax:.3e} (tol {tol:.1e})"
    return emax


def check_expand(got, want, radial, seg_ptr, l_max, dtype, what="expand"):
    """Density expansion (Eq. 1): |err| / max(|ref|, 1e-3 S) <= tol with the scale of one row of the
    sum, S[s,n,l] = sqrt((2l+1)/4pi) * sum_{k in s} |R[k,n,l]|  (R1's row scale S_0 weighted by the
    radial values: the size the terms have before they cancel).  Empty segments must be exact zeros."""
    tol = tol_for(dtype, l_max)
    got = np.asarray(got).astype(LD)
    want = np.asarray(want).astype(LD)
    R = np.abs(np.asarray(radial).astype(LD))
    n_seg = len(seg_ptr) - 1
    l_of = np.concatenate([[l] * (2 * l + 1) for l in range(l_max + 1)])
    S = np.zeros_like(want)
    for s_ in range(n_seg):
        S[s_] = R[seg_ptr[s_]:seg_ptr[s_ + 1]].sum(axis=0)[:, l_of]
    S *= np.sqrt((2 * l_of + 1) / (4 * np.pi)).astype(LD)[None, None, :]
    diff = np.abs(got - want)
    with np.errstate(invalid="ignore", divide="ignore"):
        e = diff / np.maximum(np.abs(want), LD(1e-3) * S)
    e = np.where(np.isfinite(e), e, np.where(diff == 0, 0, np.inf))
    emax = float(e.max(initial=0))
    assert emax <= tol, f"{what}: max scaled error {emax:.3e} (tol {tol:.1e})"
    return emax
