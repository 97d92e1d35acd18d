"""Seeded synthetic inputs for the five BASELINE.json configurations (C1..C5).

This module holds NO arithmetic of the method (no F, Q, c, s, Y): only random point clouds.  It
is the one module that the CUDA path's harness (tests, bench.py) and the oracle's harness both
import, so both sides receive bit-identical inputs.

Recipe.  The paper times random batches of 10k / 100k points
 and names no dataset, so these clouds are the workload itself, not a
stand-in for a public benchmark.  Everything is generated in f64 with
``numpy.random.default_rng([cfg_id, seed])`` on the host, cast to the configuration's dtype, and
the CAST values are what both the GPU and the oracle get.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Config:
    name: str
    n: int
    dtype: str          # "f32" | "f64"
    l_max: int
    normalized: bool
    gradients: bool
    hessians: bool
    vjp: bool           # forward is followed by the backward contraction (C5)
    what: str

    @property
    def n_sph(self) -> int:
        return (self.l_max + 1) ** 2

    @property
    def itemsize(self) -> int:
        return 4 if self.dtype == "f32" else 8

    @property
    def np_dtype(self):
        return np.float32 if self.dtype == "f32" else np.float64

    @property
    def out_bytes_per_point(self) -> int:
        """Algorithmic output bytes of the forward call per point."""
        comps = 1 + (3 if self.gradients else 0) + (9 if self.hessians else 0)
        return comps * self.n_sph * self.itemsize

    @property
    def in_bytes_per_point(self) -> int:
        return 3 * self.itemsize


CONFIGS = {
    "C1": Config("C1", 1_000, "f64", 4, True, True, False, False,
                 "N=1000 f64 l_max=4 normalized Y+grad, xyz~N(0,1)"),
    "C2": Config("C2", 100_000, "f32", 8, True, True, False, False,
                 "N=100000 f32 l_max=8 normalized Y+grad, 98% N(0,1) + 1% on +-z + 1% |r| in [1e-6,1e-4]"),
    "C3": Config("C3", 1_000_000, "f32", 16, False, False, False, False,
                 "N=1000000 f32 l_max=16 solid r^l Y values only, uniform in ball R=5"),
    "C4": Config("C4", 262_144, "f64", 32, True, True, True, False,
                 "N=262144 f64 l_max=32 normalized Y+grad+Hessian, uniform directions, r~U[0.5,2]"),
    "C5": Config("C5", 4_000_000, "f32", 6, True, True, False, True,
                 "N=4000000 f32 l_max=6 normalized Y+grad then VJP, xyz~N(0,1), grad_sph~N(0,1)"),
}


def _directions(rng, n):
    """Uniform directions on the unit sphere (normalised Gaussian vectors)."""
    d = rng.standard_normal((n, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    return d


def make_xyz(cfg: Config | str, n: int | None = None, seed: int = 0) -> np.ndarray:
    """Point cloud of configuration ``cfg`` ([n,3], the configuration's dtype).

    ``n`` overrides the configuration's point count (same distribution; used for the reduced
    sizes the oracle finishes in seconds).
    """
    if isinstance(cfg, str):
        cfg = CONFIGS[cfg]
    n = cfg.n if n is None else int(n)
    cid = int(cfg.name[1:])
    rng = np.random.default_rng(seed if cid == 1 else [cid, seed])  # C1: "seed 0" as given
    if cfg.name in ("C1", "C5", "C9"):       # C9: bench.py's `--workload custom` (any dtype / l_max / outputs)
        xyz = rng.standard_normal((n, 3))
    elif cfg.name == "C2":
        n_axis = n // 100                      # 1 % exactly on the +-z axis
        n_tiny = n // 100                      # 1 % with |r| in [1e-6, 1e-4]
        n_bulk = n - n_axis - n_tiny
        bulk = rng.standard_normal((n_bulk, 3))
        axis = np.zeros((n_axis, 3))
        axis[:, 2] = (0.1 + np.abs(rng.standard_normal(n_axis))) * rng.choice([-1.0, 1.0], n_axis)
        rho = 10.0 ** rng.uniform(-6.0, -4.0, n_tiny)      # log-uniform radius
        tiny = _directions(rng, n_tiny) * rho[:, None]
        xyz = np.concatenate([bulk, axis, tiny], axis=0)
        xyz = xyz[rng.permutation(n)]          # scatter the special points across warps
    elif cfg.name == "C3":
        xyz = _directions(rng, n) * (5.0 * rng.uniform(0.0, 1.0, n) ** (1.0 / 3.0))[:, None]
    elif cfg.name == "C4":
        xyz = _directions(rng, n) * rng.uniform(0.5, 2.0, n)[:, None]
    else:
        raise KeyError(cfg.name)
    return np.ascontiguousarray(xyz.astype(cfg.np_dtype))


def make_grad_sph(cfg: Config | str, n: int | None = None, seed: int = 0) -> np.ndarray:
    """Upstream gradient for the VJP ([n,L], i.i.d. N(0,1), the configuration's dtype)."""
    if isinstance(cfg, str):
        cfg = CONFIGS[cfg]
    n = cfg.n if n is None else int(n)
    rng = np.random.default_rng([100 + int(cfg.name[1:]), seed])
    # generated in f32 directly for f32 configs (4e6 x 49 would be 1.5 GB in f64)
    if cfg.dtype == "f32":
        return rng.standard_normal((n, cfg.n_sph), dtype=np.float32)
    return rng.standard_normal((n, cfg.n_sph))


def make_expand_inputs(n_seg: int, l_max: int, n_rad: int, dtype: str = "f32", mean_neighbours: float = 32.0,
                       seed: int = 0):
    """Synthetic input of the density expansion of Eq. 1, shaped like an atomistic
    neighbour list: ``n_seg`` centres with Poisson(``mean_neighbours``) neighbours each (some
    centres have none), neighbour vectors uniform in a ball of radius 5 (as C3), radial values
    i.i.d. N(0,1) -- the paper fixes no radial basis, so they are plain numbers here.
    Returns ``(xyz [N,3], radial [N,n_rad,l_max+1], seg_ptr [n_seg+1] int64)``."""
    rng = np.random.default_rng([200 + l_max, n_rad, seed])
    counts = rng.poisson(mean_neighbours, size=n_seg).astype(np.int64)
    seg_ptr = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    n = int(seg_ptr[-1])
    d = rng.standard_normal((n, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    xyz = d * (5.0 * rng.random(n) ** (1.0 / 3.0))[:, None]
    np_dt = np.float32 if dtype == "f32" else np.float64
    radial = rng.standard_normal((n, n_rad, l_max + 1)).astype(np_dt)
    return xyz.astype(np_dt), radial, seg_ptr
