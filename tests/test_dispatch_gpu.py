"""`-m gpu`: every kernel the DEFAULT dispatch can reach, against the oracle, element by element.

The forward entry point picks among separately compiled instantiations (one per l_max, element
type and derivative order, each with its own tile split, padding and store path), so every
(dtype, l_max, derivative order, variant) cell is run here with no kernel family forced:
whatever kernel `sphericart_cuda_compute` chooses for that cell is the one compared.
The same for the recompute VJP and the fused expansion.  n spans several tiles plus a ragged
tail; C2-style special points (on +-z, |r| down to 1e-6) for l_max <= 16, C4-style shells above.
Equations checked: Eq. 5, Eq. 7, Eq. 9, Eq. 10, chain rule P:108,
backward P:112, Eq. 1.
"""
import numpy as np
import pytest

import parity
from paper_2302_08381_b200 import workloads as W

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def sph():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2302_08381_b200 as pkg

    pkg.load()
    pkg.sphericart_cuda_set_option("force_kernel", "auto")     # this file tests the default dispatch
    return pkg


def _cloud(l_max, n, dtype):
    xyz = W.make_xyz("C2" if l_max <= 16 else "C4", n, seed=l_max)
    return np.ascontiguousarray(xyz.astype(np.float32 if dtype == "f32" else np.float64))


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("l_max", list(range(0, 33)))
def test_default_dispatch_every_cell(sph, oracle, dtype, l_max):
    n = 3 * 32 + 100 + 7 if l_max <= 16 else 2 * 32 + 7        # C2 cloud: >= 2 axis and 2 tiny-r points
    xyz = _cloud(l_max, n, dtype)
    x_d = torch.from_numpy(xyz).cuda()
    for normalized in (True, False):
        want = oracle.compute(xyz, l_max, normalized, True, True)
        for deriv in (0, 1, 2):
            before = sph.sphericart_cuda_launch_count()
            got = sph.compute(x_d, l_max, normalized, deriv >= 1, deriv >= 2)
            torch.cuda.synchronize()
            assert sph.sphericart_cuda_launch_count() == before + 1
            for order in range(deriv + 1):
                parity.check(got[order].cpu().numpy(), want[order], xyz, l_max, normalized, order, dtype,
                             f"{dtype} l_max={l_max} norm={normalized} deriv={deriv} order={order}")
            if deriv == 2:
                hh = got[2]
                for a in range(3):
                    for b in range(a):
                        assert torch.equal(hh[:, a, b], hh[:, b, a])


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("l_max", list(range(0, 33)))
def test_default_dispatch_vjp_recompute(sph, oracle, dtype, l_max):
    n = 3 * 32 + 100 + 7 if l_max <= 16 else 2 * 32 + 7
    xyz = _cloud(l_max, n, dtype)
    g = np.random.default_rng([7, l_max]).standard_normal((n, (l_max + 1) ** 2)).astype(xyz.dtype)
    x_d, g_d = torch.from_numpy(xyz).cuda(), torch.from_numpy(g).cuda()
    for normalized in (True, False):
        before = sph.sphericart_cuda_launch_count()
        gx = sph.vjp_recompute(x_d, g_d, normalized)
        torch.cuda.synchronize()
        assert sph.sphericart_cuda_launch_count() == before + 1
        _, wd, _ = oracle.compute(xyz, l_max, normalized, True)
        parity.check_vjp(gx.cpu().numpy(), oracle.vjp_recompute(xyz, g, l_max, normalized), wd, g, l_max, dtype,
                         f"vjp_recompute {dtype} l_max={l_max} norm={normalized}", point_scale=True)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("l_max", list(range(0, 17)) + [20, 25, 32])
def test_default_dispatch_expand(sph, oracle, dtype, l_max):
    for n_rad in (1, 7, 8, 9, 16, 17, 32):
        xyz, rad, seg = W.make_expand_inputs(37, l_max, n_rad, dtype, 19.0, seed=n_rad)
        before = sph.sphericart_cuda_launch_count()
        c = sph.expand(torch.from_numpy(xyz).cuda(), torch.from_numpy(rad).cuda(), torch.from_numpy(seg).cuda())
        torch.cuda.synchronize()
        assert sph.sphericart_cuda_launch_count() == before + 1
        parity.check_expand(c.cpu().numpy(), oracle.expand(xyz, rad, seg, l_max), rad, seg, l_max, dtype,
                            f"expand {dtype} l_max={l_max} n_rad={n_rad}")


@pytest.mark.parametrize("dtype,l_max,deriv", [("f32", 12, 1), ("f32", 16, 1), ("f32", 9, 2), ("f64", 12, 1), ("f64", 10, 2),
                                               ("f64", 14, 0), ("f32", 28, 0), ("f64", 20, 1), ("f32", 20, 2)])
def test_sweep_cells_at_bench_size(sph, oracle, dtype, l_max, deriv):
    """Cells of the l_max sweep at the size and launch configuration bench.py times them in (n sized for
    ~1.5 GB of output, at least 256 points per SM: several batches per CTA, every SM busy), default dispatch: sampled points against the
    oracle (first / last points and tile edges included) and, on EVERY point, properties that hold at any
    size: the addition theorem sum_m Y_lm^2 = (2l+1)/4pi, Euler's x . grad Y = 0 for the normalised
    harmonics, and trace(Hessian) = -l(l+1) Y / r^2."""
    es = 4 if dtype == "f32" else 8
    L = (l_max + 1) ** 2
    per_pt = L * es * (1, 4, 13)[deriv]
    import bench

    n = bench.lmax_cell_points(per_pt) + 37          # bench.py's size for the cell + a ragged tail
    tdt = torch.float32 if dtype == "f32" else torch.float64
    g = torch.Generator(device="cuda").manual_seed(1000 + l_max)
    x_d = torch.randn(n, 3, device="cuda", dtype=tdt, generator=g)
    before = sph.sphericart_cuda_launch_count()
    got = sph.compute(x_d, l_max, True, deriv >= 1, deriv >= 2)
    torch.cuda.synchronize()
    assert sph.sphericart_cuda_launch_count() == before + 1
    rng = np.random.default_rng(l_max)
    idx = np.unique(np.concatenate([rng.integers(0, n, 400 if deriv < 2 else 150),
                                    [0, 1, 2, 3, 15, 16, 31, 32, 33, n - 38, n - 37, n - 33, n - 2, n - 1]]))
    it = torch.from_numpy(idx).cuda()
    xyz = x_d.index_select(0, it).cpu().numpy()
    want = oracle.compute(xyz, l_max, True, deriv >= 1, deriv >= 2)
    for order in range(deriv + 1):
        parity.check(got[order].index_select(0, it).cpu().numpy(), want[order], xyz, l_max, True, order, dtype,
                     f"bench-size {dtype} l_max={l_max} deriv={deriv} order={order} ({sph.sphericart_cuda_last_kernel()})")
    # whole-array properties, in f64 on the device, in chunks
    eps = 1.2e-7 if dtype == "f32" else 2.3e-16
    lt = torch.from_numpy(parity.l_of_k(l_max)).cuda()
    lv = torch.arange(l_max + 1, device="cuda", dtype=torch.float64)
    for a in range(0, n, 65536):
        sl = slice(a, min(a + 65536, n))
        Y = got[0][sl].double()
        rows = torch.zeros((Y.shape[0], l_max + 1), dtype=torch.float64, device="cuda").index_add_(1, lt, Y * Y)
        rel = (rows / ((2 * lv + 1) / (4 * np.pi)) - 1).abs().max()
        assert float(rel) < 8 * (l_max + 1) * eps, f"addition theorem off by {float(rel):.3e}"
        if deriv >= 1:
            X = x_d[sl].double()
            r = X.norm(dim=1)
            G = got[1][sl].double()
            xg = torch.einsum("na,nak->nk", X, G)                      # = 0; scale: r |grad| ~ l
            assert float(xg.abs().max()) < 64 * (l_max + 1) ** 1.5 * eps, f"x.grad Y = {float(xg.abs().max()):.3e}"
        if deriv >= 2:
            H = got[2][sl].double()
            tr = H[:, 0, 0] + H[:, 1, 1] + H[:, 2, 2]
            res = tr + (lt * (lt + 1)).double()[None, :] * Y / (r * r)[:, None]
            scale = ((l_max + 1) ** 2.5) / (r * r)[:, None]
            assert float((res.abs() / scale).max()) < 64 * eps, f"trace(H) + l(l+1) Y / r^2: {float((res.abs() / scale).max()):.3e}"
