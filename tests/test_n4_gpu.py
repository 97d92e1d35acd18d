"""`-m gpu`: SURVEY 8(f) N4 on the GPU against the oracle -- the forward pass in the e3nn axis /
component / norm scale conventions (`sphericart_cuda_compute_ex`) and the second-order VJP
(`sphericart_cuda_vjp2`: double backward) -- and the recompute VJP through the
two-phase kernel at every l_max (N1)."""
import numpy as np
import pytest

import parity
from paper_2302_08381_b200 import workloads as W

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
LD = np.longdouble


@pytest.fixture(scope="module")
def sph():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2302_08381_b200 as pkg

    pkg.load()
    pkg.sphericart_cuda_set_option("force_kernel", "auto")
    return pkg


def _l_scale(oracle, scale, l_max):
    l = parity.l_of_k(l_max).astype(LD)
    four_pi = 16 * np.arctan(LD(1))
    return {oracle.SCALE_INTEGRAL: np.ones_like(l), oracle.SCALE_COMPONENT: np.sqrt(four_pi) * np.ones_like(l),
            oracle.SCALE_NORM: np.sqrt(four_pi / (2 * l + 1))}[scale]


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("l_max", [0, 1, 2, 5, 8, 11, 16, 21, 28, 32])
def test_conventions(sph, oracle, dtype, l_max):
    """Every (axes, scale) pair but the paper's own, every derivative order, both variants; the rows
    are divided by their scale before the tolerance is applied, so the metric is the one of
    tests/parity.py."""
    n = 150 if l_max <= 16 else 39
    xyz = W.make_xyz("C2" if l_max <= 16 else "C4", n, seed=100 + l_max).astype(np.float32 if dtype == "f32" else np.float64)
    x_d = torch.from_numpy(xyz).cuda()
    for axes, scale in ((oracle.AXES_E3NN, oracle.SCALE_INTEGRAL), (oracle.AXES_E3NN, oracle.SCALE_COMPONENT),
                        (oracle.AXES_E3NN, oracle.SCALE_NORM), (oracle.AXES_STANDARD, oracle.SCALE_NORM)):
        sc = _l_scale(oracle, scale, l_max)
        for normalized in (True, False):
            want = oracle.compute_convention(xyz, l_max, normalized, axes, scale, True, True)
            for deriv in (0, 1, 2):
                before = sph.sphericart_cuda_launch_count()
                got = sph.compute(x_d, l_max, normalized, deriv >= 1, deriv >= 2, axes=axes, scale=scale)
                torch.cuda.synchronize()
                assert sph.sphericart_cuda_launch_count() == before + 1
                for order in range(deriv + 1):
                    parity.check(got[order].cpu().numpy().astype(LD) / sc, want[order] / sc, xyz, l_max, normalized, order,
                                 dtype, f"conv axes={axes} scale={scale} {dtype} l_max={l_max} norm={normalized} order={order}")


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("l_max", [0, 1, 2, 3, 6, 9, 12, 16, 20, 27, 32])
def test_vjp2_double_backward(sph, oracle, dtype, l_max):
    """grad_grad_xyz and grad_grad_sph against oracle.vjp2 (compute with Hessians + plain contractions);
    floors as for the first-order VJP (tests/parity.py), with the Hessian rows for grad_grad_xyz."""
    n = 3 * 32 + 7 if l_max <= 16 else 41
    xyz = W.make_xyz("C2" if l_max <= 16 else "C4", n, seed=200 + l_max).astype(np.float32 if dtype == "f32" else np.float64)
    rng = np.random.default_rng([9, l_max])
    L = (l_max + 1) ** 2
    w = rng.standard_normal((n, L)).astype(xyz.dtype)
    v = rng.standard_normal((n, 3)).astype(xyz.dtype)
    x_d, w_d, v_d = (torch.from_numpy(a).cuda() for a in (xyz, w, v))
    tol = parity.tol_for(dtype, l_max)
    for normalized in (True, False):
        before = sph.sphericart_cuda_launch_count()
        ggx, ggs = sph.vjp2(x_d, w_d, v_d, normalized)
        torch.cuda.synchronize()
        assert sph.sphericart_cuda_launch_count() == before + 1 and sph.sphericart_cuda_last_kernel() == "tq_vjp2"
        want_x, want_w = oracle.vjp2(xyz, w, v, l_max, normalized)
        _, d, h = oracle.compute(xyz, l_max, normalized, True, True)
        # grad_grad_sph[k] = sum_a dsph[a,k] v_a: |err| / max(|ref|, 1e-3 S_1 |v|) with R1's row scale S_1 of
        # the gradients (reading R4: a harmonic whose gradient vanishes identically at a point --
        # m = 0 on the z axis -- is held to the size of its degree's gradients there, not to an exact zero)
        S1 = parity.row_scales(xyz, l_max, normalized, 1)
        sw = 1e-3 * S1 * np.sqrt((v.astype(LD) ** 2).sum(axis=1))[:, None]
        tiny = float(np.finfo(np.float32 if dtype == "f32" else np.float64).tiny)      # (reading U1)
        e = np.abs(ggs.cpu().numpy().astype(LD) - want_w) / np.maximum(np.maximum(np.abs(want_w), sw), tiny)
        e = np.where(np.isfinite(e), e, 0)
        assert float(e.max()) <= tol, f"grad_grad_sph {dtype} l_max={l_max} norm={normalized}: {float(e.max()):.3e}"
        # grad_grad_xyz[b] = sum_{a,k} ddsph[a,b,k] v_a w_k
        hn = np.sqrt((h * h).sum(axis=3)).max(axis=(1, 2))
        sx = 1e-3 * hn * np.sqrt((v.astype(LD) ** 2).sum(axis=1)) * np.sqrt((w.astype(LD) ** 2).sum(axis=1))
        e = np.abs(ggx.cpu().numpy().astype(LD) - want_x) / np.maximum(np.maximum(np.abs(want_x), sx[:, None]), tiny)
        e = np.where(np.isfinite(e), e, 0)
        assert float(e.max()) <= tol, f"grad_grad_xyz {dtype} l_max={l_max} norm={normalized}: {float(e.max()):.3e}"
        # grad_grad_sph is optional
        ggx2, none = sph.vjp2(x_d, w_d, v_d, normalized, want_grad_grad_sph=False)
        assert none is None and torch.equal(ggx2, ggx)


def test_vjp2_matches_finite_differences_of_the_gpu_backward(sph):
    """Independent of the oracle: central differences of the GPU's own recompute VJP in f64."""
    l_max, n = 7, 64
    xyz = torch.from_numpy(W.make_xyz("C4", n)).cuda()
    rng = np.random.default_rng(3)
    w = torch.from_numpy(rng.standard_normal((n, (l_max + 1) ** 2))).cuda()
    v = torch.from_numpy(rng.standard_normal((n, 3))).cuda()
    ggx, _ = sph.vjp2(xyz, w, v, True)
    h = 1e-5
    for b in range(3):
        e = torch.zeros_like(xyz)
        e[:, b] = h
        fp = (sph.vjp_recompute(xyz + e, w, True) * v).sum(dim=1)
        fm = (sph.vjp_recompute(xyz - e, w, True) * v).sum(dim=1)
        fd = (fp - fm) / (2 * h)
        assert float(((fd - ggx[:, b]).abs() / (ggx.abs().max() + 1)).max()) < 1e-6


@pytest.mark.parametrize("dtype,l_max", [("f32", 16), ("f64", 13), ("f32", 9)])
def test_contracting_modes_at_bench_size(sph, dtype, l_max):
    """The recompute VJP and the second-order VJP at a size that gives every CTA several batches (the launch
    configuration bench.py's sweep.backward times): EVERY point against the stored derivatives of the forward
    kernels contracted by torch in f64."""
    tdt = torch.float32 if dtype == "f32" else torch.float64
    L = (l_max + 1) ** 2
    n = 148 * 16 * 32 * 3 // (2 if l_max > 12 else 1) + 21
    g = torch.Generator(device="cuda").manual_seed(77 + l_max)
    x = torch.randn(n, 3, device="cuda", dtype=tdt, generator=g)
    w = torch.randn(n, L, device="cuda", dtype=tdt, generator=g)
    v = torch.randn(n, 3, device="cuda", dtype=tdt, generator=g)
    _, d, h = sph.compute(x, l_max, True, True, True)
    tol = (2e-5 if dtype == "f32" else 1e-11)
    gx = sph.vjp_recompute(x, w, True)
    ref = torch.einsum("nak,nk->na", d.double(), w.double())
    scale = d.double().norm(dim=2).max(dim=1, keepdim=True).values * w.double().norm(dim=1, keepdim=True)
    assert float(((gx.double() - ref).abs() / scale).max()) < tol
    ggx, ggs = sph.vjp2(x, w, v, True)
    assert sph.sphericart_cuda_last_kernel() == "tq_vjp2"
    ref_s = torch.einsum("nak,na->nk", d.double(), v.double())
    scale_s = d.double().norm(dim=1).max(dim=1, keepdim=True).values * v.double().norm(dim=1, keepdim=True)
    assert float(((ggs.double() - ref_s).abs() / scale_s).max()) < tol
    ref_x = torch.zeros((n, 3), dtype=torch.float64, device="cuda")
    for a in range(3):                                    # (chunked over a: h is the large tensor)
        ref_x += torch.einsum("nbk,nk->nb", h[:, a].double(), w.double()) * v[:, a:a + 1].double()
    scale_x = h.double().norm(dim=3).amax(dim=(1, 2))[:, None] * w.double().norm(dim=1, keepdim=True) * v.double().norm(dim=1, keepdim=True)
    assert float(((ggx.double() - ref_x).abs() / scale_x).max()) < tol
