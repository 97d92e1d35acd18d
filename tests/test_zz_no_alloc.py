"""`-m gpu`: `sphericart_cuda_vjp_noalloc`, the stored-derivative VJP that allocates nothing.

Its scratch is a file-scope `static __device__` array of the library (include/sphericart_cuda.h states
the size and the limit on n), so it serves callers that must not call cudaMalloc.  Checked here against
the EXISTING path, `sphericart_cuda_vjp`, on the same device buffers, within the VJP tolerance of the
other tests (tests/parity.py::check_vjp: |err| / max(|ref|, 1e-3 ||dsph|| ||grad_sph||) <= 1e-12 in f64,
5e-6 (l_max + 1) in f32) -- on TWO calls in a row with different sizes and inputs: the second call
finds the first one's partial sums in the shared scratch and must not be affected by them.  Collected
last (file name): the suite runs with `pytest -x`.  Passes alone in a fresh process and after the rest.
"""
import pytest

import parity

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def sph():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2302_08381_b200 as pkg

    pkg.load()
    pkg.sphericart_cuda_set_option("force_kernel", "auto")
    return pkg


def _inputs(n, l_max, dtype, seed):
    """dsph as the forward pass writes it (normalised harmonics of N(0,1) points), grad_sph ~ N(0,1)."""
    L = (l_max + 1) ** 2
    g = torch.Generator(device="cuda").manual_seed(seed)
    xyz = torch.randn(n, 3, device="cuda", dtype=dtype, generator=g)
    grad_sph = torch.randn(n, L, device="cuda", dtype=dtype, generator=g)
    return xyz, grad_sph


def _both(sph, dsph, grad_sph, l_max, dt_code):
    n = grad_sph.shape[0]
    st = torch.cuda.current_stream().cuda_stream
    want = torch.full((n, 3), float("nan"), device="cuda", dtype=grad_sph.dtype)
    got = torch.full((n, 3), float("nan"), device="cuda", dtype=grad_sph.dtype)
    sph.sphericart_cuda_vjp(None, dsph, grad_sph, want, n, l_max, dt_code, st)       # the existing path
    before = sph.sphericart_cuda_launch_count()
    sph.sphericart_cuda_vjp_noalloc(dsph, grad_sph, got, n, l_max, dt_code, st)
    assert sph.sphericart_cuda_launch_count() == before + 2                         # split + sum, both this library's
    assert sph.sphericart_cuda_last_kernel() == "vjp_split_sum"
    torch.cuda.synchronize()
    return got, want


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_vjp_noalloc_matches_vjp_on_two_calls_in_a_row(sph, dtype):
    tdt = torch.float32 if dtype == "f32" else torch.float64
    code = sph.F32 if dtype == "f32" else sph.F64
    # first call: long rows, few points (8 slices per row); second: shorter rows, more points, ragged
    # sizes (fewer slices, another layout of the same scratch); then the first again
    calls = [(257, 32, 1), (5003, 9, 2), (257, 32, 3), (1, 20, 4), (3000, 0, 5), (777, 3, 6)]
    for n, l_max, seed in calls:
        xyz, grad_sph = _inputs(n, l_max, tdt, seed)
        _, dsph, _ = sph.compute(xyz, l_max, True, True, False)
        got, want = _both(sph, dsph, grad_sph, l_max, code)
        assert bool(torch.isfinite(got).all())
        parity.check_vjp(got.cpu().numpy(), want.double().cpu().numpy(), dsph.cpu().numpy(), grad_sph.cpu().numpy(),
                         l_max, dtype, f"vjp_noalloc {dtype} n={n} l_max={l_max}")
    # the same call twice: bit-identical (fixed summation order, no dependence on the scratch's contents)
    xyz, grad_sph = _inputs(1234, 16, tdt, 7)
    _, dsph, _ = sph.compute(xyz, 16, True, True, False)
    a, _ = _both(sph, dsph, grad_sph, 16, code)
    sph.sphericart_cuda_vjp_noalloc(dsph[:100], grad_sph[:100], torch.empty((100, 3), device="cuda", dtype=tdt), 100, 16,
                                    code, torch.cuda.current_stream().cuda_stream)   # something else in between
    b, _ = _both(sph, dsph, grad_sph, 16, code)
    assert torch.equal(a, b)


def test_vjp_noalloc_allocates_nothing_and_rejects_oversize(sph):
    n, l_max = 4096, 12
    xyz, grad_sph = _inputs(n, l_max, torch.float32, 11)
    _, dsph, _ = sph.compute(xyz, l_max, True, True, False)
    out = torch.empty((n, 3), device="cuda", dtype=torch.float32)
    st = torch.cuda.current_stream().cuda_stream
    sph.sphericart_cuda_vjp_noalloc(dsph, grad_sph, out, n, l_max, sph.F32, st)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(10):
        sph.sphericart_cuda_vjp_noalloc(dsph, grad_sph, out, n, l_max, sph.F32, st)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                              # the driver handed out no device memory
    # the limit: one point more than the static scratch holds -> a clear error, nothing launched
    big = sph.NOALLOC_MAX_POINTS + 1
    d_big = torch.zeros((big, 3, 1), device="cuda", dtype=torch.float32)
    g_big = torch.zeros((big, 1), device="cuda", dtype=torch.float32)
    o_big = torch.zeros((big, 3), device="cuda", dtype=torch.float32)
    before = sph.sphericart_cuda_launch_count()
    with pytest.raises(sph.SphericartCudaError, match="NOALLOC_MAX_POINTS"):
        sph.sphericart_cuda_vjp_noalloc(d_big, g_big, o_big, big, 0, sph.F32, st)
    assert sph.sphericart_cuda_launch_count() == before
    # exactly the limit is served
    sph.sphericart_cuda_vjp_noalloc(d_big[:-1], g_big[:-1], o_big[:-1], big - 1, 0, sph.F32, st)
    torch.cuda.synchronize()
    assert bool((o_big == 0).all())
    # n = 0 is a no-op
    sph.sphericart_cuda_vjp_noalloc(None, None, None, 0, 4, sph.F32, st)


def test_vjp_noalloc_under_graph_capture(sph):
    """The use case: the call is captured into a CUDA graph (an allocation inside a capture fails) and
    replayed; the replays agree with the existing path."""
    n, l_max = 2000, 10
    xyz, grad_sph = _inputs(n, l_max, torch.float64, 21)
    _, dsph, _ = sph.compute(xyz, l_max, True, True, False)
    out = torch.zeros((n, 3), device="cuda", dtype=torch.float64)
    want = sph.vjp(dsph, grad_sph)
    # (as for any captured work: one call outside the capture first, so that the once-per-device set-up and the
    # lazy loading of the two kernels do not fall inside it)
    sph.sphericart_cuda_vjp_noalloc(dsph, grad_sph, out, n, l_max, sph.F64, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    s = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        with torch.cuda.graph(graph, stream=s):
            sph.sphericart_cuda_vjp_noalloc(dsph, grad_sph, out, n, l_max, sph.F64, s.cuda_stream)
    for _ in range(2):
        out.fill_(float("nan"))
        graph.replay()
        torch.cuda.synchronize()
        parity.check_vjp(out.cpu().numpy(), want.cpu().numpy(), dsph.cpu().numpy(), grad_sph.cpu().numpy(), l_max, "f64",
                         "vjp_noalloc replayed from a CUDA graph")
