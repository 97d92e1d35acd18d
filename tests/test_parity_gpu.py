"""`-m gpu`: the CUDA path, called through the C ABI, against the CPU oracle, element by element.

Reduced sizes span several 32-point tiles / 128-harmonic chunks plus a ragged tail; full
BASELINE.json sizes run in the launch configuration bench.py times and are compared on sampled
points.  Tolerance: tests/parity.py.
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

    pkg.load()  # must exist on a GPU box: no fallback
    return pkg


@pytest.fixture
def option(sph):
    """Set launch options (sphericart_cuda_set_option) for one test; defaults restored afterwards."""
    touched = {}

    def set_(name, value):
        touched[name] = True
        sph.sphericart_cuda_set_option(name, value)

    yield set_
    defaults = {"force_kernel": "auto", "tpg_lp": 0, "host_chunk_bytes": 256 << 20, "tq_images": 0, "tq_batch": 0,
                "tq_points": 0, "tq_warps": 0, "tq_direct": 0, "tq_cs_warps": 0, "tpb_split": 0, "tpb_tiles": 0}
    for name in touched:
        sph.sphericart_cuda_set_option(name, defaults[name])


def _torch_dtype(name):
    return torch.float32 if name == "f32" else torch.float64


def _run_gpu(pkg, xyz_np, l_max, normalized, gradients, hessians):
    xyz = torch.from_numpy(xyz_np).cuda()
    s, d, h = pkg.compute(xyz, l_max, normalized, gradients, hessians)
    torch.cuda.synchronize()
    return s, d, h


def _compare(oracle, xyz_np, l_max, normalized, dtype, s, d, h, what):
    ws, wd, wh = oracle.compute(xyz_np, l_max, normalized, d is not None, h is not None)
    out = [parity.check(s.cpu().numpy(), ws, xyz_np, l_max, normalized, 0, dtype, what + " values")]
    if d is not None:
        out.append(parity.check(d.cpu().numpy(), wd, xyz_np, l_max, normalized, 1, dtype, what + " gradients"))
    if h is not None:
        hh = h.cpu().numpy()
        out.append(parity.check(hh, wh, xyz_np, l_max, normalized, 2, dtype, what + " hessians"))
        for a in range(3):                      # S4: both triangles stored and exactly equal
            for b in range(a):
                assert np.array_equal(hh[:, a, b], hh[:, b, a], equal_nan=True)
    return out


# ------------------------------------------------------------------------------------------------
# the five configurations at sizes the oracle finishes in seconds
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name,n", [("C1", 1000), ("C2", 8219), ("C3", 6007), ("C4", 203), ("C5", 10007)])
def test_config_reduced(sph, oracle, name, n):
    cfg = W.CONFIGS[name]
    xyz = W.make_xyz(cfg, n)
    s, d, h = _run_gpu(sph, xyz, cfg.l_max, cfg.normalized, cfg.gradients, cfg.hessians)
    res = _compare(oracle, xyz, cfg.l_max, cfg.normalized, cfg.dtype, s, d, h, name)
    print(name, [r[2] for r in res])
    if cfg.vjp:
        g = W.make_grad_sph(cfg, n)
        gx = sph.vjp(d, torch.from_numpy(g).cuda())
        torch.cuda.synchronize()
        d_np = d.cpu().numpy()
        # isolate the contraction: oracle contracts the GPU-produced dsph ...
        want = oracle.vjp(d_np, g, cfg.l_max)
        parity.check_vjp(gx.cpu().numpy(), want, d_np, g, cfg.l_max, cfg.dtype, name + " vjp (GPU dsph)")
        # ... and end to end from the oracle's own derivatives
        _, wd, _ = oracle.compute(xyz, cfg.l_max, cfg.normalized, True)
        want = oracle.vjp(wd, g, cfg.l_max)
        parity.check_vjp(gx.cpu().numpy(), want, wd, g, cfg.l_max, cfg.dtype, name + " vjp (end to end)")


# ------------------------------------------------------------------------------------------------
# the five configurations at full size, as bench.py launches them; sampled points
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
def test_config_full_size_sampled(sph, oracle, name):
    cfg = W.CONFIGS[name]
    need = cfg.n * (cfg.out_bytes_per_point + cfg.in_bytes_per_point) * 1.05
    free, _ = torch.cuda.mem_get_info()
    if need > free:
        pytest.skip(f"{name} needs {need / 1e9:.1f} GB, {free / 1e9:.1f} GB free")
    xyz = W.make_xyz(cfg)
    s, d, h = _run_gpu(sph, xyz, cfg.l_max, cfg.normalized, cfg.gradients, cfg.hessians)
    rng = np.random.default_rng(7)
    n_s = 384 if name == "C4" else 20000
    idx = np.unique(np.concatenate([rng.integers(0, cfg.n, n_s), [0, 1, 31, 32, cfg.n - 33, cfg.n - 1]]))
    it = torch.from_numpy(idx).cuda()
    pick = lambda t: None if t is None else t.index_select(0, it)
    _compare(oracle, xyz[idx], cfg.l_max, cfg.normalized, cfg.dtype, pick(s), pick(d), pick(h), name + " full")
    # a property that holds at any size: the addition theorem on EVERY point (values only)
    l = parity.l_of_k(cfg.l_max)
    lt = torch.from_numpy(l).cuda()
    sq = (s.double() ** 2)
    rows = torch.zeros((cfg.n, cfg.l_max + 1), dtype=torch.float64, device="cuda")
    rows.index_add_(1, lt, sq)
    r2 = (torch.from_numpy(xyz).cuda().double() ** 2).sum(1)
    lv = torch.arange(cfg.l_max + 1, device="cuda", dtype=torch.float64)
    want = (2 * lv + 1) / (4 * np.pi)
    if not cfg.normalized:
        want = want[None, :] * r2[:, None] ** lv[None, :]
    rel = (rows / want - 1).abs()
    tol = 4 * (cfg.l_max + 1) * (1.2e-7 if cfg.dtype == "f32" else 1e-14)
    assert float(rel.max()) < tol, f"{name}: addition theorem off by {float(rel.max()):.3e}"
    if cfg.vjp:
        g = W.make_grad_sph(cfg)
        gt = torch.from_numpy(g).cuda()
        gx = sph.vjp(d, gt)
        torch.cuda.synchronize()
        d_np = pick(d).cpu().numpy()
        want = oracle.vjp(d_np, g[idx], cfg.l_max)
        parity.check_vjp(pick(gx).cpu().numpy(), want, d_np, g[idx], cfg.l_max, cfg.dtype, name + " full vjp")
        # whole-array property: against torch's own contraction in f64
        ref = torch.einsum("nak,nk->na", d.double(), gt.double())
        scale = d.double().norm(dim=2) * gt.double().norm(dim=1)[:, None]
        assert float(((gx.double() - ref).abs() / scale).max()) < 2e-7
        # N1 at full size, as bench.py launches it: sampled against the oracle, every point against
        # the stored-derivative route
        gr = sph.vjp_recompute(torch.from_numpy(xyz).cuda(), gt, cfg.normalized)
        torch.cuda.synchronize()
        _, wd, _ = oracle.compute(xyz[idx], cfg.l_max, cfg.normalized, True)
        parity.check_vjp(pick(gr).cpu().numpy(), oracle.vjp_recompute(xyz[idx], g[idx], cfg.l_max, cfg.normalized),
                         wd, g[idx], cfg.l_max, cfg.dtype, name + " full vjp_recompute", point_scale=True)
        pscale = scale.max(dim=1, keepdim=True).values
        assert float(((gr.double() - ref).abs() / pscale).max()) < 4e-7


def test_expand_full_size_sampled(sph, oracle):
    """N2 at the size and launch configuration bench.py times (32768 segments, ~1.05 M points,
    l_max = 8, n_rad = 8, f32): sampled segments against the oracle, every segment against
    compute() + a segment sum in torch."""
    l_max, n_rad, n_seg = 8, 8, 32768
    xyz, rad, seg = W.make_expand_inputs(n_seg, l_max, n_rad, "f32", 32.0)
    x_d, r_d, s_d = (torch.from_numpy(a).cuda() for a in (xyz, rad, seg))
    c = sph.expand(x_d, r_d, s_d)
    torch.cuda.synchronize()
    rng = np.random.default_rng(9)
    pick = np.unique(np.concatenate([rng.integers(0, n_seg, 300), [0, 1, n_seg - 1]]))
    lo, hi = seg[pick], seg[pick + 1]
    sub_idx = np.concatenate([np.arange(a, b) for a, b in zip(lo, hi)])
    sub_seg = np.concatenate([[0], np.cumsum(hi - lo)])
    want = oracle.expand(xyz[sub_idx], rad[sub_idx], sub_seg, l_max)
    parity.check_expand(c.cpu().numpy()[pick], want, rad[sub_idx], sub_seg, l_max, "f32", "expand full")
    Y = sph.compute(x_d, l_max, True)[0].double()
    l_of = torch.from_numpy(parity.l_of_k(l_max)).cuda()
    terms = r_d.double()[:, :, l_of] * Y[:, None, :]
    owner = torch.repeat_interleave(torch.arange(n_seg, device="cuda"), torch.from_numpy(np.diff(seg)).cuda())
    ref = torch.zeros((n_seg, n_rad, (l_max + 1) ** 2), dtype=torch.float64, device="cuda").index_add_(0, owner, terms)
    mag = torch.zeros_like(ref).index_add_(0, owner, terms.abs())
    assert float(((c.double() - ref).abs() / (mag + 1e-30)).max()) < 1e-6


# ------------------------------------------------------------------------------------------------
# every kernel variant at small sizes: dtype x derivative order x normalisation x l_max
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("l_max", [0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 12, 16, 17, 32])
@pytest.mark.parametrize("normalized", [False, True])
def test_all_variants_small(sph, oracle, dtype, l_max, normalized):
    rng = np.random.default_rng([l_max, int(normalized)])
    n = 77 if l_max > 9 else 333                              # several tiles + a ragged tail
    xyz = rng.standard_normal((n, 3)) * 1.2
    xyz[3] = [0, 0, 1.5]                                      # +z
    xyz[4] = [0, 0, -0.7]                                     # -z
    xyz[5] = [1e-5, -2e-5, 3e-6]                              # near the origin
    xyz[6] = [0.3, 0, 0]
    xyz = xyz.astype(np.float32 if dtype == "f32" else np.float64)
    for deriv in (0, 1, 2):
        s, d, h = _run_gpu(sph, xyz, l_max, normalized, deriv >= 1, deriv >= 2)
        _compare(oracle, xyz, l_max, normalized, dtype, s, d, h, f"{dtype} l={l_max} norm={normalized} d={deriv}")


@pytest.mark.parametrize("force", ["auto", "tpg", "w"])
def test_all_forward_kernels_agree_with_the_oracle(sph, oracle, force, option):
    """The compile-time-l_max (auto picks it for l_max <= 8), lanes-per-point and warp-per-point
    kernels are interchangeable where they all apply."""
    option("force_kernel", force)
    for dtype, l_max in (("f32", 8), ("f64", 4), ("f32", 3), ("f64", 7)):
        cfgname = "C2"
        xyz = W.make_xyz(cfgname, 2000 + 13).astype(np.float32 if dtype == "f32" else np.float64)
        s, d, h = _run_gpu(sph, xyz, l_max, True, True, False)
        _compare(oracle, xyz, l_max, True, dtype, s, d, h, f"force={force} {dtype} l={l_max}")


# ------------------------------------------------------------------------------------------------
# edge cases
# ------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n", [0, 1, 2, 31, 32, 33, 63, 64, 65])
def test_ragged_sizes(sph, oracle, n):
    for dtype, l_max, hess in (("f32", 6, False), ("f64", 4, False), ("f64", 10, True), ("f32", 3, True)):
        xyz = np.random.default_rng(n).standard_normal((n, 3)).astype(
            np.float32 if dtype == "f32" else np.float64)
        s, d, h = _run_gpu(sph, xyz, l_max, True, True, hess)
        assert s.shape == (n, (l_max + 1) ** 2)
        if n:
            _compare(oracle, xyz, l_max, True, dtype, s, d, h, f"n={n} {dtype} l={l_max}")
            g = np.random.default_rng(n + 1).standard_normal((n, (l_max + 1) ** 2)).astype(xyz.dtype)
            gx = sph.vjp(d, torch.from_numpy(g).cuda())
            d_np = d.cpu().numpy()
            parity.check_vjp(gx.cpu().numpy(), oracle.vjp(d_np, g, l_max), d_np, g, l_max, dtype)


def test_vjp_long_rows(sph, oracle):
    """Rows too long for the staged VJP kernel take the warp-per-point one."""
    for dtype, l_max, n in (("f64", 32, 41), ("f32", 32, 70), ("f64", 16, 100)):
        xyz = W.make_xyz("C4", n).astype(np.float32 if dtype == "f32" else np.float64)
        _, d, _ = _run_gpu(sph, xyz, l_max, True, True, False)
        g = np.random.default_rng(3).standard_normal((n, (l_max + 1) ** 2)).astype(xyz.dtype)
        gx = sph.vjp(d, torch.from_numpy(g).cuda())
        d_np = d.cpu().numpy()
        parity.check_vjp(gx.cpu().numpy(), oracle.vjp(d_np, g, l_max), d_np, g, l_max, dtype)


def _check_vjp_recompute(sph, oracle, xyz, l_max, normalized, dtype, what):
    n = xyz.shape[0]
    g = np.random.default_rng(l_max + 100 * n).standard_normal((n, (l_max + 1) ** 2)).astype(xyz.dtype)
    gx = sph.vjp_recompute(torch.from_numpy(xyz).cuda(), torch.from_numpy(g).cuda(), normalized)
    torch.cuda.synchronize()
    _, wd, _ = oracle.compute(xyz, l_max, normalized, True)
    want = oracle.vjp_recompute(xyz, g, l_max, normalized)
    return parity.check_vjp(gx.cpu().numpy(), want, wd, g, l_max, dtype, what, point_scale=True)


@pytest.mark.parametrize("name,n", [("C1", 1000), ("C2", 4099), ("C5", 6000), ("C2", 7), ("C3", 2049)])
def test_vjp_recompute_configs(sph, oracle, name, n):
    """N1: backward without stored derivatives against the oracle's compute + vjp, on the configs'
    own point clouds (C2: points on +-z and |r| down to 1e-6), both variants."""
    cfg = W.CONFIGS[name]
    l_max = min(cfg.l_max, 12)
    xyz = W.make_xyz(cfg, n)
    for normalized in (True, False):
        _check_vjp_recompute(sph, oracle, xyz, l_max, normalized, cfg.dtype, f"{name} vjp_recompute norm={normalized}")


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_vjp_recompute_every_l_max(sph, oracle, dtype):
    """Specialised kernels (l_max <= 8, f32 <= 12), the two-phase kernel above that, l_max = 0, ragged n."""
    for l_max in (0, 1, 2, 3, 5, 7, 8, 9, 12, 13, 20, 32):
        n = 3 * 16 + 5
        xyz = W.make_xyz("C4" if l_max > 12 else "C2", n).astype(np.float32 if dtype == "f32" else np.float64)
        for normalized in (True, False):
            _check_vjp_recompute(sph, oracle, xyz, l_max, normalized, dtype, f"{dtype} l_max={l_max} norm={normalized}")


def test_vjp_recompute_matches_stored_route_and_generic(sph, oracle, option):
    """Same numbers as forward-with-gradients followed by the stored-derivative VJP (to rounding),
    and the generic kernel agrees with the specialised one."""
    cfg = W.CONFIGS["C5"]
    n = 20_000
    xyz = W.make_xyz(cfg, n)
    g = W.make_grad_sph(cfg, n)
    x_d, g_d = torch.from_numpy(xyz).cuda(), torch.from_numpy(g).cuda()
    _, d, _ = sph.compute(x_d, cfg.l_max, True, True)
    stored = sph.vjp(d, g_d).cpu().numpy()
    before = sph.sphericart_cuda_launch_count()
    rec = sph.vjp_recompute(x_d, g_d, True).cpu().numpy()
    assert sph.sphericart_cuda_launch_count() == before + 1
    scale = np.abs(stored).max()
    assert np.max(np.abs(rec - stored)) <= 2e-6 * scale
    option("force_kernel", "generic")
    gen = sph.vjp_recompute(x_d, g_d, True).cpu().numpy()
    assert sph.sphericart_cuda_last_kernel() == "vjpr_generic"
    assert np.max(np.abs(gen - rec)) <= 2e-6 * scale
    # guard bands: grad_xyz is written exactly where it belongs
    buf = torch.full((n * 3 + 64,), 777.0, device="cuda")
    option("force_kernel", "auto")
    sph.sphericart_cuda_vjp_recompute(x_d, g_d, buf[32:-32], n, cfg.l_max, 1, 0, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert torch.all(buf[:32] == 777.0) and torch.all(buf[-32:] == 777.0) and torch.all(buf[32:-32] != 777.0)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_cooperative_kernel_long_rows(sph, oracle, dtype, option):
    """Rows with l_max >= 19 take the CTA-cooperative kernel (kernel_wc.cuh): every derivative order,
    both variants, odd and even row lengths, n below / across / not a multiple of the 128 points a
    CTA owns; and it writes the same numbers as the one-warp-per-point kernel."""
    np_dt = np.float32 if dtype == "f32" else np.float64
    cases = [(32, 1, True, True, True), (32, 127, True, True, False), (31, 129, True, True, True),
             (19, 300, True, False, True), (20, 77, False, False, False), (26, 257, True, True, True),
             (25, 130, True, False, False)]
    for l_max, n, grads, hess, normalized in cases:
        xyz = W.make_xyz("C4", n).astype(np_dt)
        s, d, h = _run_gpu(sph, xyz, l_max, normalized, grads, hess)
        _compare(oracle, xyz, l_max, normalized, dtype, s, d, h, f"wc {dtype} l_max={l_max} n={n}")
        option("force_kernel", "wc")   # (the default route may be another family)
        s, d, h = _run_gpu(sph, xyz, l_max, normalized, grads, hess)
        assert sph.sphericart_cuda_last_kernel() == "wc"
        _compare(oracle, xyz, l_max, normalized, dtype, s, d, h, f"forced wc {dtype} l_max={l_max} n={n}")
        option("force_kernel", "w1")
        s1, d1, h1 = _run_gpu(sph, xyz, l_max, normalized, grads, hess)
        assert sph.sphericart_cuda_last_kernel() == "w"
        option("force_kernel", "auto")
        for a, b in ((s, s1), (d, d1), (h, h1)):
            if a is not None:
                assert torch.equal(a, b), "cooperative and one-warp kernels disagree bit-wise"
    # guard bands around the three outputs
    n, l_max = 131, 32
    L = (l_max + 1) ** 2
    t_dt = torch.float32 if dtype == "f32" else torch.float64
    pts = torch.from_numpy(W.make_xyz("C4", n).astype(np_dt)).cuda()
    bufs = [torch.full((m + 64,), 777.0, device="cuda", dtype=t_dt) for m in (n * L, n * 3 * L, n * 9 * L)]
    views = [b[32:-32] for b in bufs]
    sph.sphericart_cuda_compute(pts, n, l_max, 1, 0 if dtype == "f32" else 1, views[0], views[1], views[2],
                                torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    for b in bufs:
        assert torch.all(b[:32] == 777.0) and torch.all(b[-32:] == 777.0) and torch.all(b[32:-32] != 777.0)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("lp", [2, 4, 8])
def test_lanes_per_point_kernel(sph, oracle, dtype, lp, option):
    """kernel_tpg.cuh (several lanes per point, run-time l_max): forced for every l_max it can take,
    every lanes-per-point variant, values and values + gradients, both variants, ragged n; C2-style
    points (on the z axis, tiny r) included."""
    np_dt = np.float32 if dtype == "f32" else np.float64
    option("force_kernel", "tpg")
    option("tpg_lp", lp)
    for l_max, n, grads, normalized in ((0, 5, True, True), (1, 33, True, False), (3, 100, False, True),
                                        (9, 131, True, True), (10, 64, True, False), (13, 77, False, False),
                                        (16, 203, True, True), (21, 50, False, True), (32, 37, False, False)):
        xyz = W.make_xyz("C2" if l_max <= 10 else "C4", n).astype(np_dt)
        before = sph.sphericart_cuda_launch_count()
        s, d, _ = _run_gpu(sph, xyz, l_max, normalized, grads, False)
        assert sph.sphericart_cuda_launch_count() == before + 1
        assert sph.sphericart_cuda_last_kernel() in ("tpg", "w", "wc")     # (tpg declines the longest rows)
        _compare(oracle, xyz, l_max, normalized, dtype, s, d, None, f"tpg {dtype} lp={lp} l_max={l_max} n={n}")


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("l_max", [0, 1, 2, 3, 5, 8, 9, 11, 12, 15, 16, 20, 23, 27, 32])
def test_two_phase_kernel(sph, oracle, dtype, l_max, option):
    """kernel_tq.cuh (recurrences lane = point, assembly lane = (l, m) pair, full-row tiles of a few
    points): forced for every derivative order and both variants; n spans several batches and tiles
    with a ragged tail, and a second n that ends inside the first tile; C2-style points (on the z
    axis, tiny r) up to l_max = 16."""
    np_dt = np.float32 if dtype == "f32" else np.float64
    option("force_kernel", "tq")
    for n in (3 * 32 + 100 + 7, 3):
        xyz = W.make_xyz("C2" if l_max <= 16 else "C4", n, seed=l_max).astype(np_dt)
        for normalized in (True, False):
            for deriv in (0, 1, 2):
                before = sph.sphericart_cuda_launch_count()
                s, d, h = _run_gpu(sph, xyz, l_max, normalized, deriv >= 1, deriv >= 2)
                assert sph.sphericart_cuda_launch_count() == before + 1
                if sph.sphericart_cuda_last_kernel() != "tq":       # rows too long for one two-point image
                    assert deriv == 2 and l_max >= 24
                    continue
                _compare(oracle, xyz, l_max, normalized, dtype, s, d, h,
                         f"tq {dtype} l_max={l_max} n={n} norm={normalized} deriv={deriv}")


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("shape", [(32, 2, 4, 2), (16, 2, 8, 1), (8, 2, 6, 2), (8, 2, 3, 1), (16, 8, 5, 2), (32, 4, 8, 1),
                                   (8, 1, 4, 1), (16, 1, 6, 2), (32, 1, 12, 2)])
def test_two_phase_kernel_shapes(sph, oracle, dtype, shape, option):
    """Every launch shape of kernel_tq.cuh the shape table can name: batches of 32 / 16 / 8 points
    (1 / 2 / 4 lanes per point in the recurrence phase), tiles of 1 / 2 / 4 / 8 points, one or two
    images; ragged n, odd and even row lengths."""
    np_dt = np.float32 if dtype == "f32" else np.float64
    option("force_kernel", "tq")
    for name, value in zip(("tq_batch", "tq_points", "tq_warps", "tq_images"), shape):
        option(name, value)
    for l_max, n in ((9, 203), (12, 77), (15, 131), (16, 1), (22, 70), (27, 41)):
        xyz = W.make_xyz("C2" if l_max <= 16 else "C4", n, seed=l_max).astype(np_dt)
        for normalized, deriv in ((True, 2), (False, 1), (True, 0)):
            s, d, h = _run_gpu(sph, xyz, l_max, normalized, deriv >= 1, deriv >= 2)
            # (a shape that does not fit these rows falls through to another kernel: compared all the same)
            _compare(oracle, xyz, l_max, normalized, dtype, s, d, h,
                     f"{sph.sphericart_cuda_last_kernel()} shape={shape} {dtype} l_max={l_max} n={n} norm={normalized} deriv={deriv}")


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("shape", [(32, 8), (32, 12), (16, 4), (16, 16), (8, 3), (8, 10)])
def test_two_phase_kernel_direct_stores(sph, oracle, dtype, shape, option):
    """The DIRECT variant of kernel_tq.cuh (no staging image: phase B stores every harmonic straight to
    the caller's arrays; the shape table names it for long rows) and CTAs of up to 16 warps: every
    derivative order, both variants, ragged n and n below one pair of points; then guard bands around
    all three output arrays (nothing written outside them, every element inside written)."""
    np_dt = np.float32 if dtype == "f32" else np.float64
    option("force_kernel", "tq")
    option("tq_batch", shape[0])
    option("tq_warps", shape[1])
    for l_max, n in ((0, 5), (3, 70), (9, 203), (14, 77), (16, 1), (23, 70), (32, 45)):
        xyz = W.make_xyz("C2" if l_max <= 16 else "C4", n, seed=l_max).astype(np_dt)
        for normalized, deriv in ((True, 2), (False, 1), (True, 0), (False, 2)):
            option("tq_direct", 4 if (l_max + deriv) % 2 else 1)      # four / two points per lane in phase B
            before = sph.sphericart_cuda_launch_count()
            s, d, h = _run_gpu(sph, xyz, l_max, normalized, deriv >= 1, deriv >= 2)
            assert sph.sphericart_cuda_launch_count() == before + 1
            assert sph.sphericart_cuda_last_kernel() == "tq"
            _compare(oracle, xyz, l_max, normalized, dtype, s, d, h,
                     f"tq direct shape={shape} {dtype} l_max={l_max} n={n} norm={normalized} deriv={deriv}")
    option("tq_direct", 4)
    l_max, n = 21, 45
    L = (l_max + 1) ** 2
    t_dt = torch.float32 if dtype == "f32" else torch.float64
    pts = torch.from_numpy(W.make_xyz("C4", n).astype(np_dt)).cuda()
    bufs = [torch.full((n * rows * L + 64,), 777.0, device="cuda", dtype=t_dt) for rows in (1, 3, 9)]
    sph.sphericart_cuda_compute(pts, n, l_max, 1, 0 if dtype == "f32" else 1, bufs[0][32:-32], bufs[1][32:-32], bufs[2][32:-32],
                                torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert sph.sphericart_cuda_last_kernel() == "tq"
    for buf in bufs:
        assert torch.all(buf[:32] == 777.0) and torch.all(buf[-32:] == 777.0) and torch.all(buf[32:-32] != 777.0)


@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("l_max", [0, 1, 2, 3, 4, 7, 8, 11, 12, 15, 16, 19, 24, 25, 31, 32])
def test_values_only_kernel(sph, oracle, dtype, l_max, option):
    """kernel_tv.cuh (values only: every Legendre entry straight into a per-point image row, the powers
    of x + iy one batch ahead): forced, both variants, every batch size, ragged n, n below one batch;
    C2-style points (on the z axis, tiny r) up to l_max = 16."""
    np_dt = np.float32 if dtype == "f32" else np.float64
    option("force_kernel", "tv")
    for batch in (0, 32, 16, 8):
        option("tq_batch", batch)
        for n in (5 * 32 + 100 + 7, 3):
            xyz = W.make_xyz("C2" if l_max <= 16 else "C4", n, seed=l_max).astype(np_dt)
            for normalized in (True, False):
                before = sph.sphericart_cuda_launch_count()
                s, _, _ = _run_gpu(sph, xyz, l_max, normalized, False, False)
                assert sph.sphericart_cuda_launch_count() == before + 1
                assert sph.sphericart_cuda_last_kernel() == "tv"
                _compare(oracle, xyz, l_max, normalized, dtype, s, None, None,
                         f"tv {dtype} l_max={l_max} n={n} batch={batch} norm={normalized}")
    # guard bands: the rows are written exactly where they belong
    n, L = 77, (l_max + 1) ** 2
    t_dt = torch.float32 if dtype == "f32" else torch.float64
    pts = torch.from_numpy(W.make_xyz("C4", n).astype(np_dt)).cuda()
    buf = torch.full((n * L + 64,), 777.0, device="cuda", dtype=t_dt)
    sph.sphericart_cuda_compute(pts, n, l_max, 1, 0 if dtype == "f32" else 1, buf[32:-32], None, None,
                                torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert torch.all(buf[:32] == 777.0) and torch.all(buf[-32:] == 777.0) and torch.all(buf[32:-32] != 777.0)


def test_stream_order_with_programmatic_dependent_launch(sph):
    """The small-grid kernels are launched as programmatic dependent launches: their CTAs may become
    resident while the previous kernel in the stream still runs, but must not read or write
    anything before it has completed.  RAW, WAR and WAW hazards against torch kernels and against
    the library's own kernels, without any synchronisation in between."""
    n, l_max = 60_000, 8
    L = (l_max + 1) ** 2
    x1 = torch.randn(n, 3, device="cuda")
    x2 = torch.randn(n, 3, device="cuda")
    ref1 = sph.compute(x1, l_max, True, True)
    ref2 = sph.compute(x2, l_max, True, True)
    torch.cuda.synchronize()
    st = torch.cuda.current_stream().cuda_stream
    for _ in range(20):
        x = x1.clone()
        s = torch.empty((n, L), device="cuda")
        d = torch.empty((n, 3, L), device="cuda")
        big = torch.randn(64 << 20, device="cuda")
        big.mul_(1.0001)                                   # something long-running in front
        x.copy_(x2)                                        # RAW: the forward must see x2
        sph.sphericart_cuda_compute(x, n, l_max, 1, 0, s, d, None, st)
        keep = s.clone()                                   # WAR: the clone must see this forward's values
        sph.sphericart_cuda_compute(x1, n, l_max, 1, 0, s, d, None, st)   # WAW on s, d
        g = torch.ones((n, L), device="cuda")
        g.mul_(2.0)                                        # RAW for the recompute VJP
        gx = sph.vjp_recompute(x1, g, True)
        torch.cuda.synchronize()
        assert torch.equal(keep, ref2[0])
        assert torch.equal(s, ref1[0]) and torch.equal(d, ref1[1])
        want = sph.vjp(ref1[1], torch.full((n, L), 2.0, device="cuda"))
        assert torch.allclose(gx, want, rtol=1e-4, atol=1e-4 * float(want.abs().max()))


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_expand_segment_layouts(sph, oracle, dtype):
    """N2, the layouts that stress how the persistent grid shares the segments among its warps (by point
    count, two binary searches over seg_ptr): one long segment among empty ones, every segment empty,
    a single segment, far more segments than points, far more warps than segments, a first segment that
    is empty; with a radial row of 16-byte multiples (one bulk load per tile) and without (cp.async)."""
    np_dt = np.float32 if dtype == "f32" else np.float64
    rng = np.random.default_rng(77)

    def run(counts, l_max, n_rad, what):
        seg = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
        n = int(seg[-1])
        xyz_all = rng.standard_normal((max(n, 1), 3)).astype(np_dt)
        rad_all = rng.standard_normal((max(n, 1), n_rad, l_max + 1)).astype(np_dt)
        xyz, rad = xyz_all[:n], rad_all[:n]
        # (no points at all: the C entry still wants non-NULL pointers, so views of a one-row allocation)
        x_d, r_d = torch.from_numpy(xyz_all).cuda()[:n], torch.from_numpy(rad_all).cuda()[:n]
        c = sph.expand(x_d, r_d, torch.from_numpy(seg).cuda())
        torch.cuda.synchronize()
        parity.check_expand(c.cpu().numpy(), oracle.expand(xyz, rad, seg, l_max), rad, seg, l_max, dtype,
                            f"expand {dtype} {what} l_max={l_max} n_rad={n_rad}")
        assert np.all(c.cpu().numpy()[np.nonzero(np.diff(seg) == 0)[0]] == 0)

    # (l_max <= 8: the compile-time kernel; above: the banded run-time kernel, n_rad <= 8 and 9..16)
    for l_max, n_rad in ((8, 8), (5, 3), (6, 7), (12, 8), (10, 3), (17, 12)):   # radial rows with and without 16-byte multiples
        run([0] * 40 + [5003] + [0] * 60, l_max, n_rad, "one long segment among empty ones")
        run([0] * 500, l_max, n_rad, "every segment empty")
        run([37], l_max, n_rad, "a single segment")
        run(rng.integers(0, 2, size=20000), l_max, n_rad, "more segments than points")
        run([700, 0, 1, 16, 17, 15], l_max, n_rad, "few segments, many warps")
        run([0, 0, 33, 4], l_max, n_rad, "leading empty segments")


@pytest.mark.parametrize("dtype", ["f32", "f64"])
def test_expand_eq1(sph, oracle, dtype):
    """N2: the fused density expansion against the oracle; every l_max with a kernel, n_rad across
    the three register variants, ragged / empty / long segments."""
    for l_max, n_rad, n_seg, mean in ((8, 8, 300, 32.0), (6, 3, 200, 5.0), (4, 16, 64, 70.0), (1, 1, 50, 2.0),
                                     (0, 2, 40, 3.0), (7, 5, 33, 17.0), (8, 12, 20, 40.0)):
        xyz, rad, seg = W.make_expand_inputs(n_seg, l_max, n_rad, dtype, mean)
        c = sph.expand(torch.from_numpy(xyz).cuda(), torch.from_numpy(rad).cuda(), torch.from_numpy(seg).cuda())
        torch.cuda.synchronize()
        want = oracle.expand(xyz, rad, seg, l_max)
        parity.check_expand(c.cpu().numpy(), want, rad, seg, l_max, dtype, f"expand {dtype} l_max={l_max} n_rad={n_rad}")
        empty = np.nonzero(np.diff(seg) == 0)[0]
        assert np.all(c.cpu().numpy()[empty] == 0)
    # the same numbers as compute() followed by a segment sum in torch (f64 accumulation)
    xyz, rad, seg = W.make_expand_inputs(100, 6, 4, dtype, 20.0)
    x_d, r_d = torch.from_numpy(xyz).cuda(), torch.from_numpy(rad).cuda()
    c = sph.expand(x_d, r_d, torch.from_numpy(seg).cuda())
    Y = sph.compute(x_d, 6, True)[0].double()
    l_of = torch.tensor(np.concatenate([[l] * (2 * l + 1) for l in range(7)]), device="cuda")
    terms = r_d.double()[:, :, l_of] * Y[:, None, :]
    ref = torch.stack([terms[seg[i]:seg[i + 1]].sum(dim=0) for i in range(100)])
    assert torch.allclose(c.double(), ref, rtol=1e-5 if dtype == "f32" else 1e-12, atol=1e-5 if dtype == "f32" else 1e-12)
    # the run-time-size kernel agrees with the compile-time one where both apply
    sph.sphericart_cuda_set_option("force_kernel", "generic")
    try:
        cg = sph.expand(x_d, r_d, torch.from_numpy(seg).cuda())
        assert sph.sphericart_cuda_last_kernel() == "expand_generic"
    finally:
        sph.sphericart_cuda_set_option("force_kernel", "auto")
    assert torch.allclose(cg.double(), ref, rtol=1e-5 if dtype == "f32" else 1e-12, atol=1e-5 if dtype == "f32" else 1e-12)


def test_origin_and_untouched_memory(sph, oracle):
    # normalised at r = 0: NaN for that point only; solid at r = 0 is defined
    xyz = np.array([[0, 0, 0], [1, 2, 3], [0, 0, 0], [-1, 0.5, 0.25]], np.float64)
    for l_max, hess in ((4, False), (11, True)):
        s, d, h = _run_gpu(sph, xyz, l_max, True, True, hess)
        s = s.cpu().numpy()
        assert np.all(np.isnan(s[[0, 2], 1:])) and np.all(np.isfinite(s[[1, 3]]))
        s, d, h = _run_gpu(sph, xyz, l_max, False, True, hess)
        _compare(oracle, xyz, l_max, False, "f64", s, d, h, "solid at the origin")
    # outputs are written exactly where they belong: guard bands around the buffers stay intact
    n, l_max = 101, 6
    L = (l_max + 1) ** 2
    pts = torch.randn(n, 3, device="cuda")
    for hess in (False, True):
        bufs = [torch.full((m + 64,), 777.0, device="cuda") for m in (n * L, n * 3 * L, n * 9 * L)]
        views = [b[32:-32] for b in bufs]             # 128-byte offset keeps the 16-byte alignment
        sph.sphericart_cuda_compute(pts, n, l_max, 1, 0, views[0], views[1], views[2] if hess else None,
                                    torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        for b, used in zip(bufs, (True, True, hess)):
            assert torch.all(b[:32] == 777.0) and torch.all(b[-32:] == 777.0)
            assert bool(torch.all(b[32:-32] != 777.0)) == used


def test_host_buffer_entry_points(sph, oracle):
    cfg = W.CONFIGS["C5"]
    n = 50_021
    xyz = W.make_xyz(cfg, n)
    L = cfg.n_sph
    s = np.empty((n, L), np.float32)
    d = np.empty((n, 3, L), np.float32)
    sph.sphericart_cuda_compute_host(xyz, n, cfg.l_max, 1, 0, s, d, None)
    idx = np.arange(0, n, 37)
    ws, wd, _ = oracle.compute(xyz[idx], cfg.l_max, True, True)
    parity.check(s[idx], ws, xyz[idx], cfg.l_max, True, 0, "f32", "host values")
    parity.check(d[idx], wd, xyz[idx], cfg.l_max, True, 1, "f32", "host gradients")
    g = W.make_grad_sph(cfg, n)
    gx = np.empty((n, 3), np.float32)
    sph.sphericart_cuda_vjp_host(None, d, g, gx, n, cfg.l_max, 0)
    parity.check_vjp(gx[idx], oracle.vjp(d[idx], g[idx], cfg.l_max), d[idx], g[idx], cfg.l_max, "f32")


def test_host_buffer_entry_points_many_chunks(sph, oracle, option):
    """The chunked two-stream path: >= 3 chunks with a ragged last one, slot reuse, pinned host
    memory, Hessians through compute_host and the VJP through vjp_host."""
    l_max, n = 5, 1000 + 13
    L = (l_max + 1) ** 2
    option("host_chunk_bytes", 13 * L * 8 * 300)          # ~300 points per chunk -> 4 chunks, last one ragged
    xyz = torch.from_numpy(W.make_xyz("C4", n)).pin_memory()
    s = torch.empty((n, L), dtype=torch.float64).pin_memory()
    d = torch.empty((n, 3, L), dtype=torch.float64).pin_memory()
    h = torch.empty((n, 3, 3, L), dtype=torch.float64).pin_memory()
    before = sph.sphericart_cuda_launch_count()
    sph.sphericart_cuda_compute_host(xyz, n, l_max, 1, 1, s, d, h)
    assert sph.sphericart_cuda_launch_count() - before >= 3
    x_np = xyz.numpy()
    ws, wd, wh = oracle.compute(x_np, l_max, True, True, True)
    parity.check(s.numpy(), ws, x_np, l_max, True, 0, "f64", "host chunks values")
    parity.check(d.numpy(), wd, x_np, l_max, True, 1, "f64", "host chunks gradients")
    parity.check(h.numpy(), wh, x_np, l_max, True, 2, "f64", "host chunks hessians")
    g = torch.from_numpy(np.random.default_rng(5).standard_normal((n, L))).pin_memory()
    gx = torch.empty((n, 3), dtype=torch.float64).pin_memory()
    option("host_chunk_bytes", 4 * L * 8 * 300)
    before = sph.sphericart_cuda_launch_count()
    sph.sphericart_cuda_vjp_host(None, d, g, gx, n, l_max, 1)
    assert sph.sphericart_cuda_launch_count() - before >= 3
    parity.check_vjp(gx.numpy(), oracle.vjp(d.numpy(), g.numpy(), l_max), d.numpy(), g.numpy(), l_max, "f64")
    # an error in a later chunk (device allocation refused) returns only after both streams have drained
    option("host_chunk_bytes", 1 << 62)
    with pytest.raises(sph.SphericartCudaError):
        sph.sphericart_cuda_compute_host(xyz, 1 << 40, l_max, 1, 1, s, d, h)
    torch.cuda.synchronize()


def test_errors_raise(sph):
    x = torch.randn(10, 3, device="cuda")
    with pytest.raises(sph.SphericartCudaError):
        sph.compute(x.cpu(), 3)
    with pytest.raises(sph.SphericartCudaError):
        sph.compute(x, 33)
    with pytest.raises(sph.SphericartCudaError):          # misaligned view
        sph.sphericart_cuda_compute(x.view(-1)[1:], 3, 2, 1, 0, torch.empty(64, device="cuda"), None, None, None)
    before = sph.sphericart_cuda_launch_count()
    sph.compute(x, 3, gradients=True)
    assert sph.sphericart_cuda_launch_count() == before + 1
