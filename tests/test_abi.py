"""`-m "not gpu"`: the C-ABI library loads and exports every symbol include/*.h declares, the Python
binding carries the same names, and argument errors are rejected before anything touches CUDA."""
import ctypes
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


def _declared_symbols():
    names = []
    for h in (ROOT / "include").glob("*.h"):
        text = re.sub(r"/\*.*?\*/", "", h.read_text(), flags=re.S)
        names += re.findall(r"\b(sphericart_cuda_\w+)\s*\(", text)
    return sorted(set(names))


@pytest.fixture(scope="module")
def lib():
    from paper_2302_08381_b200 import build

    build.build()          # nvcc cross-compiles without a GPU
    import paper_2302_08381_b200 as pkg

    return pkg


def test_header_declares_the_boundary():
    names = _declared_symbols()
    for must in ("sphericart_cuda_compute", "sphericart_cuda_vjp", "sphericart_cuda_last_error",
                 "sphericart_cuda_compute_host", "sphericart_cuda_vjp_host", "sphericart_cuda_vjp_recompute", "sphericart_cuda_expand"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    cdll = ctypes.CDLL(str(lib.library_path()))
    for name in _declared_symbols():
        assert hasattr(cdll, name), f"{name} declared in include/ but not exported"


def test_binding_has_the_same_names(lib):
    for name in _declared_symbols():
        assert callable(getattr(lib, name)), f"binding lacks {name}"


def test_argument_errors_do_not_need_a_gpu(lib):
    c = lib.load()
    assert c.sphericart_cuda_compute(None, -1, 4, 1, 0, None, None, None, None) == 1
    assert b"negative" in c.sphericart_cuda_last_error()
    assert c.sphericart_cuda_compute(None, 10, 33, 1, 0, None, None, None, None) == 1
    assert c.sphericart_cuda_compute(None, 10, -1, 1, 0, None, None, None, None) == 1
    assert c.sphericart_cuda_compute(None, 10, 4, 1, 7, None, None, None, None) == 1
    assert c.sphericart_cuda_compute(None, 10, 4, 2, 0, None, None, None, None) == 1       # normalized
    assert c.sphericart_cuda_compute(None, 10, 4, 1, 0, None, None, 16, None) == 1          # ddsph w/o dsph
    assert c.sphericart_cuda_compute(None, 10, 4, 1, 0, None, None, None, None) == 1        # NULL xyz
    assert c.sphericart_cuda_compute(8, 10, 4, 1, 0, 16, None, None, None) == 2             # misaligned
    assert c.sphericart_cuda_compute(None, 0, 4, 1, 0, None, None, None, None) == 0         # n == 0
    assert c.sphericart_cuda_vjp(None, None, None, None, 5, 4, 0, None) == 1
    assert c.sphericart_cuda_vjp(None, None, None, None, 0, 4, 0, None) == 0
    assert c.sphericart_cuda_vjp(None, 16, 16, 4, 5, 4, 0, None) == 2
    assert c.sphericart_cuda_vjp_recompute(None, None, None, 5, 4, 1, 0, None) == 1              # NULL pointers
    assert c.sphericart_cuda_vjp_recompute(None, None, None, 0, 4, 1, 0, None) == 0              # n == 0
    assert c.sphericart_cuda_vjp_recompute(16, 16, 16, 5, 4, 3, 0, None) == 1                    # normalized
    assert c.sphericart_cuda_vjp_recompute(16, 16, 16, 5, 40, 1, 0, None) == 1                   # l_max
    assert c.sphericart_cuda_vjp_recompute(16, 8, 16, 5, 4, 1, 0, None) == 2                     # misaligned
    assert c.sphericart_cuda_expand(None, None, None, 5, 4, 2, 0, None, None) == 1                # NULL pointers
    assert c.sphericart_cuda_expand(None, None, None, 0, 4, 2, 0, None, None) == 0                # n_seg == 0
    assert c.sphericart_cuda_expand(16, 16, 16, 5, 4, 0, 0, 16, None) == 1                        # n_rad
    assert c.sphericart_cuda_expand(16, 16, 12, 5, 4, 2, 0, 16, None) == 2                        # seg_ptr alignment
    with pytest.raises(lib.SphericartCudaError):
        lib.sphericart_cuda_compute(None, -1, 4, 1, 0, None, None, None, None)


def test_product_never_imports_the_oracle():
    for p in (ROOT / "paper_2302_08381_b200").rglob("*"):
        if p.suffix in (".py", ".cu", ".cuh", ".cpp", ".h"):
            text = p.read_text()
            assert "import oracle" not in text and "from oracle" not in text, p
            assert "oracle/" not in text or p.name == "workloads.py" or "shares nothing with oracle/" in text, p
    for p in (ROOT / "oracle").rglob("*.py"):
        assert "paper_2302_08381_b200 import" not in p.read_text().replace(
            "never imports it", ""), p
