"""CPU checks of the boundary: the C-ABI library builds, loads and exports every symbol include/pa.h
declares; the binding mirrors them; there is no fallback when no GPU is present."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "pa.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(pa_[a-z_]+)\s*\(", text)))


@pytest.fixture(scope="module")
def lib():
    from paper_2606_00516_b200 import build
    build.build()
    return ctypes.CDLL(os.path.join(ROOT, "paper_2606_00516_b200", "libpa_b200.so"))


def test_header_declares_the_boundary():
    names = _declared()
    for must in ("pa_kv_append", "pa_plan", "pa_batch_attention", "pa_kv_gather", "pa_timer_begin", "pa_timer_end",
                 "pa_timer_fit", "pa_create", "pa_destroy", "pa_workspace_bytes", "pa_last_error"):
        assert must in names


def test_library_exports_every_declared_symbol(lib):
    for name in _declared():
        assert hasattr(lib, name), f"{name} declared in include/pa.h but not exported"


def test_binding_mirrors_header():
    from paper_2606_00516_b200 import binding
    assert sorted(binding.EXPORTS) == _declared()


def test_no_torch_types_in_signatures():
    text = open(os.path.join(ROOT, "include", "pa.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)          # signatures only, not the prose
    assert "torch" not in text.lower() and "at::" not in text and "Tensor" not in text


def test_create_rejects_bad_shapes_without_touching_the_gpu(lib):
    from paper_2606_00516_b200.binding import PaConfig, PA_ERR_UNSUPPORTED, PA_ERR_INVALID
    ctx = ctypes.c_void_p()
    lib.pa_create.restype = ctypes.c_int32
    bad = PaConfig(32, 8, 96, 16, 64, 4, 64, 8, 0, 0)          # head_dim 96
    assert lib.pa_create(ctypes.byref(ctx), ctypes.byref(bad)) == PA_ERR_UNSUPPORTED
    bad = PaConfig(32, 8, 128, 32, 64, 4, 64, 8, 0, 0)         # block 32
    assert lib.pa_create(ctypes.byref(ctx), ctypes.byref(bad)) == PA_ERR_UNSUPPORTED
    bad = PaConfig(32, 2, 128, 16, 64, 4, 64, 8, 0, 0)         # G = 16
    assert lib.pa_create(ctypes.byref(ctx), ctypes.byref(bad)) == PA_ERR_UNSUPPORTED
    bad = PaConfig(32, 8, 128, 16, 0, 4, 64, 8, 0, 0)          # no blocks
    assert lib.pa_create(ctypes.byref(ctx), ctypes.byref(bad)) == PA_ERR_INVALID


def test_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2606_00516_b200 import binding
    with pytest.raises(binding.PaError):
        binding.PagedAttention(8, 2, 128, 64, 4, 130, 8)
