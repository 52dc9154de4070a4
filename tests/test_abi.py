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
    return sorted(set(re.findall(r"\b(pa_[a-z_0-9]+)\s*\(", text)))


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
    bad = PaConfig(32, 8, 96, 16, 64, 4, 64, 8, 0, 0, 0, 0, 0, 0)          # head_dim 96
    assert lib.pa_create(ctypes.byref(ctx), ctypes.byref(bad)) == PA_ERR_UNSUPPORTED
    bad = PaConfig(32, 8, 128, 32, 64, 4, 64, 8, 0, 0, 0, 0, 0, 0)         # block 32
    assert lib.pa_create(ctypes.byref(ctx), ctypes.byref(bad)) == PA_ERR_UNSUPPORTED
    bad = PaConfig(32, 2, 128, 16, 64, 4, 64, 8, 0, 0, 0, 0, 0, 0)         # G = 16
    assert lib.pa_create(ctypes.byref(ctx), ctypes.byref(bad)) == PA_ERR_UNSUPPORTED
    bad = PaConfig(32, 8, 128, 16, 0, 4, 64, 8, 0, 0, 0, 0, 0, 0)          # no blocks
    assert lib.pa_create(ctypes.byref(ctx), ctypes.byref(bad)) == PA_ERR_INVALID
    bad = PaConfig(32, 8, 128, 16, 64, 4, 64, 8, 0, 0, 0, 5, 0, 0)   # tune_bundles_per_stream out of range
    assert lib.pa_create(ctypes.byref(ctx), ctypes.byref(bad)) == PA_ERR_INVALID


def test_config_struct_matches_header():
    """pa_config in include/pa.h and binding.PaConfig list the same fields in the same order."""
    from paper_2606_00516_b200.binding import PaConfig
    text = open(os.path.join(ROOT, "include", "pa.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} pa_config;", text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = re.findall(r"\b(?:u?int32_t|int64_t)\s+(\w+)\s*;", body)
    assert names == [f[0] for f in PaConfig._fields_]


def test_crossover_scalars_match_the_oracle(lib):
    """N3 host arithmetic of the product (pa_crossover_*) against the oracle's Eq. 3 / Eq. 7 (no GPU needed)."""
    import numpy as np
    import oracle
    f64 = ctypes.c_double
    lib.pa_crossover_theta0.argtypes = [f64, ctypes.POINTER(f64), ctypes.POINTER(f64)]
    lib.pa_crossover_eq7.argtypes = [ctypes.POINTER(f64), ctypes.POINTER(f64)]
    for x in [1e-9, 1e-4, 0.01, 0.3068528194400547, 0.9, 3.0, 50.0, 1e4]:
        th, ze = f64(), f64()
        assert lib.pa_crossover_theta0(x, ctypes.byref(th), ctypes.byref(ze)) == 0
        oth, oze = oracle.theta0(x)
        assert abs(th.value - oth) < 1e-12 and abs(ze.value - oze) < 1e-10 * max(1.0, oze)
    th, ze = f64(), f64()
    assert lib.pa_crossover_theta0(0.0, ctypes.byref(th), ctypes.byref(ze)) == -1
    rng = np.random.default_rng(78)
    for _ in range(100):
        v = [rng.uniform(1e-4, 5e-2), rng.uniform(1e-6, 1e-4), rng.uniform(1e-4, 5e-2), rng.uniform(1e-6, 1e-4),
             rng.uniform(1e-4, 5e-2), rng.uniform(1e-6, 1e-4), rng.uniform(1, 3000), rng.uniform(1, 3000),
             rng.uniform(0.05, 3.0), float(rng.integers(1, 2000)), float(rng.integers(1, 4000))]
        out = (f64 * 5)()
        assert lib.pa_crossover_eq7((f64 * 11)(*v), out) == 0
        o = oracle.eq7(*v)
        for got, key in zip(out, ("lhs", "rhs", "beta_eb_w", "tp_eb", "tp_mb")):
            assert abs(got - o[key]) <= 1e-12 * max(abs(o[key]), 1e-30) + 1e-20
    bad = (f64 * 11)(1, 1, 1, 1, 1, 1, 0, 0, 1, 1, 1)
    assert lib.pa_crossover_eq7(bad, (f64 * 5)()) == -1


def test_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2606_00516_b200 import binding
    with pytest.raises(binding.PaError):
        binding.PagedAttention(8, 2, 128, 64, 4, 130, 8)
