"""pa_decode_attention_static: the allocation-free decode entry point (scratch in a static __device__ array).

Collected last on purpose (the suite runs with pytest -x).  The GPU test compares the entry point with the existing
path (pa_plan + pa_batch_attention with a caller workspace) on the same device tensors, within the parity tolerance of
tests/gpu_common.py, on calls made back to back on one stream: the scratch array keeps the previous call's contents,
so the second and third calls run over stale partials and counters of a different shape.
"""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2606_00516_b200 import binding
from paper_2606_00516_b200.synth import device as sdev
from paper_2606_00516_b200.synth import gen, workloads
from tests import gpu_common as gc
from tests import helpers


def test_static_scratch_limit_is_enforced_before_any_cuda_call():
    """Sizes beyond the static scratch are rejected with PA_ERR_WORKSPACE and a message (host check: runs without a GPU)."""
    lib = binding.load_library()
    cap = binding.static_scratch_bytes()
    assert cap == 16 * 1024 * 1024
    hq, d = 32, 128
    n_seq = cap // (hq * d * 4) + 1           # the unsplit partials alone exceed the array
    one = C.c_void_p(256)                     # never dereferenced: the size check comes first
    rc = lib.pa_decode_attention_static(one, one, one, one, one, n_seq, hq, 8, d, 64, 1000, C.c_float(0.1), one, 0, None)
    assert rc == binding.PA_ERR_WORKSPACE
    msg = lib.pa_static_last_error().decode()
    assert "static scratch" in msg and str(cap) in msg
    # shape rules as for pa_create
    assert lib.pa_decode_attention_static(one, one, one, one, one, 4, hq, 8, 96, 64, 1000, C.c_float(0.1), one, 0,
                                          None) == binding.PA_ERR_UNSUPPORTED
    assert lib.pa_decode_attention_static(one, one, one, one, one, 4, hq, 8, d, 64, 64 * 16 + 1, C.c_float(0.1), one, 0,
                                          None) == binding.PA_ERR_INVALID
    assert lib.pa_decode_attention_static(one, one, one, one, one, 0, hq, 8, d, 64, 1000, C.c_float(0.1), one, 0,
                                          None) == binding.PA_OK
    assert lib.pa_static_last_error().decode() == ""


def _existing_path(batch):
    inp = helpers.host_inputs(batch)
    d = gc.run_gpu(batch, inp)                # kv_append + pa_plan + pa_batch_attention, caller workspace
    return inp, d


def _static_call(batch, d):
    out = torch.full_like(d["q"], float("nan"))
    binding.decode_attention_static(d["q"], d["k_pool"], d["v_pool"], d["cl"], d["bt"], int(batch.kv_lens.max()),
                                    batch.softmax_scale, out)
    return out


@pytest.mark.gpu
def test_static_entry_point_matches_existing_path_on_calls_in_a_row():
    W = workloads
    # A: 64 decode sequences, Hq 32 / Hkv 8 / D 128, ragged contexts (3 splits); B: Hq 4 / Hkv 1 / D 256, long
    # contexts, few groups (up to 32 splits, several of them empty for the short sequences)
    a = W.random_batch(231, W.QWEN3_8B, n_decode=64, n_prefill=0, max_ctx=2000, max_q=1)
    b = W.random_batch(232, W.GEMMA3_1B, n_decode=13, n_prefill=0, max_ctx=9000, max_q=1)
    inp_a, da = _existing_path(a)
    inp_b, db = _existing_path(b)
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    out_a1 = _static_call(a, da)
    out_b = _static_call(b, db)               # different shape over A's leftovers
    out_a2 = _static_call(a, da)              # and A again over B's
    torch.cuda.synchronize()
    # the calls themselves took nothing from the allocator beyond the three output tensors made here
    assert torch.cuda.memory_allocated() - before <= 2 * (2 * out_a1.numel() * 2 + out_b.numel() * 2)
    for name, out, d in (("A call 1", out_a1, da), ("B call 2", out_b, db), ("A call 3", out_a2, da)):
        gc.check_close(sdev.bits(out), gen.bf16_to_f64(sdev.bits(d["out"])), f"static vs existing path, {name}")
    assert (sdev.bits(out_a1) == sdev.bits(out_a2)).all(), "same inputs, different result: stale scratch leaked in"
    # and against the oracle, like every other parity test
    ref_a, _, _ = gc.run_oracle(a, inp_a)
    gc.check_close(sdev.bits(out_a1), ref_a, "static vs oracle, A")
    ref_b, _, _ = gc.run_oracle(b, inp_b)
    gc.check_close(sdev.bits(out_b), ref_b, "static vs oracle, B")
    for d in (da, db):
        if d["own"]:
            d["pa"].close()
