"""Device-side materialisation of a synthetic batch (torch tensors + the libpa_synth.so fill kernel).

Input generation only.  ``fill_bf16`` writes the same stream as ``gen.bf16_normal`` (bit-for-bit,
checked in tests/test_gpu_parity.py::test_device_generator_matches_host).
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np
import torch

from . import gen
from .workloads import Batch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libpa_synth.so")
_lib = None


def _load():
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise RuntimeError(f"{_LIB_PATH} not built — run `python -m paper_2606_00516_b200.build`")
        _lib = C.CDLL(_LIB_PATH)
        _lib.synth_fill_bf16.argtypes = [C.c_void_p, C.c_int64, C.c_uint64, C.c_uint32, C.c_int64, C.c_void_p]
        _lib.synth_fill_bf16.restype = C.c_int32
        _lib.synth_read_probe.argtypes = [C.c_void_p, C.c_int64, C.c_int32, C.c_void_p, C.c_void_p]
        _lib.synth_read_probe.restype = C.c_int32
    return _lib


def fill_bf16(t: torch.Tensor, seed: int, tensor_id: int, start: int = 0) -> torch.Tensor:
    """Fill a contiguous bf16 CUDA tensor with stream elements [start, start + numel)."""
    assert t.is_cuda and t.dtype == torch.bfloat16 and t.is_contiguous()
    rc = _load().synth_fill_bf16(t.data_ptr(), t.numel(), seed, tensor_id, start, torch.cuda.current_stream().cuda_stream)
    if rc != 0:
        raise RuntimeError(f"synth_fill_bf16 failed: cuda error {rc}")
    return t


def read_probe(buf: torch.Tensor, mode: int, sink: torch.Tensor) -> None:
    """Enqueue one read-only pass over ``buf`` on the current stream (mode 0: ld.global, 1: bulk copies into shared
    memory).  Measurement support for bench.py's read ceiling; ``sink`` is a 1-element int64 CUDA tensor."""
    nbytes = buf.numel() * buf.element_size()
    rc = _load().synth_read_probe(buf.data_ptr(), nbytes - nbytes % 16384, mode, sink.data_ptr(),
                                  torch.cuda.current_stream().cuda_stream)
    if rc != 0:
        raise RuntimeError(f"synth_read_probe failed: cuda error {rc}")


@dataclass
class DeviceBatch:
    batch: Batch
    q: torch.Tensor
    k_new: torch.Tensor
    v_new: torch.Tensor
    k_pool: torch.Tensor
    v_pool: torch.Tensor
    cu_seqlens_q: torch.Tensor
    context_lens: torch.Tensor
    block_tables: torch.Tensor
    out: torch.Tensor


def materialise(batch: Batch, device="cuda:0", pools=None, refill: bool = True) -> DeviceBatch:
    """Allocate and fill every tensor of the batch on the device.  ``pools`` lets callers reuse one
    (k_pool, v_pool) pair across batches of the same shape/num_blocks; it is refilled with the batch's own streams
    unless ``refill`` is False (timing loops that share one resident pool between batches: the values stay seeded
    N(0,1) bf16, only the seed is another batch's)."""
    sh = batch.shape
    dev = torch.device(device)
    n = batch.n_tok
    q = torch.empty((n, sh.num_q_heads, sh.head_dim), dtype=torch.bfloat16, device=dev)
    k_new = torch.empty((n, sh.num_kv_heads, sh.head_dim), dtype=torch.bfloat16, device=dev)
    v_new = torch.empty_like(k_new)
    pshape = (batch.num_blocks, sh.num_kv_heads, sh.block_size, sh.head_dim)
    if pools is None:
        k_pool = torch.empty(pshape, dtype=torch.bfloat16, device=dev)
        v_pool = torch.empty(pshape, dtype=torch.bfloat16, device=dev)
    else:
        k_pool, v_pool = pools
        assert tuple(k_pool.shape) == pshape
    with torch.cuda.device(dev):
        if n:
            fill_bf16(q, batch.seed, gen.TENSOR_Q)
            fill_bf16(k_new, batch.seed, gen.TENSOR_K_NEW)
            fill_bf16(v_new, batch.seed, gen.TENSOR_V_NEW)
        if refill or pools is None:
            fill_bf16(k_pool, batch.seed, gen.TENSOR_K_POOL)
            fill_bf16(v_pool, batch.seed, gen.TENSOR_V_POOL)
    out = torch.zeros_like(q)
    return DeviceBatch(batch, q, k_new, v_new, k_pool, v_pool,
                       torch.from_numpy(batch.cu_seqlens_q).to(dev), torch.from_numpy(batch.context_lens).to(dev),
                       torch.from_numpy(np.ascontiguousarray(batch.block_tables)).to(dev), out)


def bits(t: torch.Tensor) -> np.ndarray:
    """bf16 CUDA/CPU tensor → uint16 bit patterns (numpy, host)."""
    return t.detach().contiguous().view(torch.int16).cpu().numpy().view(np.uint16)
