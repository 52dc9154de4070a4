"""Seeded synthetic input generator (host side, numpy) — shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic (no attention, no softmax, no paging
index map).  It only produces the raw inputs both sides consume:

* ``bf16_normal(seed, tensor_id, start, count)`` — bf16 bit patterns ~N(0,1), a pure
  function of ``(seed, tensor_id, linear_index)`` so that any element of an 84–150 GB
  pool can be regenerated without holding the pool (SURVEY.md §8(d) "Generator").
  ``synth_fill.cu`` implements the *same integer recipe* on the device; the two are
  cross-checked bit-for-bit in ``tests/test_synth.py``.
* ``block_permutation`` — the seeded random permutation block tables are sliced from
  (BASELINE.json configs: "block table a random permutation of free blocks").

Recipe (integer-exact, no floating-point rounding ambiguity between host and device):

    key  = splitmix64(seed * 0x100000001B3 + tensor_id)              (uint64 wrap)
    h0   = splitmix64(key + 2*i), h1 = splitmix64(key + 2*i + 1)
    S    = sum of the twelve 10-bit fields h0[0:60], h1[0:60]         (Irwin–Hall, n = 12)
    x    = (2*S - 12276) * 2**-11         exact in fp32; mean 0, variance 1 - 2**-20
    bf16 = round-to-nearest-even of x to 8 significand bits           (bit trick on the fp32 pattern)
"""
from __future__ import annotations

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_C1 = np.uint64(0xBF58476D1CE4E5B9)
_C2 = np.uint64(0x94D049BB133111EB)
_FNV = 0x100000001B3

# tensor ids used by every workload (so tests, bench and oracle name the same streams)
TENSOR_Q = 1
TENSOR_K_NEW = 2
TENSOR_V_NEW = 3
TENSOR_K_POOL = 4
TENSOR_V_POOL = 5


def _splitmix64(x: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        z = x + _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * _C1
        z = (z ^ (z >> np.uint64(27))) * _C2
        return z ^ (z >> np.uint64(31))


def stream_key(seed: int, tensor_id: int) -> int:
    """64-bit key of one tensor's value stream."""
    x = np.array([(int(seed) * _FNV + int(tensor_id)) & 0xFFFFFFFFFFFFFFFF], dtype=np.uint64)
    return int(_splitmix64(x)[0])


def bf16_normal_at(seed: int, tensor_id: int, index: np.ndarray) -> np.ndarray:
    """bf16 bit patterns (uint16) of the stream at arbitrary linear indices."""
    idx = np.asarray(index, dtype=np.uint64)
    key = np.uint64(stream_key(seed, tensor_id))
    with np.errstate(over="ignore"):
        h0 = _splitmix64(key + np.uint64(2) * idx)
        h1 = _splitmix64(key + np.uint64(2) * idx + np.uint64(1))
    s = np.zeros(idx.shape, dtype=np.int64)
    mask = np.uint64(0x3FF)
    for f in range(6):
        sh = np.uint64(10 * f)
        s += ((h0 >> sh) & mask).astype(np.int64)
        s += ((h1 >> sh) & mask).astype(np.int64)
    x = ((2 * s - 12276).astype(np.float32)) * np.float32(2.0 ** -11)  # exact
    u = x.view(np.uint32)
    u = u + (np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1)))  # RNE to bf16
    return (u >> np.uint32(16)).astype(np.uint16)


def bf16_normal(seed: int, tensor_id: int, start: int, count: int, chunk: int = 1 << 22) -> np.ndarray:
    """bf16 bit patterns of stream elements [start, start+count)."""
    out = np.empty(count, dtype=np.uint16)
    for lo in range(0, count, chunk):
        hi = min(count, lo + chunk)
        out[lo:hi] = bf16_normal_at(seed, tensor_id, np.arange(start + lo, start + hi, dtype=np.uint64))
    return out


def bf16_to_f64(bits: np.ndarray) -> np.ndarray:
    """Exact widening of bf16 bit patterns to float64 (format conversion only)."""
    u = np.asarray(bits, dtype=np.uint16).astype(np.uint32) << np.uint32(16)
    return u.view(np.float32).astype(np.float64)


def f32_to_bf16(x: np.ndarray) -> np.ndarray:
    """RNE fp32 → bf16 bit patterns (finite inputs; NaN maps to a quiet NaN)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    u = x.view(np.uint32)
    r = ((u + (np.uint32(0x7FFF) + ((u >> np.uint32(16)) & np.uint32(1)))) >> np.uint32(16)).astype(np.uint16)
    return np.where(np.isnan(x), np.uint16(0x7FC0), r)


def block_permutation(seed: int, num_blocks: int) -> np.ndarray:
    """Seeded random permutation of [0, num_blocks) (int32) that block tables are sliced from."""
    rng = np.random.Generator(np.random.PCG64(int(seed) + 0x5EED))
    return rng.permutation(num_blocks).astype(np.int32)
