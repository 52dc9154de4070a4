"""Seeded synthetic batch descriptors shaped like BASELINE.json's configs (C1–C5).

Shared by the tests, ``bench.py`` and (through the tests) the oracle.  Holds NO method
arithmetic: a batch is lengths + block tables + stream ids; values come from ``gen.py`` (host)
or ``device.py`` (device fill of the same streams).  The recipe for every config is stated in
DESIGN.md §"Input recipe" with the SURVEY.md §8(c) reading (R12–R16) it follows.

Batch convention: decode sequences first (``q_len == 1``), then prefill
chunks; ``context_lens[s]`` = tokens cached before this step ("ctx").
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

from . import gen

BLOCK = 16


@dataclass
class Shape:
    num_q_heads: int
    num_kv_heads: int
    head_dim: int
    block_size: int = BLOCK

    @property
    def kv_bytes_per_token(self) -> int:  # K and V, bf16 (SURVEY §8 "kvb")
        return 2 * self.num_kv_heads * self.head_dim * 2

    @property
    def q_bytes_per_token(self) -> int:  # Q (or O), bf16 (SURVEY §8 "qb")
        return self.num_q_heads * self.head_dim * 2


QWEN3_4B = Shape(32, 8, 128)
QWEN3_8B = Shape(32, 8, 128)
GEMMA3_1B = Shape(4, 1, 256)
QWEN3_30B_A3B = Shape(32, 4, 128)
TINY = Shape(8, 2, 128)


@dataclass
class Batch:
    name: str
    shape: Shape
    seed: int
    num_blocks: int
    q_lens: np.ndarray            # int32 [n_seq]
    context_lens: np.ndarray      # int32 [n_seq]
    num_decode_seqs: int
    block_tables: np.ndarray      # int32 [n_seq, max_blocks_per_seq], -1 beyond ceil(kv_len/16)
    cu_seqlens_q: np.ndarray = field(init=False)

    def __post_init__(self):
        self.q_lens = np.asarray(self.q_lens, dtype=np.int32)
        self.context_lens = np.asarray(self.context_lens, dtype=np.int32)
        cu = np.zeros(len(self.q_lens) + 1, dtype=np.int64)
        np.cumsum(self.q_lens, out=cu[1:])
        assert cu[-1] < 2 ** 31
        self.cu_seqlens_q = cu.astype(np.int32)

    @property
    def n_seq(self) -> int:
        return int(len(self.q_lens))

    @property
    def n_tok(self) -> int:
        return int(self.cu_seqlens_q[-1])

    @property
    def n_decode_tok(self) -> int:
        return int(self.q_lens[: self.num_decode_seqs].sum())

    @property
    def r(self) -> float:
        """Realised decode ratio r = n_decode / n_tok."""
        return self.n_decode_tok / max(1, self.n_tok)

    @property
    def kv_lens(self) -> np.ndarray:
        return (self.context_lens.astype(np.int64) + self.q_lens.astype(np.int64))

    @property
    def max_blocks_per_seq(self) -> int:
        return int(self.block_tables.shape[1])

    @property
    def softmax_scale(self) -> float:
        return 1.0 / math.sqrt(self.shape.head_dim)

    # ---- algorithmic work (SURVEY.md §8(d) "Algorithmic work per unit") ----
    def algorithmic_bytes(self) -> int:
        """Attention: KV read once per KV head + Q read + O write + block ids."""
        sh = self.shape
        kv = int(self.kv_lens.sum()) * sh.kv_bytes_per_token
        qo = 2 * self.n_tok * sh.q_bytes_per_token
        bt = int(np.ceil(self.kv_lens / sh.block_size).sum()) * 4
        return kv + qo + bt

    def algorithmic_flops(self) -> int:
        """4·D·Hq·Σ(q·ctx + q(q+1)/2): QKᵀ and PV over the causal pairs only."""
        q = self.q_lens.astype(np.int64)
        c = self.context_lens.astype(np.int64)
        pairs = int((q * c + q * (q + 1) // 2).sum())
        return 4 * self.shape.head_dim * self.shape.num_q_heads * pairs

    def append_bytes(self) -> int:
        return 2 * self.n_tok * self.shape.kv_bytes_per_token

    # ---- host materialisation (small configs / sampled rows) ----
    def q_bits(self) -> np.ndarray:
        sh = self.shape
        n = self.n_tok * sh.num_q_heads * sh.head_dim
        return gen.bf16_normal(self.seed, gen.TENSOR_Q, 0, n).reshape(self.n_tok, sh.num_q_heads, sh.head_dim)

    def kv_new_bits(self):
        sh = self.shape
        n = self.n_tok * sh.num_kv_heads * sh.head_dim
        shp = (self.n_tok, sh.num_kv_heads, sh.head_dim)
        return (gen.bf16_normal(self.seed, gen.TENSOR_K_NEW, 0, n).reshape(shp),
                gen.bf16_normal(self.seed, gen.TENSOR_V_NEW, 0, n).reshape(shp))

    def pool_elems(self) -> int:
        sh = self.shape
        return self.num_blocks * sh.num_kv_heads * sh.block_size * sh.head_dim

    def pool_bits(self):
        """Whole K and V pools by physical linear index (only for pools that fit the host)."""
        n = self.pool_elems()
        return (gen.bf16_normal(self.seed, gen.TENSOR_K_POOL, 0, n),
                gen.bf16_normal(self.seed, gen.TENSOR_V_POOL, 0, n))


def _tables(seed: int, num_blocks: int, kv_lens: np.ndarray, min_width: int = 1) -> np.ndarray:
    """Consecutive slices, in batch order, of one seeded permutation of [0, num_blocks)."""
    nblk = (np.asarray(kv_lens, dtype=np.int64) + BLOCK - 1) // BLOCK
    total = int(nblk.sum())
    if total > num_blocks:
        raise ValueError(f"batch needs {total} blocks, pool has {num_blocks}")
    perm = gen.block_permutation(seed, num_blocks)
    width = max(min_width, int(nblk.max()) if len(nblk) else 1)
    bt = np.full((len(nblk), width), -1, dtype=np.int32)
    off = 0
    for s, n in enumerate(nblk):
        bt[s, :n] = perm[off:off + n]
        off += int(n)
    return bt


def make_batch(name, shape, seed, q_lens, context_lens, num_decode_seqs, num_blocks=None,
               min_table_width: int = 1) -> Batch:
    q_lens = np.asarray(q_lens, dtype=np.int32)
    context_lens = np.asarray(context_lens, dtype=np.int32)
    kv = context_lens.astype(np.int64) + q_lens
    need = int(((kv + BLOCK - 1) // BLOCK).sum())
    if num_blocks is None:
        num_blocks = max(64, -(-need // 1024) * 1024)
    bt = _tables(seed, num_blocks, kv, min_table_width)
    return Batch(name, shape, seed, num_blocks, q_lens, context_lens, int(num_decode_seqs), bt)


def n_decode_for(r: float, n_tok: int) -> int:
    """R12: n_dec = floor(r·n_tok + 0.5)."""
    return int(math.floor(r * n_tok + 0.5))


def config1() -> Batch:
    """C1 tiny: 8/2/128, [dec ctx 48, dec ctx 100, pre 64/ctx 0, pre 64/ctx 0], seed 0, 64 blocks."""
    return make_batch("C1-tiny", TINY, 0, [1, 1, 64, 64], [48, 100, 0, 0], 2, num_blocks=64, min_table_width=8)


def config2(r: float, n_tok: int = 2048, ctx: int = 16, prompt: int = 512, num_blocks: int = 8192) -> Batch:
    """C2 Qwen3-4B shape: n_dec decode seqs at ctx 16 + 512-token prompts (ctx 0) + remainder (R13)."""
    i = int(round(10 * r))
    nd = n_decode_for(r, n_tok)
    npre = n_tok - nd
    q = [1] * nd + [prompt] * (npre // prompt) + ([npre % prompt] if npre % prompt else [])
    c = [ctx] * nd + [0] * (len(q) - nd)
    need = sum(-(-(a + b) // BLOCK) for a, b in zip(q, c))
    nb = max(num_blocks, -(-need // 1024) * 1024)
    return make_batch(f"C2-qwen3-4b-n{n_tok}-r{r:.1f}", QWEN3_4B, 200 + i, q, c, nd, num_blocks=nb)


def config3(n_seq: int = 256, lo: int = 512, hi: int = 4096, num_blocks: int = 65536) -> Batch:
    """C3 Gemma-3-1B shape pure decode: 256 seqs, ctx ~ U{512..4096}, seed 3."""
    rng = np.random.default_rng(3)
    ctx = rng.integers(lo, hi + 1, n_seq)
    return make_batch("C3-gemma3-1b-decode", GEMMA3_1B, 3, [1] * n_seq, ctx, n_seq, num_blocks=num_blocks)


def config4(r: float, n_tok: int = 8192, chunk: int = 2048, num_blocks: int | None = None) -> Batch:
    """C4 Qwen3-8B shape: decode ctx lognormal(median 2048, σ 0.7 — R14) clipped [256, 8192];
    prefill chunks of 2048 over prior ctx ~ U{0..4096}; seed 400+i; pool sized to the batch, or ``num_blocks``
    (``c4_pool_blocks()``: the one pool that serves every r, as bench.py and the full-size parity tests use it)."""
    i = int(round(10 * r))
    nd = n_decode_for(r, n_tok)
    npre = n_tok - nd
    rng = np.random.default_rng(400 + i)
    dc = np.clip(np.exp(rng.normal(math.log(2048), 0.7, nd)), 256, 8192).astype(np.int64)
    nch, rem = npre // chunk, npre % chunk
    pc = rng.integers(0, 4097, nch + (1 if rem else 0))
    q = [1] * nd + [chunk] * nch + ([rem] if rem else [])
    c = list(dc) + list(pc)
    return make_batch(f"C4-qwen3-8b-n{n_tok}-r{r:.1f}", QWEN3_8B, 400 + i, q, c, nd, num_blocks=num_blocks)


_C4_POOL_BLOCKS = None


def c4_pool_blocks() -> int:
    """Blocks of the one pool pair that holds any C4 batch (n_tok 8192, every r of the sweep): the largest need
    (r = 1.0: ~1.3 M blocks x 32 KB per pool = ~42 GB per pool), rounded up to a multiple of 1024."""
    global _C4_POOL_BLOCKS
    if _C4_POOL_BLOCKS is None:
        _C4_POOL_BLOCKS = max(config4(i / 10).num_blocks for i in range(11))
    return _C4_POOL_BLOCKS


def config5(variant: str = "r1.0", n_dec: int = 1024, num_blocks: int | None = None) -> Batch:
    """C5 Qwen3-30B-A3B shape: 1024 decode seqs ctx ~ U{4096..32768}, seed 7; R15 prefill variants
    'r1.0' (none), 'r0.2' (4 chunks × 1024, ctx 0), 'r0.059' (4 chunks × 4096, ctx 0)."""
    rng = np.random.default_rng(7)
    dc = rng.integers(4096, 32769, n_dec)
    pre = {"r1.0": [], "r0.2": [1024] * 4, "r0.059": [4096] * 4}[variant]
    q = [1] * n_dec + pre
    c = list(dc) + [0] * len(pre)
    return make_batch(f"C5-qwen3-30b-a3b-{variant}", QWEN3_30B_A3B, 7, q, c, n_dec, num_blocks=num_blocks)


def random_batch(seed: int, shape: Shape, n_decode: int, n_prefill: int, max_ctx: int, max_q: int,
                 num_blocks: int | None = None) -> Batch:
    """Ragged random batch for parity tests: lengths straddle block (16) and tile (128) edges."""
    rng = np.random.default_rng(seed)
    dc = rng.integers(0, max_ctx + 1, n_decode)
    pq = rng.integers(1, max_q + 1, n_prefill)
    pc = rng.integers(0, max_ctx + 1, n_prefill)
    pc[rng.random(n_prefill) < 0.3] = 0
    q = [1] * n_decode + list(pq)
    c = list(dc) + list(pc)
    return make_batch(f"rand-{seed}", shape, seed, q, c, n_decode, num_blocks=num_blocks)


# ------------------------------------------------------------------------------------------------ N4
# Length statistics of the paper's workloads (App. E.1, Table 9): input range and mean, output
# range, mean and standard deviation.  Only these statistics are used — no dataset item is present or needed.
# (WildChat's input columns in Table 9 count conversation turns, not tokens, so it is left out.)
TABLE9 = {
    "sharegpt-like": dict(in_range=(1, 20448), in_mean=105, out_range=(2, 500), out_mean=280, out_std=153),
    "longbench-like": dict(in_range=(1000, 4000), in_mean=2492, out_range=(1, 19), out_mean=11, out_std=4),
    "numinamath-like": dict(in_range=(16, 1395), in_mean=122, out_range=(800, 3149), out_mean=1039, out_std=228),
}


def _draw_lengths(rng, n: int, lo: int, hi: int, mean: float) -> np.ndarray:
    """n integer lengths in [lo, hi] whose mean is ~`mean`: lognormal (sigma 1) shifted to `lo`, clipped at `hi`;
    for a narrow range (mean near the middle) this is close to uniform, for a long-tailed one it is heavy-tailed."""
    if mean - lo <= 0:
        return np.full(n, lo, dtype=np.int64)
    if (hi - lo) < 4 * (mean - lo):           # mean is not far below the top: uniform around it
        half = min(mean - lo, hi - mean)
        return rng.integers(int(mean - half), int(mean + half) + 1, n)
    mu = math.log(mean - lo) - 0.5           # E[lognormal(mu, 1)] = exp(mu + 1/2)
    return np.clip(lo + np.exp(rng.normal(mu, 1.0, n)), lo, hi).astype(np.int64)


def table9_batch(name: str, r: float, n_tok: int = 2048, shape: Shape = QWEN3_8B, seed: int = 900) -> Batch:
    """One steady-state serving step shaped like a Table 9 workload: n_dec = round(r n_tok) decode
    sequences whose context = prompt length + tokens generated so far (uniform in [0, O)), and prefill prompts drawn
    from the input-length statistics until the remaining token budget is filled (the last one is cut, i.e. chunked
    prefill)."""
    st = TABLE9[name]
    rng = np.random.default_rng(seed + sorted(TABLE9).index(name) * 16 + int(round(10 * r)))
    nd = n_decode_for(r, n_tok)
    L = _draw_lengths(rng, nd, *st["in_range"], st["in_mean"])
    O = np.clip(rng.normal(st["out_mean"], st["out_std"], nd), *st["out_range"]).astype(np.int64)
    dc = L + (rng.random(nd) * O).astype(np.int64)
    q, c = [1] * nd, list(dc)
    left = n_tok - nd
    while left > 0:
        p = int(min(left, _draw_lengths(rng, 1, *st["in_range"], st["in_mean"])[0]))
        q.append(p)
        c.append(0)
        left -= p
    return make_batch(f"N4-{name}-r{r:.1f}", shape, seed, q, c, nd)
