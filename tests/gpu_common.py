"""Shared plumbing of the -m gpu parity tests: run the CUDA path through the C-ABI binding and the
oracle on the same seeded inputs.  Imports both sides — allowed only under tests/."""
from __future__ import annotations

import numpy as np
import torch

import oracle
from paper_2606_00516_b200 import binding
from paper_2606_00516_b200.synth import device as sdev
from paper_2606_00516_b200.synth import gen
from tests import helpers

MAX_ABS, MEAN_ABS = 2e-2, 2e-3     # north_star tolerance: bf16 in, fp32 accumulate, bf16 out
# Scale-aware bound on top of it: outputs of long contexts are small (|o| ~ sqrt(e/kv_len)), so the
# absolute bound alone would pass errors as large as the output.  Per element
#     |got - ref| <= REL_ELEM * |ref| + REL_RMS * rms(ref)
# with REL_ELEM = 2^-8 (one bf16 ulp of the output; rounding is half of it) and REL_RMS = 8 * 2^-8 (P rounded to
# bf16 before the PV contraction: relative 2^-9 per weight, a random walk over the keys, so a few 2^-9 * rms(ref);
# the factor leaves room for the maximum over millions of elements), and on average
#     mean|got - ref| <= REL_MEAN * mean|ref|,  REL_MEAN = 2^-7.
REL_ELEM, REL_RMS, REL_MEAN = 2.0 ** -8, 8 * 2.0 ** -8, 2.0 ** -7


def bf16_tensor(bits: np.ndarray, dev="cuda:0") -> torch.Tensor:
    return torch.from_numpy(np.ascontiguousarray(bits).view(np.int16)).to(dev).view(torch.bfloat16)


def make_ctx(batch, flags=0, max_tokens=None, **tune):
    sh = batch.shape
    return binding.PagedAttention(sh.num_q_heads, sh.num_kv_heads, sh.head_dim, batch.num_blocks,
                                  max_seqs=max(1, batch.n_seq), max_tokens=max(1, max_tokens or batch.n_tok),
                                  max_blocks_per_seq=batch.max_blocks_per_seq, flags=flags, **tune)


def nan_fill_device(batch, pool: torch.Tensor):
    """Overwrite every slot that holds no cached context with the NaN sentinel (R8)."""
    invalid = torch.from_numpy(~helpers.slot_valid_mask(batch, "ctx")).to(pool.device)     # [nb, 16]
    pool.view(torch.int16).masked_fill_(invalid[:, None, :, None], int(np.int16(np.uint16(0x7FC0).view(np.int16))))


def run_gpu(batch, inp=None, flags=0, repeat=1, pa=None, order="plan_first", tune=None, keep_pool_copy=None,
            pre_append=None):
    """The hot path through the C ABI.  ``inp`` = host_inputs dict (small cases) or None (device fill + NaN
    sentinel).  ``order``:
      "plan_first"  pa_plan, then kv_append + batch_attention back to back — the sequence bench.py times (the attention
                    launch comes up under the append by programmatic dependent launch);
      "graph"       the same, with kv_append + batch_attention captured into a CUDA graph and replayed `repeat` times
                    (bench.py's headline loop);
      "plan_between" kv_append, pa_plan (memset + upload on the stream), batch_attention (the round-1 test order).
    Returns dict of device tensors + the context."""
    dev = "cuda:0"
    if inp is not None:
        d = dict(q=bf16_tensor(inp["q"]), k_new=bf16_tensor(inp["k_new"]), v_new=bf16_tensor(inp["v_new"]),
                 k_pool=bf16_tensor(inp["k_pool"]), v_pool=bf16_tensor(inp["v_pool"]))
    else:
        db = sdev.materialise(batch, dev)
        nan_fill_device(batch, db.k_pool)
        nan_fill_device(batch, db.v_pool)
        d = dict(q=db.q, k_new=db.k_new, v_new=db.v_new, k_pool=db.k_pool, v_pool=db.v_pool)
    if keep_pool_copy is None:
        keep_pool_copy = batch.pool_elems() <= (1 << 29)
    d["pool_before"] = (d["k_pool"].clone(), d["v_pool"].clone()) if keep_pool_copy else None
    cu = torch.from_numpy(batch.cu_seqlens_q).to(dev)
    cl = torch.from_numpy(batch.context_lens).to(dev)
    bt = torch.from_numpy(np.ascontiguousarray(batch.block_tables)).to(dev)
    own = pa is None
    pa = pa or make_ctx(batch, flags, **(tune or {}))
    out = torch.full_like(d["q"], float("nan"))
    if pre_append is not None:
        pre_append(d)               # e.g. checksum the pools before anything is written

    def append():
        pa.kv_append(d["k_new"], d["v_new"], d["k_pool"], d["v_pool"], cu, cl, bt, batch.n_seq, batch.n_tok)

    def attention():
        pa.batch_attention(d["q"], d["k_pool"], d["v_pool"], cu, cl, bt, batch.softmax_scale, out)

    if order == "plan_between":
        append()
        pa.plan(batch.cu_seqlens_q, batch.context_lens, batch.n_seq, batch.num_decode_seqs)
        for _ in range(repeat):
            out.fill_(float("nan"))
            attention()
    elif order == "plan_first":
        pa.plan(batch.cu_seqlens_q, batch.context_lens, batch.n_seq, batch.num_decode_seqs)
        for _ in range(repeat):
            out.fill_(float("nan"))
            append()
            attention()
    elif order == "graph":
        pa.plan(batch.cu_seqlens_q, batch.context_lens, batch.n_seq, batch.num_decode_seqs)
        torch.cuda.synchronize()
        side = torch.cuda.Stream()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side, capture_error_mode="thread_local"):
            append()
            attention()
        for _ in range(max(2, repeat)):
            out.fill_(float("nan"))
            torch.cuda.synchronize()
            graph.replay()
        d["graph"] = graph
    else:
        raise ValueError(order)
    torch.cuda.synchronize()
    d.update(out=out, cu=cu, cl=cl, bt=bt, pa=pa, own=own)
    return d


def oracle_shape(batch):
    sh = batch.shape
    return oracle.PagedShape(sh.num_q_heads, sh.num_kv_heads, sh.head_dim, sh.block_size)


def run_oracle(batch, inp, rows=None, n_threads=8):
    osh = oracle_shape(batch)
    kp, vp = inp["k_pool"].copy(), inp["v_pool"].copy()
    oracle.kv_append(osh, inp["k_new"], inp["v_new"], kp, vp, batch.cu_seqlens_q, batch.context_lens, batch.block_tables)
    ref = oracle.attention(osh, inp["q"], kp, vp, batch.cu_seqlens_q, batch.context_lens, batch.block_tables,
                           batch.softmax_scale, rows=rows, n_threads=n_threads)
    return ref, kp, vp


def check_close(out_bits: np.ndarray, ref: np.ndarray, what=""):
    got = gen.bf16_to_f64(out_bits)
    assert np.isfinite(got).all(), f"{what}: non-finite outputs ({np.count_nonzero(~np.isfinite(got))})"
    err = np.abs(got - ref)
    assert err.max() <= MAX_ABS, f"{what}: max abs err {err.max():.4g} > {MAX_ABS} at {np.unravel_index(err.argmax(), err.shape)}"
    assert err.mean() <= MEAN_ABS, f"{what}: mean abs err {err.mean():.4g} > {MEAN_ABS}"
    # scale-aware bounds, per (token row, q head): the output scale differs by orders of magnitude between a 17-key
    # and a 150k-key row of the same batch
    aref = np.abs(ref)
    rms = np.sqrt((ref * ref).mean(axis=-1, keepdims=True))
    excess = err - (REL_ELEM * aref + REL_RMS * rms)
    assert excess.max() <= 0, (f"{what}: |err| exceeds 2^-8|ref| + 8*2^-8 rms(ref) by {excess.max():.4g} at "
                               f"{np.unravel_index(excess.argmax(), excess.shape)} (err {err.flat[excess.argmax()]:.4g}, "
                               f"row rms {rms.flat[excess.argmax() // ref.shape[-1]]:.4g})")
    ratio = err.mean(axis=-1) / np.maximum(aref.mean(axis=-1), 1e-300)
    assert ratio.max() <= REL_MEAN, f"{what}: mean|err| / mean|ref| = {ratio.max():.4g} > 2^-7 for a (row, head)"
    check_close.last = dict(max_abs=float(err.max()), mean_abs=float(err.mean()),
                            worst_elem_excess=float(excess.max()), worst_row_mean_ratio=float(ratio.max()))
    print(f"[parity] {what}: max_abs {err.max():.3e} mean_abs {err.mean():.3e} | worst elem margin {excess.max():.3e} "
          f"| worst (row, head) mean ratio {ratio.max():.3e} (bound {REL_MEAN:.3e})")
    return float(err.max()), float(err.mean())


def check_sampled_sequences(batch, d, seqs, prefill_row_stride=16, n_threads=8, what=""):
    """Full-size parity on a sample of sequences without a host copy of the pool: the sampled sequences' blocks
    are gathered from the DEVICE pool (post-append) into a compact host pool with relabelled block ids, and the
    oracle runs on the mini-batch made of those sequences only.  Legitimate by the oracle's own invariances
    (P9 block relabelling, P11 batch permutation/subsetting).  Also checks kv_append placement bit-exactly for the
    sampled sequences.  Prefill chunks are checked on every `prefill_row_stride`-th row plus first and last."""
    sh = batch.shape
    b = sh.block_size
    seqs = [int(s) for s in seqs]
    dec = [s for s in seqs if s < batch.num_decode_seqs]
    pre = [s for s in seqs if s >= batch.num_decode_seqs]
    order = dec + pre                                            # decode first (R11)
    q_lens = batch.q_lens[order]
    ctx = batch.context_lens[order]
    kv = ctx.astype(np.int64) + q_lens
    nblk = (kv + b - 1) // b
    width = int(nblk.max())
    tables = np.full((len(order), width), -1, dtype=np.int32)
    phys = []
    off = 0
    for i, s in enumerate(order):
        n = int(nblk[i])
        tables[i, :n] = np.arange(off, off + n, dtype=np.int32)
        phys.append(batch.block_tables[s, :n].astype(np.int64))
        off += n
    phys = torch.from_numpy(np.concatenate(phys)).to(d["k_pool"].device)
    kp = sdev.bits(d["k_pool"].index_select(0, phys))            # [off, Hkv, b, D] compact, post-append
    vp = sdev.bits(d["v_pool"].index_select(0, phys))
    rows_src = np.concatenate([np.arange(batch.cu_seqlens_q[s], batch.cu_seqlens_q[s + 1]) for s in order])
    idx = torch.from_numpy(rows_src).to(d["q"].device)
    q = sdev.bits(d["q"].index_select(0, idx))
    out = sdev.bits(d["out"].index_select(0, idx))
    k_new = sdev.bits(d["k_new"].index_select(0, idx))
    v_new = sdev.bits(d["v_new"].index_select(0, idx))
    cu = np.zeros(len(order) + 1, dtype=np.int32)
    np.cumsum(q_lens, out=cu[1:])
    # ---- append placement, bit-exact: token j of sequence i sits in slot(ctx_i + j)
    for i in range(len(order)):
        t = ctx[i] + np.arange(q_lens[i])
        blk = tables[i, t // b]
        assert (kp[blk, :, t % b, :] == k_new[cu[i]:cu[i + 1]]).all(), f"{what}: K append placement, seq {order[i]}"
        assert (vp[blk, :, t % b, :] == v_new[cu[i]:cu[i + 1]]).all(), f"{what}: V append placement, seq {order[i]}"
    # ---- attention on the sampled rows
    rows = []
    for i in range(len(order)):
        r = np.arange(cu[i], cu[i + 1])
        if i >= len(dec) and len(r) > 2:
            r = np.unique(np.concatenate([r[::prefill_row_stride], r[:1], r[-1:]]))
        rows.append(r)
    rows = np.concatenate(rows).astype(np.int64)
    ref = oracle.attention(oracle_shape(batch), q, kp, vp, cu, ctx, tables, batch.softmax_scale, rows=rows,
                           n_threads=n_threads)
    return check_close(out[rows], ref, what)


# ------------------------------------------------------------------------------------------------ full-size pool checks
_CHUNK = 1 << 27      # elements per checksum chunk (256 MB of bf16)


def _weights(dev):
    g = torch.Generator(device=dev)
    g.manual_seed(12345)
    return torch.randint(1, 1 << 15, (_CHUNK,), dtype=torch.int32, device=dev, generator=g)


def pool_checksum(pool: torch.Tensor, w: torch.Tensor) -> int:
    """Position-weighted checksum of the pool's bit patterns: sum over all elements of bits(e) * w[index(e) mod CHUNK]
    (mod 2^64), computed chunk by chunk on the device, so a 75 GB pool needs ~1.5 GB of temporaries."""
    flat = pool.view(torch.int16).view(-1)
    total = 0
    for i in range(0, flat.numel(), _CHUNK):
        c = flat[i:i + _CHUNK]
        total += int((c.to(torch.int32) * w[: c.numel()]).sum(dtype=torch.int64).item())
    return total & ((1 << 64) - 1)


def append_targets(batch, dev):
    """Linear element offsets [n_tok, Hkv, D] (int64, device) of the slots kv_append must write, from the oracle-side
    definition slot(s, t) = (block_tables[s][t // 16], t % 16) and the documented pool layout."""
    sh = batch.shape
    b = sh.block_size
    rows_seq = np.repeat(np.arange(batch.n_seq), batch.q_lens)
    j = np.arange(batch.n_tok) - batch.cu_seqlens_q[:-1][rows_seq]
    t = batch.context_lens[rows_seq].astype(np.int64) + j
    blk = batch.block_tables[rows_seq, t // b].astype(np.int64)
    base = (blk * sh.num_kv_heads * b + (t % b)) * sh.head_dim                       # head 0, d 0
    off = base[:, None, None] + (np.arange(sh.num_kv_heads, dtype=np.int64) * b * sh.head_dim)[None, :, None] + \
        np.arange(sh.head_dim, dtype=np.int64)[None, None, :]
    return torch.from_numpy(off).to(dev)


def expected_checksum_after_append(before: int, pool_old_at_targets, new_rows, targets, w) -> int:
    """Checksum the pool must have after kv_append if exactly the target slots changed to the new rows."""
    wt = w[(targets % _CHUNK).view(-1)].to(torch.int64)
    delta = ((new_rows.view(torch.int16).view(-1).to(torch.int64) - pool_old_at_targets.view(torch.int16).view(-1).to(torch.int64)) * wt).sum()
    return (before + int(delta.item())) & ((1 << 64) - 1)
