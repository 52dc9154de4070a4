"""Test helpers: host materialisation of a synthetic batch and a brute-force dense evaluation.

Nothing here is imported by the product path.  The dense evaluation is the pin P1 of
SURVEY.md §8(c): a second, differently structured statement of softmax attention (contiguous
un-paged K/V gathered with numpy fancy indexing, full [q_len × kv_len] score matrix, explicit
−inf mask, numpy matmuls) used to pin oracle/oracle.c — it is not the oracle.
"""
from __future__ import annotations

import numpy as np

from paper_2606_00516_b200.synth import gen

NAN_BF16 = np.uint16(0x7FC0)


def slot_valid_mask(batch, upto: str) -> np.ndarray:
    """Bool [num_blocks, block] — slots holding logical positions < ctx ('ctx') or < kv_len ('kv')."""
    b = batch.shape.block_size
    mask = np.zeros((batch.num_blocks, b), dtype=bool)
    lens = batch.context_lens if upto == "ctx" else batch.kv_lens
    for s in range(batch.n_seq):
        n = int(lens[s])
        for i in range((n + b - 1) // b):
            blk = int(batch.block_tables[s, i])
            mask[blk, : min(b, n - i * b)] = True
    return mask


def host_inputs(batch, nan_fill: bool = True):
    """q, k_new, v_new and the pools BEFORE append, pools shaped [nb, Hkv, b, D] (uint16 bf16 bits).

    With ``nan_fill`` every slot that does not hold cached context (positions ≥ ctx, unused
    blocks) is a NaN sentinel, so a missed append or a read past kv_len poisons the result (R8).
    """
    sh = batch.shape
    kp, vp = batch.pool_bits()
    shape4 = (batch.num_blocks, sh.num_kv_heads, sh.block_size, sh.head_dim)
    kp, vp = kp.reshape(shape4).copy(), vp.reshape(shape4).copy()
    if nan_fill:
        invalid = ~slot_valid_mask(batch, "ctx")          # [nb, b]
        kp[np.broadcast_to(invalid[:, None, :, None], shape4)] = NAN_BF16
        vp[np.broadcast_to(invalid[:, None, :, None], shape4)] = NAN_BF16
    k_new, v_new = batch.kv_new_bits()
    return dict(q=batch.q_bits(), k_new=k_new, v_new=v_new, k_pool=kp, v_pool=vp)


def dense_sequence_kv(batch, k_pool, v_pool, s: int):
    """Contiguous fp64 K, V [kv_len, Hkv, D] of sequence s via numpy fancy indexing."""
    b = batch.shape.block_size
    kv_len = int(batch.kv_lens[s])
    t = np.arange(kv_len)
    blk = batch.block_tables[s, t // b]
    K = gen.bf16_to_f64(k_pool[blk, :, t % b, :])
    V = gen.bf16_to_f64(v_pool[blk, :, t % b, :])
    return K, V


def dense_attention(batch, q_bits, k_pool, v_pool, scale: float, return_weights: bool = False):
    """Brute-force fp64 attention [n_tok, Hq, D] from the post-append pools (pin P1)."""
    sh = batch.shape
    G = sh.num_q_heads // sh.num_kv_heads
    out = np.zeros((batch.n_tok, sh.num_q_heads, sh.head_dim))
    weights = {}
    qf = gen.bf16_to_f64(q_bits)
    for s in range(batch.n_seq):
        q0, q1 = int(batch.cu_seqlens_q[s]), int(batch.cu_seqlens_q[s + 1])
        if q1 == q0:
            continue
        ctx = int(batch.context_lens[s])
        K, V = dense_sequence_kv(batch, k_pool, v_pool, s)
        kv_len = K.shape[0]
        jj = np.arange(q1 - q0)[:, None]
        tt = np.arange(kv_len)[None, :]
        visible = tt <= ctx + jj
        for h in range(sh.num_q_heads):
            g = h // G
            S = scale * (qf[q0:q1, h, :] @ K[:, g, :].T)
            S = np.where(visible, S, -np.inf)
            P = np.exp(S - S.max(axis=1, keepdims=True))
            P /= P.sum(axis=1, keepdims=True)
            out[q0:q1, h, :] = P @ V[:, g, :]
            if return_weights:
                weights[(s, h)] = P
    return (out, weights) if return_weights else out
