"""Pins for oracle/oracle.c (SURVEY.md §8(c) "What pins the oracle", P1–P15).

Each pin ties the oracle to something other than itself: a differently structured brute-force
evaluation, closed forms, invariants, a library routine (torch SDPA fp64), hand-derived golden
values (tests/golden/).  A plausible mistake in the oracle (dropped term, wrong sign/index,
transposed operand, off-by-one causal bound, wrong GQA map, wrong slot map) fails one of them.
CPU only.
"""
import math
import os

import numpy as np
import pytest

import oracle
from paper_2606_00516_b200.synth import gen, workloads
from tests import helpers

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _run_oracle(batch, inp, rows=None, **kw):
    sh = batch.shape
    osh = oracle.PagedShape(sh.num_q_heads, sh.num_kv_heads, sh.head_dim, sh.block_size)
    kp, vp = inp["k_pool"].copy(), inp["v_pool"].copy()
    oracle.kv_append(osh, inp["k_new"], inp["v_new"], kp, vp, batch.cu_seqlens_q, batch.context_lens,
                     batch.block_tables)
    out = oracle.attention(osh, inp["q"], kp, vp, batch.cu_seqlens_q, batch.context_lens, batch.block_tables,
                           batch.softmax_scale, rows=rows, **kw)
    return out, kp, vp, osh


def _bits(x):
    return gen.f32_to_bf16(np.asarray(x, dtype=np.float32))


def _custom(shape, q, k_seq, v_seq, q_lens, ctx_lens, num_blocks=None, seed=11):
    """Batch with hand-chosen values: k_seq/v_seq[s] are float arrays [kv_len, Hkv, D]; the first ctx
    rows are pre-cached, the rest arrive as k_new/v_new."""
    nd = 0
    batch = workloads.make_batch("custom", shape, seed, q_lens, ctx_lens, nd, num_blocks=num_blocks)
    b = shape.block_size
    shape4 = (batch.num_blocks, shape.num_kv_heads, b, shape.head_dim)
    kp = np.full(shape4, helpers.NAN_BF16, dtype=np.uint16)
    vp = np.full(shape4, helpers.NAN_BF16, dtype=np.uint16)
    k_new, v_new = [], []
    for s in range(batch.n_seq):
        ctx = int(ctx_lens[s])
        for t in range(ctx):
            blk = batch.block_tables[s, t // b]
            kp[blk, :, t % b, :] = _bits(k_seq[s][t])
            vp[blk, :, t % b, :] = _bits(v_seq[s][t])
        k_new.append(_bits(k_seq[s][ctx:]))
        v_new.append(_bits(v_seq[s][ctx:]))
    inp = dict(q=_bits(q), k_new=np.concatenate(k_new), v_new=np.concatenate(v_new), k_pool=kp, v_pool=vp)
    return batch, inp


# ------------------------------------------------------------------ P1 brute force
@pytest.mark.parametrize("case", ["config1", "ragged-a", "ragged-b", "edge-lens"])
def test_p1_bruteforce_dense(case):
    if case == "config1":
        batch = workloads.config1()
    elif case == "ragged-a":
        batch = workloads.random_batch(101, workloads.TINY, n_decode=5, n_prefill=3, max_ctx=70, max_q=40)
    elif case == "ragged-b":
        batch = workloads.random_batch(102, workloads.Shape(4, 1, 64), n_decode=3, n_prefill=4, max_ctx=50, max_q=33)
    else:  # kv_len in {1, 15, 16, 17, 33}, ctx = 0 and q_len = 1 cases
        batch = workloads.make_batch("edge", workloads.Shape(4, 2, 32), 103, [1, 1, 1, 1, 17, 1], [0, 14, 15, 16, 16, 32],
                                     4)
    inp = helpers.host_inputs(batch)
    out, kp, vp, _ = _run_oracle(batch, inp)
    ref = helpers.dense_attention(batch, inp["q"], kp, vp, batch.softmax_scale)
    assert np.isfinite(out).all()
    np.testing.assert_allclose(out, ref, rtol=0, atol=1e-12)


# ------------------------------------------------------------------ P2 softmax rows
def test_p2_weights_sum_to_one_and_nonnegative():
    batch = workloads.config1()
    inp = helpers.host_inputs(batch)
    _, kp, vp, osh = _run_oracle(batch, inp)
    for row in (0, 1, 2, 17, 65, 66, 129):
        for h in (0, 3, 7):
            p, lse = oracle.attention_weights(osh, inp["q"], kp, vp, batch.cu_seqlens_q, batch.context_lens,
                                              batch.block_tables, batch.softmax_scale, row, h)
            s = int(np.searchsorted(batch.cu_seqlens_q, row, side="right") - 1)
            n_j = int(batch.context_lens[s]) + (row - int(batch.cu_seqlens_q[s])) + 1
            assert len(p) == n_j                      # R2/R3: ctx + j + 1 visible keys
            assert (p >= 0).all()
            assert abs(p.sum() - 1.0) < 1e-12
            assert math.isfinite(lse)


def test_p2_weights_match_dense_weights():
    batch = workloads.config1()
    inp = helpers.host_inputs(batch)
    _, kp, vp, osh = _run_oracle(batch, inp)
    _, W = helpers.dense_attention(batch, inp["q"], kp, vp, batch.softmax_scale, return_weights=True)
    row, h, s = 70, 5, 3
    p, _ = oracle.attention_weights(osh, inp["q"], kp, vp, batch.cu_seqlens_q, batch.context_lens,
                                    batch.block_tables, batch.softmax_scale, row, h)
    j = row - int(batch.cu_seqlens_q[s])
    np.testing.assert_allclose(p, W[(s, h)][j, : len(p)], atol=1e-14)
    assert (W[(s, h)][j, len(p):] == 0).all()


# ------------------------------------------------------------------ P3 shift invariance
def test_p3_score_shift_invariance():
    sh = workloads.Shape(2, 1, 16)
    rng = np.random.default_rng(5)
    n = 23
    K = rng.integers(-3, 4, (n, 1, 16)).astype(np.float64)
    V = rng.normal(size=(n, 1, 16))
    q = np.zeros((1, 2, 16))
    q[0, 0, 0], q[0, 1, 0] = 2.0, -1.0            # only component 0 is non-zero
    b1, i1 = _custom(sh, q, [K], [V], [1], [n - 1])
    K2 = K.copy()
    K2[:, :, 0] += 5.0                              # shifts every score of head h by scale*q_h0*5 exactly
    b2, i2 = _custom(sh, q, [K2], [V], [1], [n - 1])
    o1 = _run_oracle(b1, i1)[0]
    o2 = _run_oracle(b2, i2)[0]
    np.testing.assert_allclose(o1, o2, rtol=0, atol=1e-14)


# ------------------------------------------------------------------ P4–P6 PV closed forms
def test_p4_equal_keys_give_mean_of_v():
    sh = workloads.Shape(4, 2, 32)
    rng = np.random.default_rng(6)
    n, qn = 37, 5                                     # prefill of 5 over ctx 32
    K = np.tile(rng.normal(size=(1, 2, 32)), (n, 1, 1))
    V = rng.normal(size=(n, 2, 32))
    q = rng.normal(size=(qn, 4, 32))
    batch, inp = _custom(sh, q, [K], [V], [qn], [n - qn])
    out = _run_oracle(batch, inp)[0]
    Vb = gen.bf16_to_f64(_bits(V))
    for j in range(qn):
        n_j = n - qn + j + 1
        for h in range(4):
            np.testing.assert_allclose(out[j, h], Vb[:n_j, h // 2].mean(axis=0), atol=1e-14)


def test_p5_single_key_returns_v_row_exactly():
    sh = workloads.Shape(4, 2, 32)
    rng = np.random.default_rng(7)
    K, V, q = rng.normal(size=(1, 2, 32)), rng.normal(size=(1, 2, 32)), rng.normal(size=(1, 4, 32))
    batch, inp = _custom(sh, q, [K], [V], [1], [0])
    out = _run_oracle(batch, inp)[0]
    Vb = gen.bf16_to_f64(_bits(V))
    for h in range(4):
        assert (out[0, h] == Vb[0, h // 2]).all()


def test_p6_dominant_key_selects_its_v_row():
    sh = workloads.Shape(2, 2, 16)
    n, star = 20, 13
    K = np.zeros((n, 2, 16)); K[star, :, 0] = 1.0
    rng = np.random.default_rng(8)
    V = rng.normal(size=(n, 2, 16))
    q = np.zeros((1, 2, 16)); q[0, :, 0] = 160.0      # scale*q.k = 0.25*160 = 40 above the rest
    batch, inp = _custom(sh, q, [K], [V], [1], [n - 1])
    out = _run_oracle(batch, inp)[0]
    Vb = gen.bf16_to_f64(_bits(V))
    for h in range(2):
        np.testing.assert_allclose(out[0, h], Vb[star, h], rtol=0, atol=1e-15 + (n * math.exp(-40.0)) * 4)


# ------------------------------------------------------------------ golden closed forms
def _read_golden(name):
    vals = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split("=")
                vals[k.strip()] = [float(x) for x in v.split()]
    return vals


def test_golden_two_key_sigmoid():
    g = _read_golden("attention_closed_forms.txt")
    sh = workloads.Shape(1, 1, 4)                       # scale = 1/sqrt(4) = 0.5
    K = np.array([[[0, 0, 0, 0.0]], [[1, 0, 0, 0.0]]])
    V = np.array([[[1, 0, 2, -4.0]], [[0, 1, 6, 4.0]]])
    q = np.array([[[2, 0, 0, 0.0]]])                    # z = (0, 1)
    batch, inp = _custom(sh, q, [K], [V], [1], [1])
    out, kp, vp, osh = _run_oracle(batch, inp)
    np.testing.assert_allclose(out[0, 0], g["two_key_o"], rtol=0, atol=1e-15)
    p, lse = oracle.attention_weights(osh, inp["q"], kp, vp, batch.cu_seqlens_q, batch.context_lens,
                                      batch.block_tables, batch.softmax_scale, 0, 0)
    np.testing.assert_allclose(p, g["two_key_p"], rtol=0, atol=1e-15)
    np.testing.assert_allclose(lse, g["two_key_lse"][0], rtol=0, atol=1e-15)


def test_golden_causal_three_token_prefill():
    g = _read_golden("attention_closed_forms.txt")
    sh = workloads.Shape(1, 1, 4)
    K = np.zeros((3, 1, 4))                             # all scores 0 -> uniform over visible keys
    V = np.array([[[3, 0, 0, 0.0]], [[0, 3, 0, 0.0]], [[0, 0, 3, 0.0]]])
    q = np.ones((3, 1, 4))
    batch, inp = _custom(sh, q, [K], [V], [3], [0])
    out = _run_oracle(batch, inp)[0]
    for j in range(3):
        np.testing.assert_allclose(out[j, 0], g[f"causal_row{j}"], rtol=0, atol=1e-15)


# ------------------------------------------------------------------ P7–P8 causal / context
def _one_seq(shape, seed, total):
    rng = np.random.default_rng(seed)
    K = rng.normal(size=(total, shape.num_kv_heads, shape.head_dim))
    V = rng.normal(size=(total, shape.num_kv_heads, shape.head_dim))
    q = rng.normal(size=(total, shape.num_q_heads, shape.head_dim))
    return q, K, V


def test_p7_decode_equals_last_row_of_full_prefill():
    sh = workloads.TINY
    c = 52
    q, K, V = _one_seq(sh, 9, c + 1)
    bp, ip = _custom(sh, q, [K], [V], [c + 1], [0])
    full = _run_oracle(bp, ip)[0]
    bd, idd = _custom(sh, q[c:], [K], [V], [1], [c])
    dec = _run_oracle(bd, idd)[0]
    assert (dec[0] == full[c]).all()


def test_p8_chunk_equivalence():
    sh = workloads.Shape(4, 2, 64)
    q, K, V = _one_seq(sh, 10, 128)
    b1, i1 = _custom(sh, q, [K], [V], [128], [0])
    one = _run_oracle(b1, i1)[0]
    b2, i2 = _custom(sh, q[:64], [K[:64]], [V[:64]], [64], [0])
    first = _run_oracle(b2, i2)[0]
    b3, i3 = _custom(sh, q[64:], [K], [V], [64], [64])
    second = _run_oracle(b3, i3)[0]
    assert (one[:64] == first).all() and (one[64:] == second).all()


# ------------------------------------------------------------------ P9–P11 paging / batching
def test_p9_block_relabelling_invariance():
    batch = workloads.config1()
    inp = helpers.host_inputs(batch)
    out = _run_oracle(batch, inp)[0]
    perm = np.random.default_rng(12).permutation(batch.num_blocks)      # new_id = perm[old_id]
    inv = np.argsort(perm)
    b2 = workloads.config1()
    b2.block_tables = np.where(batch.block_tables >= 0, perm[np.maximum(batch.block_tables, 0)], -1).astype(np.int32)
    i2 = dict(inp, k_pool=inp["k_pool"][inv].copy(), v_pool=inp["v_pool"][inv].copy())
    out2 = _run_oracle(b2, i2)[0]
    assert (out == out2).all()


def test_p10_append_then_gather_roundtrip_and_untouched_slots():
    batch = workloads.random_batch(104, workloads.TINY, n_decode=4, n_prefill=3, max_ctx=45, max_q=37)
    inp = helpers.host_inputs(batch)
    _, kp, vp, osh = _run_oracle(batch, inp)
    new_mask = helpers.slot_valid_mask(batch, "kv") & ~helpers.slot_valid_mask(batch, "ctx")
    untouched = ~np.broadcast_to(new_mask[:, None, :, None], kp.shape)
    assert (kp[untouched] == inp["k_pool"][untouched]).all()
    assert (vp[untouched] == inp["v_pool"][untouched]).all()
    for s in range(batch.n_seq):
        ctx, kv = int(batch.context_lens[s]), int(batch.kv_lens[s])
        kg, vg = oracle.kv_gather(osh, kp, vp, batch.block_tables, s, kv)
        q0, q1 = batch.cu_seqlens_q[s], batch.cu_seqlens_q[s + 1]
        assert (kg[ctx:] == inp["k_new"][q0:q1]).all() and (vg[ctx:] == inp["v_new"][q0:q1]).all()
        Kd, Vd = helpers.dense_sequence_kv(batch, kp, vp, s)           # independent numpy gather
        assert (gen.bf16_to_f64(kg) == Kd).all() and (gen.bf16_to_f64(vg) == Vd).all()
        assert not np.isnan(Kd).any()


def test_p11_batch_order_permutation():
    sh = workloads.TINY
    q_lens, ctxs = [1, 1, 9, 30, 1], [20, 3, 0, 17, 64]
    rng = np.random.default_rng(13)
    seqs = []
    for ql, c in zip(q_lens, ctxs):
        seqs.append((rng.normal(size=(ql, 8, 128)), rng.normal(size=(c + ql, 2, 128)), rng.normal(size=(c + ql, 2, 128))))

    def run(order):
        q = np.concatenate([seqs[i][0] for i in order])
        b, inp = _custom(sh, q, [seqs[i][1] for i in order], [seqs[i][2] for i in order],
                         [q_lens[i] for i in order], [ctxs[i] for i in order], seed=14 + order[0])
        out = _run_oracle(b, inp)[0]
        return {i: out[b.cu_seqlens_q[k]:b.cu_seqlens_q[k + 1]] for k, i in enumerate(order)}

    a, b = run([0, 1, 2, 3, 4]), run([3, 0, 4, 2, 1])
    for i in range(5):
        assert (a[i] == b[i]).all()


# ------------------------------------------------------------------ P12 GQA
def test_p12_gqa_mapping():
    rng = np.random.default_rng(15)
    n = 19
    K, V = rng.normal(size=(n, 2, 32)), rng.normal(size=(n, 2, 32))
    q = rng.normal(size=(1, 4, 32))
    q[0, 1] = q[0, 0]                                 # heads 0,1 share KV head 0 and the same q
    q[0, 2] = q[0, 0]                                 # head 2 -> KV head 1: same q, different KV
    batch, inp = _custom(workloads.Shape(4, 2, 32), q, [K], [V], [1], [n - 1])
    out = _run_oracle(batch, inp)[0]
    assert (out[0, 0] == out[0, 1]).all()
    assert not np.allclose(out[0, 0], out[0, 2])
    # Hq == Hkv: head h of the GQA run with KV head h//2 equals an independent MHA run on that KV head
    bm, im = _custom(workloads.Shape(2, 2, 32), q[:, [0, 2]], [K], [V], [1], [n - 1])
    outm = _run_oracle(bm, im)[0]
    assert (outm[0, 0] == out[0, 0]).all() and (outm[0, 1] == out[0, 2]).all()


# ------------------------------------------------------------------ P13 split / merge algebra
def test_p13_partials_merge_to_unsplit():
    batch = workloads.random_batch(105, workloads.TINY, n_decode=2, n_prefill=1, max_ctx=300, max_q=20)
    inp = helpers.host_inputs(batch)
    out, kp, vp, osh = _run_oracle(batch, inp, return_lse=True)
    out, lse = out
    rng = np.random.default_rng(16)
    for row in (0, 1, batch.n_tok - 1):
        s = int(np.searchsorted(batch.cu_seqlens_q, row, side="right") - 1)
        n_j = int(batch.context_lens[s]) + row - int(batch.cu_seqlens_q[s]) + 1
        cuts = np.unique(np.concatenate([[0, n_j], rng.integers(1, max(2, n_j), 4)]))
        cuts = cuts[cuts <= n_j]
        for h in (0, 6):
            parts = [oracle.attention_partial(osh, inp["q"], kp, vp, batch.cu_seqlens_q, batch.context_lens,
                                              batch.block_tables, batch.softmax_scale, row, h, int(a), int(b))
                     for a, b in zip(cuts[:-1], cuts[1:])]
            o, l = oracle.merge([p[0] for p in parts], [p[1] for p in parts], np.stack([p[2] for p in parts]))
            np.testing.assert_allclose(o, out[row, h], rtol=0, atol=1e-13)
            assert abs(l - lse[row, h]) < 1e-12


# ------------------------------------------------------------------ P14 library special case
def test_p14_torch_sdpa_causal_fp64():
    torch = pytest.importorskip("torch")
    sh = workloads.TINY
    G = sh.num_q_heads // sh.num_kv_heads
    n = 77
    q, K, V = _one_seq(sh, 17, n)
    batch, inp = _custom(sh, q, [K], [V], [n], [0])
    out = _run_oracle(batch, inp)[0]
    tq = torch.from_numpy(gen.bf16_to_f64(_bits(q))).permute(1, 0, 2)[None]            # [1,Hq,n,D]
    tk = torch.from_numpy(gen.bf16_to_f64(_bits(K))).permute(1, 0, 2).repeat_interleave(G, 0)[None]
    tv = torch.from_numpy(gen.bf16_to_f64(_bits(V))).permute(1, 0, 2).repeat_interleave(G, 0)[None]
    ref = torch.nn.functional.scaled_dot_product_attention(tq, tk, tv, is_causal=True,
                                                           scale=batch.softmax_scale)[0].permute(1, 0, 2).numpy()
    np.testing.assert_allclose(out, ref, rtol=0, atol=1e-12)


# ------------------------------------------------------------------ P15 timer fit + kappa
def test_p15_fit_exact_lines_and_symmetric_noise():
    n = np.array([512, 1024, 2048, 4096], dtype=np.float64)
    a, b = 3.5e-6, 1.25e-8
    al, be, r2 = oracle.fit(n, a + b * n)
    assert abs(al - a) < 1e-12 * max(1, abs(a)) + 1e-18 and abs(be - b) < 1e-12 * b and abs(r2 - 1) < 1e-12
    nn = np.repeat(n, 2)
    eps = np.tile([1e-7, -1e-7], 4)
    al2, be2, r22 = oracle.fit(nn, a + b * nn + eps)
    assert abs(al2 - a) < 1e-15 and abs(be2 - b) < 1e-18 and r22 < 1.0
    with pytest.raises(ValueError):
        oracle.fit([7, 7, 7], [1, 2, 3])


def test_p15_fit_golden_hand_derived():
    g = _read_golden("fit_closed_forms.txt")
    al, be, r2 = oracle.fit(g["n"], g["T"])
    assert abs(al - g["alpha"][0]) < 1e-14 and abs(be - g["beta"][0]) < 1e-14 and abs(r2 - g["r2"][0]) < 1e-14


def test_kappa_exact_quadratic_and_eq10():
    c0, c1, c2 = 2.0, 5.0, -3.0
    r = np.linspace(0, 1, 11)
    K = c0 + c1 * r + c2 * r * r
    c, kappa = oracle.quadratic_kappa(r, K)
    np.testing.assert_allclose(c, [c0, c1, c2], atol=1e-11)
    assert abs(kappa - 2 * c2 / (c0 + c1 + c2)) < 1e-11          # Eq. 11
    Kbar = (1 - r) * K[0] + r * K[-1]
    np.testing.assert_allclose(K - Kbar, -c[2] * r * (1 - r), atol=1e-11)   # Eq. 10


def test_kappa_literal_value():
    """K(r) = 2 + 5 r - 3 r^2: K(1) = 4, kappa = 2·(-3)/4 = -1.5 (Eq. 11), as a literal."""
    r = np.linspace(0, 1, 11)
    _, kappa = oracle.quadratic_kappa(r, 2 + 5 * r - 3 * r * r)
    assert abs(kappa - (-1.5)) < 1e-11


# ------------------------------------------------------------------ N3: Eq. 3 (theta0) and Eq. 7 (crossover)
def test_eq7_golden_hand_worked():
    g = _read_golden("eq7_closed_forms.txt")
    o = oracle.eq7(*g["params"])
    assert abs(o["beta_eb_w"] - g["beta_eb_w"][0]) < 1e-15
    assert abs(o["lhs"] - g["lhs"][0]) < 1e-15 and abs(o["rhs"] - g["rhs"][0]) < 1e-15
    assert abs(1 / o["tp_eb"] - g["inv_tp_eb"][0]) < 1e-12 and abs(1 / o["tp_mb"] - g["inv_tp_mb"][0]) < 1e-12
    assert o["lhs"] > o["rhs"] and o["tp_mb"] < o["tp_eb"]


def test_eq7_is_the_throughput_comparison_of_prop_3_4():
    """Proposition 3.4: TP_MB > TP_EB  iff  LHS < RHS.  Algebraically 1/TP_MB - 1/TP_EB = (mu_L + mu_O)(LHS - RHS);
    checked on random parameter draws, so a dropped term, a swapped mu or a wrong sign on either side breaks it."""
    rng = np.random.default_rng(77)
    flips = 0
    for _ in range(400):
        ap, ad, amb = rng.uniform(1e-4, 5e-2, 3)
        bp, bd = rng.uniform(1e-6, 1e-4, 2)
        bmb = rng.uniform(0.5, 1.5) * (bp + bd) / 2
        muL, muO = rng.uniform(1, 3000), rng.uniform(1, 3000)
        N = rng.integers(8, 4096)
        th = rng.uniform(0.05, 0.95)
        k0, zeta = max(1.0, np.floor(th * N)), -np.log(1 - th)
        o = oracle.eq7(ap, bp, ad, bd, amb, bmb, muL, muO, zeta, k0, N)
        d_inv = 1 / o["tp_mb"] - 1 / o["tp_eb"]
        assert abs(d_inv - (muL + muO) * (o["lhs"] - o["rhs"])) < 1e-12 * max(1.0, abs(1 / o["tp_eb"]))
        assert (o["tp_mb"] > o["tp_eb"]) == (o["lhs"] < o["rhs"])
        flips += o["lhs"] < o["rhs"]
        # beta_EB^w is a weighted average of beta_p and beta_d, and equals either one when the other weight is 0
        assert min(bp, bd) - 1e-18 <= o["beta_eb_w"] <= max(bp, bd) + 1e-18
    assert 20 < flips < 380                                   # both regimes occur in the sample
    assert abs(oracle.eq7(1, 3e-5, 1, 7e-5, 1, 0, 10, 0, 1, 1, 1)["beta_eb_w"] - 3e-5) < 1e-20
    assert abs(oracle.eq7(1, 3e-5, 1, 7e-5, 1, 0, 0, 10, 1, 1, 1)["beta_eb_w"] - 7e-5) < 1e-20
    with pytest.raises(ValueError):
        oracle.eq7(1, 1, 1, 1, 1, 1, 0, 0, 1, 1, 1)


def test_theta0_golden_and_residual():
    g = _read_golden("eq7_closed_forms.txt")
    for x, th, ze in zip(g["theta0_x"], g["theta0_value"], g["theta0_zeta"]):
        t, z = oracle.theta0(x)
        assert abs(t - th) < 1e-12 and abs(z - ze) < 1e-12
    # Proposition 3.1: theta0 depends only on x = p0 alpha_p / alpha_d, is increasing in it, and solves Eq. 3
    prev = 0.0
    for x in [1e-6, 1e-3, 0.05, 0.3, 1.0, 7.0, 100.0]:
        t, z = oracle.theta0(x)
        assert 0 < t < 1 and t > prev
        assert abs(t / (1 - t) + np.log(1 - t) - x) < 1e-9 * max(1.0, x)
        assert abs(z + np.log(1 - t)) < 1e-12
        prev = t
    # small-x asymptote: theta^2/2 + O(theta^3) = x  ->  theta0 ~ sqrt(2x)
    assert abs(oracle.theta0(1e-8)[0] / np.sqrt(2e-8) - 1) < 1e-3
    with pytest.raises(ValueError):
        oracle.theta0(0.0)
