"""-m gpu parity tests: the CUDA path through the C ABI vs the fp64 oracle on the same seeded inputs.

Bar (north_star): kv_append placement and block-table gathers bit-exact; attention max abs error
<= 2e-2 and mean abs error <= 2e-3 (bf16 in, fp32 accumulate, bf16 out).  Every pool slot that holds
no cached context is a NaN sentinel and every unused table entry is -1 (R8), so a stray read or a
missed append poisons the output.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_00516_b200 import binding
from paper_2606_00516_b200.synth import device as sdev
from paper_2606_00516_b200.synth import gen, workloads
from tests import gpu_common as gc
from tests import helpers

pytestmark = pytest.mark.gpu


def _small_case(name):
    W = workloads
    if name == "C1":
        return W.config1()
    if name == "ragged-tiny":
        return W.random_batch(201, W.TINY, n_decode=9, n_prefill=4, max_ctx=300, max_q=150)
    if name == "ragged-g4-d128":
        return W.random_batch(202, W.QWEN3_4B, n_decode=17, n_prefill=3, max_ctx=700, max_q=260)
    if name == "ragged-g8-d128":
        return W.random_batch(203, W.QWEN3_30B_A3B, n_decode=11, n_prefill=2, max_ctx=500, max_q=130)
    if name == "ragged-g4-d256":
        return W.random_batch(204, W.GEMMA3_1B, n_decode=13, n_prefill=3, max_ctx=900, max_q=140)
    if name == "ragged-g1-d128":
        return W.random_batch(205, W.Shape(4, 4, 128), n_decode=7, n_prefill=2, max_ctx=200, max_q=70)
    if name == "ragged-g8-d256":    # widest group at the larger head size
        return W.random_batch(212, W.Shape(16, 2, 256), n_decode=9, n_prefill=2, max_ctx=600, max_q=200)
    if name == "ragged-g3-d128":    # odd group: the second head group of a prefill unit has one active q-head tile
        return W.random_batch(213, W.Shape(6, 2, 128), n_decode=10, n_prefill=3, max_ctx=500, max_q=260)
    if name == "ragged-g5-d128":
        return W.random_batch(214, W.Shape(5, 1, 128), n_decode=8, n_prefill=2, max_ctx=400, max_q=150)
    if name == "ragged-g2-d256":
        return W.random_batch(215, W.Shape(4, 2, 256), n_decode=8, n_prefill=3, max_ctx=700, max_q=300)
    if name == "edge-lens":     # kv_len in {1, 15, 16, 17, 33, 128, 129}
        return W.make_batch("edge", W.TINY, 206, [1, 1, 1, 1, 1, 1, 1, 17, 1, 128, 129],
                            [0, 14, 15, 16, 32, 127, 128, 16, 0, 0, 127], 7)
    if name == "decode-only":
        return W.random_batch(207, W.QWEN3_8B, n_decode=64, n_prefill=0, max_ctx=2000, max_q=1)
    if name == "prefill-only":
        return W.random_batch(208, W.QWEN3_8B, n_decode=0, n_prefill=3, max_ctx=400, max_q=300)
    raise KeyError(name)


SMALL = ["C1", "ragged-tiny", "ragged-g4-d128", "ragged-g8-d128", "ragged-g4-d256", "ragged-g1-d128", "ragged-g8-d256",
         "ragged-g3-d128", "ragged-g5-d128", "ragged-g2-d256", "edge-lens",
         "decode-only", "prefill-only"]


def test_device_generator_matches_host():
    n = 1 << 16
    for seed, tid, start in [(0, gen.TENSOR_Q, 0), (7, gen.TENSOR_K_POOL, 3_000_000_001), (203, gen.TENSOR_V_NEW, 12345)]:
        t = torch.empty(n + 3, dtype=torch.bfloat16, device="cuda:0")
        sdev.fill_bf16(t, seed, tid, start)
        assert (sdev.bits(t) == gen.bf16_normal(seed, tid, start, n + 3)).all()


@pytest.mark.parametrize("name", SMALL)
def test_kv_append_and_gather_bit_exact(name):
    batch = _small_case(name)
    inp = helpers.host_inputs(batch)
    d = gc.run_gpu(batch, inp)
    _, kp, vp = gc.run_oracle(batch, inp, rows=np.zeros(0, dtype=np.int64))
    assert (sdev.bits(d["k_pool"]) == kp).all(), "K pool differs from the oracle's after append"
    assert (sdev.bits(d["v_pool"]) == vp).all(), "V pool differs from the oracle's after append"
    osh = gc.oracle_shape(batch)
    sh = batch.shape
    for s in range(batch.n_seq):
        kv = int(batch.kv_lens[s])
        if kv == 0:
            continue
        k_out = torch.empty((kv, sh.num_kv_heads, sh.head_dim), dtype=torch.bfloat16, device="cuda:0")
        v_out = torch.empty_like(k_out)
        d["pa"].kv_gather(d["k_pool"], d["v_pool"], d["bt"][s], kv, k_out, v_out)
        kg, vg = oracle.kv_gather(osh, kp, vp, batch.block_tables, s, kv)
        assert (sdev.bits(k_out) == kg).all() and (sdev.bits(v_out) == vg).all()


MODE_FLAGS = {0: 0, 1: binding.PA_FLAG_PREFILL_P_SMEM}     # prefill variant: P staged in TMEM (default) / in shared memory


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("name", SMALL)
def test_attention_parity_small(name, mode):
    batch = _small_case(name)
    inp = helpers.host_inputs(batch)
    d = gc.run_gpu(batch, inp, flags=MODE_FLAGS[mode])
    assert d["pa"].plan_info(8) == mode
    ref, kp, vp = gc.run_oracle(batch, inp)
    assert (sdev.bits(d["k_pool"]) == kp).all() and (sdev.bits(d["v_pool"]) == vp).all()
    gc.check_close(sdev.bits(d["out"]), ref, f"{name}/mode{mode}")


@pytest.mark.parametrize("seed", range(300, 314))
def test_random_shapes_and_mixes(seed):
    """Shapes and mixes nobody picked by hand: head_dim, KV heads, group size 1..8, decode / prefill counts and length
    ranges are all drawn from the seed; every row against the oracle, pools bit-exact, alternating launch orders."""
    rng = np.random.default_rng(seed)
    d = int(rng.choice([128, 256]))
    hkv = int(rng.choice([1, 2, 4, 8]))
    g = int(rng.integers(1, min(8, 32 // hkv) + 1))
    n_dec, n_pre = int(rng.integers(0, 48)), int(rng.integers(0, 4))
    if n_dec + n_pre == 0:
        n_dec = 1
    batch = workloads.random_batch(seed, workloads.Shape(hkv * g, hkv, d), n_dec, n_pre,
                                   max_ctx=int(rng.choice([40, 300, 1500])), max_q=int(rng.choice([20, 130, 300])))
    inp = helpers.host_inputs(batch)
    dd = gc.run_gpu(batch, inp, flags=(0, binding.PA_FLAG_PREFILL_P_SMEM)[seed % 3 == 0], order=("plan_first", "graph")[seed % 2])
    ref, kp, vp = gc.run_oracle(batch, inp)
    assert (sdev.bits(dd["k_pool"]) == kp).all() and (sdev.bits(dd["v_pool"]) == vp).all(), "pools differ after append"
    gc.check_close(sdev.bits(dd["out"]), ref, f"fuzz seed {seed}: Hq {hkv * g} Hkv {hkv} D {d}, {n_dec} decode + {n_pre} prefill")


def test_one_bundle_per_stream_leaves_none_over():
    """Planner (host logic, needs a device only for the upload): with one static bundle per stream no bundle may be left
    over for a second wave, whatever the mix of short (uncut) and long groups; checked on 80 seed-drawn batches (plans only)."""
    rng = np.random.default_rng(4242)
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    seen_k1 = 0
    for i in range(80):
        hkv = int(rng.choice([1, 2, 4, 8]))
        shape = workloads.Shape(hkv * int(rng.integers(1, 5)), hkv, int(rng.choice([128, 256])))
        n_dec = int(rng.integers(200, 3000))
        ctx_hi = int(rng.choice([16, 40, 128, 300, 700]))
        n_pre = int(rng.integers(0, 3))
        batch = workloads.random_batch(5000 + i, shape, n_dec, n_pre, max_ctx=ctx_hi, max_q=200)
        pa = gc.make_ctx(batch)
        pa.plan(batch.cu_seqlens_q, batch.context_lens, batch.n_seq, batch.num_decode_seqs)
        if pa.plan_info(7) == 1 and pa.plan_info(10) == 1:
            seen_k1 += 1
            streams = (sms - pa.plan_info(6)) * 8
            assert pa.plan_info(1) <= streams, (f"batch {i}: {pa.plan_info(1)} bundles for {streams} streams "
                                                f"({n_dec} decode seqs, ctx <= {ctx_hi}, Hkv {hkv})")
        pa.close()
    assert seen_k1 >= 40


@pytest.mark.parametrize("order", ["plan_between", "graph"])
@pytest.mark.parametrize("name", ["C1", "ragged-g4-d128", "ragged-g4-d256", "edge-lens", "decode-only", "prefill-only"])
def test_call_orders_small(name, order):
    """The same result whether the plan is uploaded between append and attention (round-1 test order) or the
    append -> attention pair is replayed from a CUDA graph after planning (bench.py's headline loop)."""
    batch = _small_case(name)
    inp = helpers.host_inputs(batch)
    d = gc.run_gpu(batch, inp, order=order, repeat=2)
    ref, kp, vp = gc.run_oracle(batch, inp)
    assert (sdev.bits(d["k_pool"]) == kp).all() and (sdev.bits(d["v_pool"]) == vp).all()
    gc.check_close(sdev.bits(d["out"]), ref, f"{name}/{order}")


@pytest.mark.parametrize("tune", [dict(tune_prefill_ctas=1), dict(tune_prefill_ctas=100), dict(tune_bundles_per_stream=4),
                                  dict(tune_bundles_per_stream=1, tune_min_bundle_blocks=1),
                                  dict(tune_min_bundle_blocks=64), dict(tune_levels=8), dict(tune_levels=3, tune_bundles_per_stream=2),
                                  dict(tune_levels=8, tune_min_bundle_blocks=64)])
def test_planner_knobs_change_the_schedule_not_the_result(tune):
    """pa_config.tune_* (the documented replacements of round 1's environment variables): any setting is a valid plan."""
    batch = _small_case("ragged-g4-d128")
    inp = helpers.host_inputs(batch)
    ref, _, _ = gc.run_oracle(batch, inp)
    d = gc.run_gpu(batch, inp, tune=tune)
    if "tune_prefill_ctas" in tune:
        assert d["pa"].plan_info(6) == min(tune["tune_prefill_ctas"], 147, d["pa"].plan_info(3) * 8 * 2)
    if "tune_bundles_per_stream" in tune:
        assert d["pa"].plan_info(7) == tune["tune_bundles_per_stream"]
    if "tune_levels" in tune:
        assert d["pa"].plan_info(10) == tune["tune_levels"]
    gc.check_close(sdev.bits(d["out"]), ref, f"knobs/{tune}")
    long = workloads.make_batch("split", workloads.GEMMA3_1B, 209, [1, 1, 1], [5000, 3333, 4097], 3)
    inp = helpers.host_inputs(long)
    ref, _, _ = gc.run_oracle(long, inp)
    d = gc.run_gpu(long, inp, tune=tune, repeat=2)
    gc.check_close(sdev.bits(d["out"]), ref, f"knobs-long/{tune}")


@pytest.mark.parametrize("levels", [2, 8])
@pytest.mark.parametrize("r", [0.5, 1.0])
def test_guided_handout_many_groups_per_bundle(r, levels):
    """Guided hand-out (pa_config.tune_levels, PlanView::n_levels): bundles of many short groups taken piece by piece,
    every row against the oracle, twice on one plan (tickets and queue reset).  min_bundle_blocks makes the bundles long."""
    batch = workloads.config2(r, n_tok=1024, ctx=40)
    inp = helpers.host_inputs(batch)
    ref, kp, vp = gc.run_oracle(batch, inp)
    d = gc.run_gpu(batch, inp, tune=dict(tune_levels=levels, tune_min_bundle_blocks=96), repeat=2)
    assert d["pa"].plan_info(10) == levels
    assert (sdev.bits(d["k_pool"]) == kp).all() and (sdev.bits(d["v_pool"]) == vp).all()
    gc.check_close(sdev.bits(d["out"]), ref, f"guided/r{r}/L{levels}")


@pytest.mark.parametrize("name", ["C1", "ragged-g4-d128", "ragged-g4-d256"])
def test_debug_simple_kernel_parity(name):
    batch = _small_case(name)
    inp = helpers.host_inputs(batch)
    d = gc.run_gpu(batch, inp, flags=binding.PA_FLAG_DEBUG_SIMPLE)
    ref, _, _ = gc.run_oracle(batch, inp)
    gc.check_close(sdev.bits(d["out"]), ref, name + "/simple")


def test_split_kv_groups_merge_in_launch():
    """Few long decode sequences: every (seq, head) group is cut into many items -> partials + last-arriver merge."""
    W = workloads
    batch = W.make_batch("split", W.GEMMA3_1B, 209, [1, 1, 1], [5000, 3333, 4097], 3)
    inp = helpers.host_inputs(batch)
    d = gc.run_gpu(batch, inp, repeat=3)          # repeat: counters must self-reset between launches
    assert d["pa"].plan_info(2) > 3, "expected split items"
    ref, _, _ = gc.run_oracle(batch, inp)
    gc.check_close(sdev.bits(d["out"]), ref, "split")


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("shape_name", ["QWEN3_4B", "GEMMA3_1B"])
def test_prefill_running_max_growth(shape_name, mode):
    """Scores that grow along the keys: the prefill softmax exponentiates a tile against the reference max left by
    earlier tiles, so the three regimes must all match the oracle: growth below 2^8 (reference kept),
    above 2^8 (lazy rescale of l and O at the next tile) and above 2^64 within one tile (exact power-of-two fix-up)."""
    W = workloads
    shape = getattr(W, shape_name)
    ctx, q_len = 500, 300
    batch = W.make_batch("growth", shape, 211, [1, q_len], [40, ctx], 1)
    inp = helpers.host_inputs(batch)
    gain = {0: 0.0, 1: 12.0, 2: 12.0, 3: 120.0, 4: 120.0, 5: 1.0}      # per 128 keys; the rest keeps its N(0,1) draw
    b = shape.block_size
    bits = lambda v: gen.f32_to_bf16(np.array([v], dtype=np.float32))[0]
    row0 = int(batch.cu_seqlens_q[1])
    inp["q"][row0:row0 + q_len, :, 0] = bits(8.0)
    for t in range(ctx + q_len):
        if t // 128 not in gain:
            continue
        v = bits(gain[t // 128])
        if t < ctx:
            inp["k_pool"][int(batch.block_tables[1, t // b]), :, t % b, 0] = v
        else:
            inp["k_new"][row0 + t - ctx, :, 0] = v
    d = gc.run_gpu(batch, inp, flags=MODE_FLAGS[mode])
    ref, _, _ = gc.run_oracle(batch, inp)
    gc.check_close(sdev.bits(d["out"]), ref, f"growth/{shape_name}/mode{mode}")


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("shape_name", ["QWEN3_4B", "GEMMA3_1B"])
def test_prefill_overflow_rows_are_recomputed(shape_name, mode):
    """Beyond the one-pass limit: the scores of one 128-key tile exceed everything before them by > 2^127 (here ~200
    and ~400 nats).  The tensor-core pass overflows for those rows, the launch detects it (row sum not finite) and
    its last CTA recomputes them with the plain loop (include/pa.h "Range"): the result is still the oracle's."""
    W = workloads
    shape = getattr(W, shape_name)
    ctx, q_len = 500, 300
    batch = W.make_batch("overflow", shape, 217, [1, q_len, 70], [40, ctx, 300], 1)
    inp = helpers.host_inputs(batch)
    scale = batch.softmax_scale
    gain = {2: 200.0 / (8.0 * scale), 4: 400.0 / (8.0 * scale), 5: 0.0}     # nats above the N(0,1) background, per 128 keys
    b = shape.block_size
    bits = lambda v: gen.f32_to_bf16(np.array([v], dtype=np.float32))[0]
    row0 = int(batch.cu_seqlens_q[1])
    inp["q"][row0:row0 + q_len, :, 0] = bits(8.0)
    for t in range(ctx + q_len):
        if t // 128 not in gain:
            continue
        v = bits(gain[t // 128])
        if t < ctx:
            inp["k_pool"][int(batch.block_tables[1, t // b]), :, t % b, 0] = v
        else:
            inp["k_new"][row0 + t - ctx, :, 0] = v
    d = gc.run_gpu(batch, inp, flags=MODE_FLAGS[mode], repeat=2)        # repeat: the redo counter must self-reset
    redone = int(d["pa"].workspace[:64].view(torch.int32)[4].item())    # workspace counter [4]: rows redone since pa_plan
    assert redone >= 2 * 100 * shape.num_q_heads, f"expected the overflow rows to take the redo path, got {redone}"
    ref, _, _ = gc.run_oracle(batch, inp)
    gc.check_close(sdev.bits(d["out"]), ref, f"overflow/{shape_name}/mode{mode}")


@pytest.mark.parametrize("shape_name,ctx", [("GEMMA3_1B", 150000), ("QWEN3_30B_A3B", 60000)])
def test_one_long_sequence_split_over_every_worker(shape_name, ctx):
    """A single decode sequence with a very long context: its (sequence, KV head) groups are cut into as many parts
    as there are decode streams (hundreds per group), all merged in the launch by whichever stream arrives last."""
    W = workloads
    batch = W.make_batch("long1", getattr(W, shape_name), 216, [1], [ctx], 1)
    d = gc.run_gpu(batch, None, repeat=2)
    assert d["pa"].plan_info(2) >= 148, "expected the groups to be split across the streams"
    gc.check_sampled_sequences(batch, d, [0], what=f"long1/{shape_name}")


@pytest.mark.parametrize("shape_name,ctx", [("GEMMA3_1B", 150000), ("QWEN3_30B_A3B", 60000)])
def test_long_sequence_with_peaked_scores(shape_name, ctx):
    """The same split-over-every-stream launch with O(1) outputs: four keys far apart score ~25 nats above the
    N(0,1) background (which carries e^12..13 of mass in total), so the result is essentially the mean of their V
    rows and an error in any part's (m, l, o) or in the merge shows at full scale, not at the 1/sqrt(kv_len) scale of
    a flat softmax."""
    W = workloads
    shape = getattr(W, shape_name)
    batch = W.make_batch("long1-peaked", shape, 218, [1], [ctx], 1)
    peaks = [7, ctx // 3 + 5, (2 * ctx) // 3 + 11, ctx - 2]

    def peak(d):
        d["q"][0, :, 0] = 8.0
        val = 25.0 / (8.0 * batch.softmax_scale)
        for t in peaks:
            d["k_pool"][int(batch.block_tables[0, t // 16]), :, t % 16, 0] = val
    d = gc.run_gpu(batch, None, repeat=2, pre_append=peak)
    assert d["pa"].plan_info(2) >= 148
    gc.check_sampled_sequences(batch, d, [0], what=f"long1-peaked/{shape_name}")
    assert float(d["out"].float().abs().mean()) > 0.1, "outputs should be O(1) in this case"


def test_repeated_launches_are_deterministic_and_reset_state():
    batch = _small_case("ragged-g4-d128")
    inp = helpers.host_inputs(batch)
    d1 = gc.run_gpu(batch, inp, repeat=1)
    d2 = gc.run_gpu(batch, inp, repeat=4)
    assert (sdev.bits(d1["out"]) == sdev.bits(d2["out"])).all()


def _device_pool_is_the_host_stream(batch, pool_bits, tensor_id, seed=1):
    """The device-filled pool must be the seeded host stream (sampled), so the oracle's inputs are not the CUDA path's."""
    idx = np.random.default_rng(seed).integers(0, batch.pool_elems(), 4096)
    valid = helpers.slot_valid_mask(batch, "ctx")
    flat_valid = np.broadcast_to(valid[:, None, :, None], pool_bits.shape).reshape(-1)[idx]
    host = gen.bf16_normal_at(batch.seed, tensor_id, idx.astype(np.uint64))
    assert (pool_bits.reshape(-1)[idx][flat_valid] == host[flat_valid]).all()


@pytest.mark.parametrize("order", ["plan_first", "graph"])
@pytest.mark.parametrize("r", [i / 10 for i in range(11)])
def test_config2_timed_sequence_all_rows(r, order):
    """C2 at every r of the sweep, in exactly the sequence bench.py times: pa_plan first, then kv_append and
    batch_attention back to back (the attention launch comes up under the append by programmatic dependent launch),
    eagerly and replayed from a CUDA graph.  ALL 2048 x 32 output rows vs the oracle; both pools bit-exact."""
    batch = workloads.config2(r)
    d = gc.run_gpu(batch, None, order=order, repeat=2)
    inp = dict(q=batch.q_bits(), k_new=batch.kv_new_bits()[0], v_new=batch.kv_new_bits()[1],
               k_pool=sdev.bits(d["pool_before"][0]), v_pool=sdev.bits(d["pool_before"][1]))
    _device_pool_is_the_host_stream(batch, inp["k_pool"], gen.TENSOR_K_POOL)
    ref, kp, vp = gc.run_oracle(batch, inp, n_threads=16)
    assert (sdev.bits(d["k_pool"]) == kp).all() and (sdev.bits(d["v_pool"]) == vp).all()
    gc.check_close(sdev.bits(d["out"]), ref, f"{batch.name}/{order}")


@pytest.mark.parametrize("ctx,r", [(128, 0.8), (64, 0.6), (256, 0.2), (512, 1.0)])
def test_ctx_sweep_points_parity(ctx, r):
    """N2 shapes (n_tok 1024, decode ctx 64..512): mixed launches whose decode groups are short enough never to be
    cut, so bundles close per group (the bundle list must hold one bundle per group) — sampled rows vs the oracle."""
    batch = workloads.config2(r, n_tok=1024, ctx=ctx, num_blocks=40960)
    d = gc.run_gpu(batch, None)
    rng = np.random.default_rng(ctx)
    seqs = list(rng.choice(batch.num_decode_seqs, 48, replace=False)) + list(range(batch.num_decode_seqs, batch.n_seq))
    gc.check_sampled_sequences(batch, d, seqs, prefill_row_stride=8, what=batch.name + f"/ctx{ctx}")
    assert torch.isfinite(d["out"].float()).all()


@pytest.mark.parametrize("name,r", [("sharegpt-like", 0.5), ("numinamath-like", 0.9), ("longbench-like", 0.5)])
def test_table9_shaped_batches_parity(name, r):
    """N4: steady-state steps whose context / prompt lengths follow the statistics of the paper's Table 9
     — ragged decode contexts plus chunked prompts in one mixed launch, sampled vs the oracle."""
    import gc as pygc
    pygc.collect()
    torch.cuda.empty_cache()
    batch = workloads.table9_batch(name, r)
    d = gc.run_gpu(batch, None)
    rng = np.random.default_rng(9)
    seqs = list(rng.choice(batch.num_decode_seqs, 40, replace=False)) + list(range(batch.num_decode_seqs, batch.n_seq))
    gc.check_sampled_sequences(batch, d, seqs, prefill_row_stride=16, what=batch.name)
    assert torch.isfinite(d["out"].float()).all()


def test_config3_all_rows():
    """C3 (Gemma-3-1B shape, 256 decode sequences): every output row vs the oracle, pools bit-exact."""
    batch = workloads.config3()
    d = gc.run_gpu(batch, None)
    inp = dict(q=batch.q_bits(), k_new=batch.kv_new_bits()[0], v_new=batch.kv_new_bits()[1],
               k_pool=sdev.bits(d["pool_before"][0]), v_pool=sdev.bits(d["pool_before"][1]))
    _device_pool_is_the_host_stream(batch, inp["v_pool"], gen.TENSOR_V_POOL, seed=4)
    ref, kp, vp = gc.run_oracle(batch, inp, n_threads=16)
    assert (sdev.bits(d["k_pool"]) == kp).all() and (sdev.bits(d["v_pool"]) == vp).all()
    gc.check_close(sdev.bits(d["out"]), ref, batch.name)


def _full_size_case(batch, n_decode_sample, seed, expect_mixed=None):
    """Full-size configuration in the launch sequence bench.py times (plan, then append + attention).  Checks
    (i) kv_append changed exactly its target slots: position-weighted checksums of BOTH whole pools before and after
        (every other byte untouched, at full size), and the placement of the sampled sequences bit-exactly;
    (ii) attention of >= 128 sampled decode sequences and of every 16th row (+ first/last) of every prefill chunk vs the
        oracle; (iii) every output finite (no NaN sentinel leaked anywhere)."""
    import gc as pygc
    pygc.collect()
    torch.cuda.empty_cache()
    dev = "cuda:0"
    w = gc._weights(dev)
    state = {}

    def before(d):
        tg = gc.append_targets(batch, dev)
        state["tg"] = tg
        for name in ("k", "v"):
            pool = d[f"{name}_pool"]
            state[name] = (gc.pool_checksum(pool, w), pool.view(-1)[tg.view(-1)].clone())
    d = gc.run_gpu(batch, None, pre_append=before, keep_pool_copy=False)
    for name in ("k", "v"):
        c0, old = state[name]
        want = gc.expected_checksum_after_append(c0, old, d[f"{name}_new"], state["tg"], w)
        assert gc.pool_checksum(d[f"{name}_pool"], w) == want, f"{batch.name}: {name.upper()} pool changed outside the append targets"
        assert (d[f"{name}_pool"].view(-1)[state["tg"].view(-1)].view(torch.int16) == d[f"{name}_new"].view(-1).view(torch.int16)).all()
    rng = np.random.default_rng(seed)
    nd = batch.num_decode_seqs
    seqs = list(rng.choice(nd, min(nd, n_decode_sample), replace=False)) if nd else []
    seqs += list(range(nd, batch.n_seq))
    gc.check_sampled_sequences(batch, d, seqs, prefill_row_stride=16, n_threads=16, what=batch.name)
    assert torch.isfinite(d["out"].float()).all()
    if expect_mixed is True:
        assert d["pa"].plan_info(6) > 0 and d["pa"].plan_info(1) > 0, "expected a mixed launch"
    return d


@pytest.mark.parametrize("r", [0.0, 0.1, 0.5, 1.0])
def test_config4_full_size_sampled(r):
    """C4 (Qwen3-8B shape, n_tok 8192): r = 0 (2048-token chunks over prior context, the tensor-bound point), 0.1 and 0.5
    (mixed launches) and 1.0 (8192 decode sequences, ~84 GB of KV) — PAPER.md:L62, L437, L508."""
    batch = workloads.config4(r, num_blocks=workloads.c4_pool_blocks())       # the pool bench.py's headline loop uses
    _full_size_case(batch, 128, 45 + int(10 * r), expect_mixed=(0 < r < 1) or None)


@pytest.mark.parametrize("variant", ["r1.0", "r0.2", "r0.059"])
def test_config5_full_size_sampled(variant):
    """C5 (Qwen3-30B-A3B shape, G = 8) on the 150 GB pool (3.75e10 elements per pool: 64-bit block addressing); R15's three
    variants.  Skips loudly when the device cannot hold the pool — it never shrinks it."""
    import gc as pygc
    pygc.collect()
    torch.cuda.empty_cache()
    nb = int(150e9 // (32 * 1024))
    free, _ = torch.cuda.mem_get_info()
    need = 2 * nb * 4 * 16 * 128 * 2 + 6e9
    if free < need:
        pytest.skip(f"C5 needs {need / 1e9:.0f} GB free for the 150 GB pool, device has {free / 1e9:.0f} GB")
    batch = workloads.config5(variant, num_blocks=nb)
    assert batch.num_blocks == int(150e9 // 32768)
    assert batch.block_tables.max() > (1 << 31) // (4 * 16 * 128), "block ids must reach past 2^31 elements"
    _full_size_case(batch, 128, 57, expect_mixed=(variant != "r1.0") or None)


def test_empty_and_degenerate_batches():
    W = workloads
    pa = binding.PagedAttention(8, 2, 128, 64, 8, 256, 8)
    dev = "cuda:0"
    z = torch.zeros(1, dtype=torch.int32, device=dev)
    # n_seq = 0: every call is a no-op returning OK
    pa.plan(np.zeros(1, np.int32), np.zeros(0, np.int32), 0, 0)
    pa.kv_append(None, None, None, None, z, z, z, 0, 0)
    q = torch.zeros((1, 8, 128), dtype=torch.bfloat16, device=dev)
    pa.batch_attention(q, q, q, z, z, z, 0.1, q)
    # q_len = 0 sequence inside the prefill range (R10)
    batch = W.make_batch("zero-q", W.TINY, 210, [1, 0, 5, 0], [20, 40, 3, 0], 1, num_blocks=64, min_table_width=8)
    inp = helpers.host_inputs(batch)
    d = gc.run_gpu(batch, inp, pa=pa)
    ref, _, _ = gc.run_oracle(batch, inp)
    gc.check_close(sdev.bits(d["out"]), ref, "zero-q")


def test_error_codes():
    pa = binding.PagedAttention(8, 2, 128, 64, 4, 64, 8)
    with pytest.raises(binding.PaError) as e:
        pa.plan(np.array([0, 2, 3], np.int32), np.array([5, 5], np.int32), 2, 1)        # decode q_len = 2
    assert e.value.code == binding.PA_ERR_INVALID
    with pytest.raises(binding.PaError) as e:
        pa.plan(np.array([0, 1, 0], np.int32), np.array([5, 5], np.int32), 2, 1)        # non-monotone
    assert e.value.code == binding.PA_ERR_INVALID
    with pytest.raises(binding.PaError) as e:
        pa.plan(np.array([0, 1], np.int32), np.array([8 * 16], np.int32), 1, 1)         # kv_len > table width
    assert e.value.code == binding.PA_ERR_INVALID
    with pytest.raises(binding.PaError) as e:
        pa.plan(np.arange(6, dtype=np.int32), np.zeros(5, np.int32), 5, 5)              # n_seq > max_seqs
    assert e.value.code == binding.PA_ERR_INVALID
    with pytest.raises(binding.PaError) as e:
        pa.timer_fit(0.5)
    assert e.value.code == binding.PA_ERR_TIMER
    with pytest.raises(binding.PaError) as e:
        binding.PagedAttention(8, 2, 64, 64, 4, 64, 8)
    assert e.value.code == binding.PA_ERR_UNSUPPORTED
    ws = pa.workspace
    pa.workspace = ws[: 1024]
    with pytest.raises(binding.PaError) as e:
        pa.plan(np.array([0, 1], np.int32), np.array([3], np.int32), 1, 1)
    assert e.value.code == binding.PA_ERR_WORKSPACE
    pa.workspace = ws


def test_timer_fit_matches_oracle_fit():
    pa = binding.PagedAttention(8, 2, 128, 64, 4, 64, 8)
    rng = np.random.default_rng(4)
    ns, Ts = [], []
    for n in (512, 1024, 2048, 4096):
        reps = 3e-6 + 1.1e-8 * n + rng.normal(0, 2e-7, 7)
        for t in reps:
            pa.timer_record(0.3, n, float(abs(t)))
        ns.append(n)
        Ts.append(float(np.median(np.abs(reps))))
    a, b, r2, npts = pa.timer_fit(0.3)
    oa, ob, or2 = oracle.fit(ns, Ts)
    assert npts == 4 and abs(a - oa) < 1e-15 and abs(b - ob) < 1e-18 and abs(r2 - or2) < 1e-12
    pa.timer_begin()
    sec = pa.timer_end(0.7, 128)
    assert 0 <= sec < 1.0


def test_timer_kappa_matches_oracle_quadratic():
    """N1 (App. A.3, Eq. 9-11): the library's quadratic fit of K(r) and kappa vs the oracle's."""
    pa = binding.PagedAttention(8, 2, 128, 64, 4, 64, 8)
    rng = np.random.default_rng(5)
    rs = [i / 10 for i in range(11)]
    Ks = []
    for r in rs:
        reps = 20e-6 + 30e-6 * r - 12e-6 * r * r + rng.normal(0, 2e-7, 9)
        for t in reps:
            pa.timer_record(r, 2048, float(t))
        pa.timer_record(r, 512, 1e-6)                      # other n_tok: must not enter the fit
        Ks.append(float(np.median(reps)))
    c, kappa, npts = pa.timer_kappa(2048)
    oc, okappa = oracle.quadratic_kappa(np.array(rs), np.array(Ks))
    assert npts == 11
    assert np.allclose(c, oc, rtol=1e-9, atol=1e-15) and abs(kappa - okappa) < 1e-9
    with pytest.raises(binding.PaError) as e:
        pa.timer_kappa(4096)                               # no samples at this n_tok
    assert e.value.code == binding.PA_ERR_TIMER
