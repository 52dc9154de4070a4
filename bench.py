#!/usr/bin/env python
"""bench.py — attention tokens/s and roofline fraction vs decode ratio r (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--quick]

Workload (N = 1): BASELINE.json configs[3] (C4) — the largest r-swept single-GPU configuration: Qwen3-8B-shaped
attention layer (32 q heads / 8 KV heads, head_dim 128, block 16), n_tok = 8192 per step, decode contexts
lognormal (median 2048, clipped to [256, 8192]), 2048-token prefill chunks over prior context U{0..4096}, decode
ratio r swept 0.0 … 1.0 (L35/L494 "Attention time grows with r").  One *step* = kv_append +
batch_attention (SURVEY §8(a) a3–a7, planned once per batch by a1) over one synthetic batch; the K timed steps cycle
through the 11 r-batches (r_i = (i mod 11)/10), which share one pool pair sized for r = 1 (2 x 42 GB): every step
streams far more than L2 holds, so every step starts cold.  `value` = tokens / device time of those K steps (CUDA
events on the launching stream, inputs resident in HBM); the same loop carries an event pair around every attention
launch — the live per-launch durations behind `roofline` (at these millisecond scales the events perturb nothing).
`e2e` = the same steps through the public binding from pinned HOST buffers (H2D of q/k_new/v_new and the descriptors,
pa_plan, kv_append, batch_attention, D2H of the output, per step).

Also in the same line: `peaks` (MEASURED_PEAKS.json + read-only streaming probes measured in this run), the C4 per-r
table with fractions against copy rate / read probe / 8 TB/s, alpha/beta/R² of T = alpha + beta·n_tok per r through
pa_timer_* for C4 (n_tok 2048/4096/8192) and C2 (512…4096), the C2 table (Qwen3-4B shape, ctx 16, the paper's Fig. 1/2
regime), kappa with a bootstrap interval (N1), the exclusive-vs-mixed comparison and Eq. 7 evaluated from our fits (N3),
the decode-context sweep (N2), Table-9-shaped batches (N4), C3 (Gemma-3-1B decode), a long-context point and C5
(Qwen3-30B-A3B shape on the 150 GB pool, three variants); the oracle timed on the host cores (cpu_baseline).
Multi-GPU: the path has no exchange step ("replicas only"): each rank runs the same workload on its own
GPU, value = Σ tokens / max-over-ranks time.  `--gpus N` without a torchrun environment launches the N ranks itself.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "attention_tokens_per_s"
UNIT = "tokens/s"
R_GRID = [i / 10 for i in range(11)]
FIT_NTOK_C2 = [512, 1024, 2048, 4096]       # DESIGN R18
FIT_NTOK_C4 = [2048, 4096, 8192]
L2_FLUSH_BYTES = 512 << 20
# dram__bytes_read.sum + dram__bytes_write.sum per pa_attention_kernel launch from an OFFLINE ncu capture of the 11
# launches of one C4 r-cycle (profiles/r2_c4_cycle_traffic.csv, made with the command named in the .md beside it);
# the live line labels it as such.  No capture file = null.
NCU_TRAFFIC = {"bytes_per_launch": None, "source": None}
_traffic_file = os.path.join(ROOT, "profiles", "r2_c4_cycle_traffic.csv")
if os.path.exists(_traffic_file):
    import csv
    with open(_traffic_file) as _f:
        _rows = list(csv.DictReader(_f))
    if _rows:
        NCU_TRAFFIC = {"bytes_per_launch": sum(float(x["dram_read_bytes"]) + float(x["dram_write_bytes"]) for x in _rows) / len(_rows),
                       "source": "profiles/r2_c4_cycle_traffic.csv (mean over the %d launches of one r-cycle)" % len(_rows)}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=float(d["hbm_gbs"]), tf_burst=float(d["bf16_tflops"]),
                    tf_sust=float(d.get("bf16_tflops_sustained", d["bf16_tflops"])), src="measured")
    return dict(hbm=6650.0, tf_burst=1590.0, tf_sust=1400.0, src="fallback")


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples SM clock and throttle reasons (NVML) during the measured region."""

    def __init__(self, index: int, period: float = 0.05):
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._th = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {getattr(nv, n): n for n in dir(nv) if n.startswith("nvmlClocksThrottleReason") and
                 isinstance(getattr(nv, n), int)}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                bits = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for b, n in names.items():
                    if b and (bits & b) and n not in ("nvmlClocksThrottleReasonNone", "nvmlClocksThrottleReasonAll"):
                        self.reasons.add(n.replace("nvmlClocksThrottleReason", ""))
            except Exception:
                pass
            self._stop.wait(self.period)

    def __enter__(self):
        if self.nv:
            self._th = threading.Thread(target=self._loop, daemon=True)
            self._th.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._th:
            self._th.join()

    def summary(self):
        busy = [s for s in self.samples if s > 0]
        ignore = {"GpuIdle", "ApplicationsClocksSetting"}
        return {"sm_mhz": float(np.median(busy)) if busy else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons - ignore), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------ ranks
def max_over_ranks(seconds: float, device=None) -> float:
    """Replicas only: the job's time is the slowest rank's device time.  all_reduce(MAX) on the
    process group's device (cuda for nccl, cpu for the gloo tests); identity without a process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(seconds)
    t = torch.tensor([seconds], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(tokens_per_rank: int, seconds: float, world: int) -> float:
    """Whole-job tokens/s of `world` identical replicas (weak scaling): Σ tokens ÷ max-over-ranks time."""
    return world * tokens_per_rank / seconds


def replica_launch_command(n: int, argv: list[str], port: int) -> list[str]:
    """`bench.py --gpus N` outside torchrun: the command that starts the N replica ranks (one per GPU)."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr",
            "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *argv]


# ------------------------------------------------------------------------------------------------ ours
class Prepared:
    """A batch resident in HBM with its context and plan (inputs filled by the seeded device generator)."""

    def __init__(self, batch, dev, pools=None, refill=True):
        import torch
        from paper_2606_00516_b200 import binding
        from paper_2606_00516_b200.synth import device as sdev
        self.batch = batch
        self.db = sdev.materialise(batch, dev, pools=pools, refill=refill)
        sh = batch.shape
        self.pa = binding.PagedAttention(sh.num_q_heads, sh.num_kv_heads, sh.head_dim, batch.num_blocks,
                                         max_seqs=batch.n_seq, max_tokens=batch.n_tok,
                                         max_blocks_per_seq=batch.max_blocks_per_seq, device=dev.index or 0)
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        self.plan()
        self.plan_call_seconds = time.perf_counter() - t0           # the binding's call: host lists + enqueue of the upload
        self.plan_first_seconds = self.pa.plan_info(9) * 1e-9        # inside pa_plan (C side), first call on a fresh context
        torch.cuda.synchronize(dev)
        ns = []
        for _ in range(5):                                           # steady state: the same batch planned again (as per step)
            self.plan()
            ns.append(self.pa.plan_info(9))
            torch.cuda.synchronize(dev)
        self.plan_host_seconds = float(np.median(ns)) * 1e-9
        self.launches = 1 + self.pa.plan_info(5)

    def plan(self):
        b = self.batch
        self.pa.plan(b.cu_seqlens_q, b.context_lens, b.n_seq, b.num_decode_seqs)

    def append(self):
        d, b = self.db, self.batch
        self.pa.kv_append(d.k_new, d.v_new, d.k_pool, d.v_pool, d.cu_seqlens_q, d.context_lens, d.block_tables,
                          b.n_seq, b.n_tok)

    def attention(self):
        d, b = self.db, self.batch
        self.pa.batch_attention(d.q, d.k_pool, d.v_pool, d.cu_seqlens_q, d.context_lens, d.block_tables,
                                b.softmax_scale, d.out)

    def step(self):
        self.append()
        self.attention()

    def check_finite(self):
        import torch
        assert bool(torch.isfinite(self.db.out.float()).all()), f"{self.batch.name}: non-finite attention output"


def _roof_seconds(batch, peaks):
    """max(bytes/BW, flops/F) with the measured peaks (SURVEY §8(d) "Which roofline")."""
    tb = batch.algorithmic_bytes() / (peaks["hbm"] * 1e9)
    tf = batch.algorithmic_flops() / (peaks["tf_sust"] * 1e12)
    return max(tb, tf), ("hbm" if tb >= tf else "tensor")


class L2Flush:
    """Cold AND clean L2 between repetitions: write a 512 MB buffer (evicts everything), then read a second 256 MB
    buffer, so that the ~126 MB of dirty lines the write leaves behind are written back before the timed kernel
    starts instead of competing with it for HBM."""

    def __init__(self, dev):
        import torch
        self.w = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
        self.r = torch.zeros(L2_FLUSH_BYTES // 8, dtype=torch.int32, device=dev)

    def zero_(self):
        self.w.zero_()
        self.r.sum()


def _read_probe(dev, peaks):
    """Read-only streaming ceiling of this GPU, measured in this run (SURVEY §7 "HBM target denominator"): 8 GiB read
    once per repetition by two plain probes (16-byte ld.global loads; 16 KB bulk copies into shared memory)."""
    import torch
    from paper_2606_00516_b200.synth import device as sdev
    nbytes = 8 << 30
    buf = torch.empty(nbytes, dtype=torch.uint8, device=dev)
    buf.zero_()
    sink = torch.zeros(1, dtype=torch.int64, device=dev)
    out = {}
    for mode, name in ((0, "ld_global_16B"), (1, "bulk_copy_16KB")):
        for _ in range(2):
            sdev.read_probe(buf, mode, sink)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(7)]
        torch.cuda.synchronize()
        for a, b in ev:
            a.record()
            sdev.read_probe(buf, mode, sink)
            b.record()
        torch.cuda.synchronize()
        ts = [a.elapsed_time(b) * 1e-3 for a, b in ev]
        out[name] = {"best_gbs": nbytes / min(ts) / 1e9, "median_gbs": nbytes / float(np.median(ts)) / 1e9}
    del buf
    torch.cuda.empty_cache()
    peaks["read_probe_gbs"] = max(v["best_gbs"] for v in out.values())
    peaks["read_probe"] = {"bytes": nbytes, **out, "note": "read-only pass over 8 GiB, best of 7, CUDA events; the larger of "
                           "the two probes is the read ceiling used for frac_of_read_probe"}


def _timed_reps(fn, reps, warmup, flush=None):
    """Per-rep CUDA-event times (seconds) on the current stream, optional L2 flush between reps."""
    import torch
    for _ in range(warmup):
        if flush is not None:
            flush.zero_()
        fn()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
    torch.cuda.synchronize()
    for a, b in ev:
        if flush is not None:
            flush.zero_()
        a.record()
        fn()
        b.record()
    torch.cuda.synchronize()
    return [a.elapsed_time(b) * 1e-3 for a, b in ev]


def _point(prep, peaks, reps, warmup, flush):
    """Cold-L2 statistics of one batch: T(append+attention), attention alone, roofline fractions."""
    b = prep.batch
    t_step = _timed_reps(prep.step, reps, warmup, flush)
    t_attn = _timed_reps(prep.attention, reps, warmup, flush)
    prep.check_finite()
    roof, bound = _roof_seconds(b, peaks)
    med_a = float(np.median(t_attn))
    gbs = b.algorithmic_bytes() / med_a / 1e9
    out = {"name": b.name, "r": round(b.r, 4), "n_tok": b.n_tok, "n_seq": b.n_seq,
           "T_step_us_median": float(np.median(t_step)) * 1e6, "T_step_us_min": float(np.min(t_step)) * 1e6,
           "T_attn_us_median": med_a * 1e6, "T_attn_us_min": float(np.min(t_attn)) * 1e6,
           "tokens_per_s": b.n_tok / float(np.median(t_step)),
           "alg_bytes": b.algorithmic_bytes(), "alg_flops": b.algorithmic_flops(),
           "achieved_GBps": gbs, "achieved_TFLOPs": b.algorithmic_flops() / med_a / 1e12,
           "roofline_us": roof * 1e6, "bound": bound, "roofline_frac": roof / med_a,
           "plan_host_us": prep.plan_host_seconds * 1e6, "plan_first_call_us": prep.plan_first_seconds * 1e6,
           "plan_call_us": prep.plan_call_seconds * 1e6,
           "launches_per_step": prep.launches,
           "decode_items": prep.pa.plan_info(0), "decode_bundles": prep.pa.plan_info(1),
           "split_items": prep.pa.plan_info(2), "prefill_tiles": prep.pa.plan_info(3),
           "prefill_ctas": prep.pa.plan_info(6)}
    if bound == "hbm":
        out["frac_of_copy_rate"] = gbs / peaks["hbm"]
        out["frac_of_read_probe"] = gbs / peaks["read_probe_gbs"] if peaks.get("read_probe_gbs") else None
        out["frac_of_nominal_8TBps"] = gbs / 8000.0
    else:
        out["frac_of_bf16_burst"] = out["achieved_TFLOPs"] / peaks["tf_burst"]
        out["frac_of_bf16_sustained"] = out["achieved_TFLOPs"] / peaks["tf_sust"]
    return out


# ------------------------------------------------------------------------------------------------ oracle legs
def _oracle_sample(batch, n_dec_rows, n_pre_rows, seed):
    """A bounded, seeded sample of a batch for the oracle: `n_dec_rows` decode sequences and `n_pre_rows` prefill rows,
    with a COMPACT host pool that holds only the blocks of the sampled sequences (block ids relabelled; values are the
    seeded streams of the physical blocks), so no host copy of a 40-150 GB pool is needed."""
    import oracle
    from paper_2606_00516_b200.synth import gen
    sh = batch.shape
    rng = np.random.default_rng(seed)
    nd = batch.num_decode_seqs
    dec = sorted(rng.choice(nd, min(n_dec_rows, nd), replace=False)) if nd else []
    pre_rows_all = np.arange(batch.n_decode_tok, batch.n_tok)
    pre_rows = np.sort(rng.choice(pre_rows_all, min(n_pre_rows, len(pre_rows_all)), replace=False)) if len(pre_rows_all) else []
    pre = sorted(set(int(np.searchsorted(batch.cu_seqlens_q, r, side="right") - 1) for r in pre_rows))
    order = list(dec) + pre
    b = sh.block_size
    q_lens, ctx = batch.q_lens[order], batch.context_lens[order]
    nblk = (ctx.astype(np.int64) + q_lens + b - 1) // b
    tables = np.full((len(order), max(1, int(nblk.max()) if len(order) else 1)), -1, dtype=np.int32)
    per_blk = sh.num_kv_heads * b * sh.head_dim
    shape4 = (int(nblk.sum()), sh.num_kv_heads, b, sh.head_dim)
    kp, vp = np.zeros(shape4, np.uint16), np.zeros(shape4, np.uint16)
    off = 0
    for i, s in enumerate(order):
        n = int(nblk[i])
        tables[i, :n] = np.arange(off, off + n)
        for k in range(n):
            blk = int(batch.block_tables[s, k])
            kp[off + k] = gen.bf16_normal(batch.seed, gen.TENSOR_K_POOL, blk * per_blk, per_blk).reshape(shape4[1:])
            vp[off + k] = gen.bf16_normal(batch.seed, gen.TENSOR_V_POOL, blk * per_blk, per_blk).reshape(shape4[1:])
        off += n
    cu = np.zeros(len(order) + 1, dtype=np.int32)
    np.cumsum(q_lens, out=cu[1:])
    src_rows = np.concatenate([np.arange(batch.cu_seqlens_q[s], batch.cu_seqlens_q[s + 1]) for s in order]) if order else np.zeros(0, np.int64)
    qd = sh.num_q_heads * sh.head_dim
    kd = sh.num_kv_heads * sh.head_dim
    q = np.stack([gen.bf16_normal(batch.seed, gen.TENSOR_Q, int(r) * qd, qd) for r in src_rows]).reshape(-1, sh.num_q_heads, sh.head_dim)
    kn = np.stack([gen.bf16_normal(batch.seed, gen.TENSOR_K_NEW, int(r) * kd, kd) for r in src_rows]).reshape(-1, sh.num_kv_heads, sh.head_dim)
    vn = np.stack([gen.bf16_normal(batch.seed, gen.TENSOR_V_NEW, int(r) * kd, kd) for r in src_rows]).reshape(-1, sh.num_kv_heads, sh.head_dim)
    # rows of the compact batch to evaluate: every sampled decode row, and the sampled prefill rows
    pos = {int(r): i for i, r in enumerate(src_rows)}
    rows = np.array(list(range(len(dec))) + [pos[int(r)] for r in pre_rows], dtype=np.int64)
    osh = oracle.PagedShape(sh.num_q_heads, sh.num_kv_heads, sh.head_dim, sh.block_size)
    return dict(osh=osh, q=q, k_new=kn, v_new=vn, k_pool=kp, v_pool=vp, cu=cu, ctx=ctx.astype(np.int32), tables=tables,
                rows=rows, scale=batch.softmax_scale, n_rows=len(rows))


def _oracle_step(s, cores):
    import oracle
    oracle.kv_append(s["osh"], s["k_new"], s["v_new"], s["k_pool"], s["v_pool"], s["cu"], s["ctx"], s["tables"])
    oracle.attention(s["osh"], s["q"], s["k_pool"], s["v_pool"], s["cu"], s["ctx"], s["tables"], s["scale"],
                     rows=s["rows"], n_threads=cores)
    return s["n_rows"]


ORACLE_SAMPLE = ("per step: kv_append of the sampled sequences + attention of <= 24 sampled decode rows and <= 8 sampled "
                 "prefill rows (seeded) of the C4 batch at r = (i mod 11)/10, all 32 q heads, fp64 oracle on a compact "
                 "host pool holding those sequences' blocks")


def _oracle_samples():
    from paper_2606_00516_b200.synth import workloads
    nb = workloads.c4_pool_blocks()
    return [_oracle_sample(workloads.config4(r, num_blocks=nb), 24, 8, 1000 + i) for i, r in enumerate(R_GRID)]


def _cpu_baseline(seconds_budget=12.0):
    """The oracle, as it stands, on this host's cores, on a bounded sample of the headline workload (C4 r-cycle)."""
    cores = os.cpu_count() or 1
    samples = _oracle_samples()
    steps, rows, dt = 0, 0, 0.0
    while dt < seconds_budget and steps < 2000:
        t0 = time.perf_counter()
        rows += _oracle_step(samples[steps % len(samples)], cores)
        dt += time.perf_counter() - t0
        steps += 1
    return {"value": rows / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt, "steps": steps,
            "sample": f"{steps} steps; {ORACLE_SAMPLE}; {cores} threads, {dt:.1f} s of CPU work; value = sampled token rows / s"}


# ------------------------------------------------------------------------------------------------ main arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_00516_b200.synth import workloads

    rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    local = int(os.environ.get("LOCAL_RANK", 0))
    dev = torch.device("cuda", local)
    torch.cuda.set_device(dev)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    peaks = _peaks()
    K, W = args.steps, max(3, args.warmup)
    reps = args.reps

    sampler = ClockSampler(local)
    with sampler:
        if rank == 0:
            _read_probe(dev, peaks)
        flush = L2Flush(dev)
        # ---------------- headline: K steps cycling the 11 r-batches of C4 over one shared pool pair
        nb = workloads.c4_pool_blocks()
        preps, pools = [], None
        for r in R_GRID:
            p = Prepared(workloads.config4(r, num_blocks=nb), dev, pools=pools, refill=pools is None)
            pools = (p.db.k_pool, p.db.v_pool)
            preps.append(p)
        n_cyc = len(preps)
        torch.cuda.synchronize()
        for i in range(max(W, n_cyc)):
            preps[i % n_cyc].step()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(K)]
        e_end = torch.cuda.Event(enable_timing=True)
        launches = 0
        for i in range(K):
            p = preps[i % n_cyc]
            ev[i][0].record()
            p.append()
            ev[i][1].record()
            p.attention()
            ev[i][2].record()
            launches += p.launches
        e_end.record()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        sec = ev[0][0].elapsed_time(e_end) * 1e-3
        for p in preps:
            p.check_finite()
        tokens = sum(preps[i % n_cyc].batch.n_tok for i in range(K))
        attn_sec = [e[1].elapsed_time(e[2]) * 1e-3 for e in ev]
        app_sec = [e[0].elapsed_time(e[1]) * 1e-3 for e in ev]
        sec = max_over_ranks(sec, dev)

        # ---------------- e2e: host buffers in, host result out, through the public binding
        e2e = _e2e(preps, K, W, dev)
        e2e["seconds"] = max_over_ranks(e2e["seconds"], dev)
        e2e_value = job_throughput(tokens, e2e.pop("seconds"), world)

        c4 = c2 = extra = cpu = roofline = eq7 = None
        if rank == 0:
            roofline = _roofline(preps, K, attn_sec, app_sec, sec, peaks)
            c4 = {"table": [_point(p, peaks, max(5, reps // 2), 2, flush if p.batch.algorithmic_bytes() < (1 << 30) else None)
                            for p in preps]}
            if not args.quick:
                c4["fits"] = _fit_sweep(dev, "c4", FIT_NTOK_C4, W, max(5, reps // 2), flush, pools, nb)
            del preps, pools, p
            torch.cuda.empty_cache()
            c2 = _c2_section(dev, peaks, args, W, reps, flush)
            extra = _other_configs(dev, peaks, args, W, flush)
            if not args.quick:
                eq7 = _eq7_report(c4.get("fits"), c2.get("fits"))
            cpu = _cpu_baseline()
    clocks = sampler.summary()

    if rank == 0:
        line = {"metric": METRIC, "value": job_throughput(tokens, sec, world), "unit": UNIT, "n_gpus": world, "steps": K,
                "warmup": max(W, n_cyc), "ms_per_step": sec / K * 1e3, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
                "config": {"workload": "C4 Qwen3-8B-shaped attention layer (32/8/128, block 16), n_tok=8192/step, decode ctx "
                                       "lognormal(median 2048) in [256, 8192], 2048-token prefill chunks over prior ctx "
                                       "U{0..4096}, r cycled 0.0..1.0 over the K steps (BASELINE configs[3])",
                           "n_tok": 8192, "r_grid": R_GRID, "pool_blocks": nb,
                           "l2": "inputs larger than L2: the 11 r-batches share one 2 x %.0f GB pool pair and each step streams "
                                 "0.2-84 GB; per-point tables of sub-GB batches flush L2 between reps (512 MB write + 256 MB "
                                 "read)" % (nb * 32768 / 1e9),
                           "multi_gpu": "replicas only", "launch": "eager; CUDA events around every launch of the timed loop"},
                "e2e": {"value": e2e_value, "unit": UNIT, **e2e},
                "gpu_launches": launches, "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu,
                "c4": c4, "c2": c2, "eq7": eq7, "other_configs": extra, "peaks": peaks}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def _roofline(preps, K, attn_sec, app_sec, sec, peaks):
    """Dominant kernel = pa_attention_kernel, the ONE launch of every batch_attention call (decode streams + tcgen05
    prefill units + merge).  achieved = algorithmic bytes per launch / average launch duration, both averaged over the K
    launches of the timed loop itself."""
    n = len(preps)
    b_bytes = [preps[i % n].batch.algorithmic_bytes() for i in range(K)]
    roofs = [_roof_seconds(preps[i % n].batch, peaks) for i in range(K)]
    mean_bytes, mean_sec = float(np.mean(b_bytes)), float(np.mean(attn_sec))
    gbs = mean_bytes / mean_sec / 1e9
    hb = [i for i in range(K) if roofs[i][1] == "hbm"]
    tb = [i for i in range(K) if roofs[i][1] == "tensor"]
    per_bound = {}
    if hb:
        g = sum(b_bytes[i] for i in hb) / sum(attn_sec[i] for i in hb) / 1e9
        per_bound["hbm"] = {"launches": len(hb), "achieved_GBps": g, "frac_of_copy_rate": g / peaks["hbm"],
                            "frac_of_read_probe": g / peaks["read_probe_gbs"], "frac_of_nominal_8TBps": g / 8000.0}
    if tb:
        f = sum(preps[i % n].batch.algorithmic_flops() for i in tb) / sum(attn_sec[i] for i in tb) / 1e12
        per_bound["tensor"] = {"launches": len(tb), "achieved_TFLOPs": f, "frac_of_bf16_burst": f / peaks["tf_burst"],
                               "frac_of_bf16_sustained": f / peaks["tf_sust"]}
    return {"kernel": "pa::pa_attention_kernel<128, true> (single mixed launch per step; all K launches of the timed loop)",
            "bound": "hbm", "achieved": gbs, "peak": peaks["hbm"], "unit": "GB/s", "frac": gbs / peaks["hbm"],
            "traffic": NCU_TRAFFIC.get("bytes_per_launch"),
            "traffic_source": ("OFFLINE ncu capture, not measured in this run: " + str(NCU_TRAFFIC.get("source")))
            if NCU_TRAFFIC.get("bytes_per_launch") else None,
            "peak_source": peaks["src"] + " (MEASURED_PEAKS.json hbm_gbs: device copy, read + write bytes)",
            "frac_of_read_probe": gbs / peaks["read_probe_gbs"], "frac_of_nominal_8TBps": gbs / 8000.0,
            "alg_bytes_per_launch": mean_bytes, "launch_us": mean_sec * 1e6,
            "kernel_share_of_step": float(np.sum(attn_sec)) / sec, "kv_append_share_of_step": float(np.sum(app_sec)) / sec,
            "roofline_time_frac": float(sum(r[0] for r in roofs) / np.sum(attn_sec)),
            "per_r_launch_us": [float(np.mean([attn_sec[i] for i in range(K) if i % n == j])) * 1e6 for j in range(n)],
            "per_r_roofline_frac": [float(np.sum([roofs[i][0] for i in range(K) if i % n == j]) /
                                          np.sum([attn_sec[i] for i in range(K) if i % n == j])) for j in range(n)],
            "bound_note": "10 of the 11 r-batches are HBM-bound, r = 0 is tensor-bound (per_bound)", "per_bound": per_bound}


def _e2e(preps, K, W, dev):
    """Step from HOST buffers: H2D(q, k_new, v_new, descriptors) + plan + append + attention + D2H(out)."""
    import torch
    host = []
    for p in preps:
        d = p.db
        h = {k: getattr(d, k).cpu().pin_memory() for k in ("q", "k_new", "v_new", "cu_seqlens_q", "context_lens",
                                                            "block_tables")}
        h["out"] = torch.empty_like(d.out, device="cpu").pin_memory()
        host.append(h)

    # Three streams, as a serving engine would run it: the H2D of step i+1 and the D2H of step i-1 overlap the
    # kernels of step i (every r-batch has its own device buffers, so the only hazards are a batch's own previous use).
    n = len(preps)
    s_in, s_run, s_out = torch.cuda.Stream(dev), torch.cuda.Stream(dev), torch.cuda.Stream(dev)
    last_out = [None] * n          # event: the previous D2H of this batch's output buffer has finished

    def one(i):
        p, h = preps[i % n], host[i % n]
        d = p.db
        with torch.cuda.stream(s_in):
            if last_out[i % n] is not None:
                s_in.wait_event(last_out[i % n])        # inputs of this batch are being overwritten: its last step is done
            for k in ("q", "k_new", "v_new", "cu_seqlens_q", "context_lens", "block_tables"):
                getattr(d, k).copy_(h[k], non_blocking=True)
            e_in = torch.cuda.Event()
            e_in.record(s_in)
        with torch.cuda.stream(s_run):
            s_run.wait_event(e_in)
            p.plan()
            p.step()
            e_run = torch.cuda.Event()
            e_run.record(s_run)
        with torch.cuda.stream(s_out):
            s_out.wait_event(e_run)
            h["out"].copy_(d.out, non_blocking=True)
            e_out = torch.cuda.Event()
            e_out.record(s_out)
        last_out[i % n] = e_out

    torch.cuda.synchronize()
    for i in range(W):
        one(i)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for i in range(K):
        one(i)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    for h in host:
        assert bool(torch.isfinite(h["out"].float()).all()), "e2e: non-finite output on the host"
    bi = np.mean([sum(h[k].numel() * h[k].element_size() for k in h if k != "out") for h in host])
    bo = np.mean([h["out"].numel() * h["out"].element_size() for h in host])
    return {"seconds": dt, "h2d_bytes_per_step": int(bi), "d2h_bytes_per_step": int(bo),
            "includes": "per step: H2D inputs+descriptors (pinned), pa_plan, kv_append, batch_attention, D2H output; copies on "
                        "their own streams overlap the neighbouring steps' kernels; wall clock over the K steps"}


def _split_parts(batch):
    """The decode-only and the prefill-only half of a mixed batch (same sequences, same seed) — SURVEY §8(f) N3."""
    from paper_2606_00516_b200.synth import workloads
    nd = batch.num_decode_seqs
    q, c = batch.q_lens, batch.context_lens
    dec = workloads.make_batch(batch.name + "-dec", batch.shape, batch.seed, q[:nd], c[:nd], nd,
                               num_blocks=batch.num_blocks) if nd > 0 else None
    pre = workloads.make_batch(batch.name + "-pre", batch.shape, batch.seed, q[nd:], c[nd:], 0,
                               num_blocks=batch.num_blocks) if nd < batch.n_seq else None
    return dec, pre


class GraphTimer:
    """Low-noise time of one microsecond-scale step: the batch is replicated on `copies` independent buffer sets (pools,
    q, k_new, v_new, out: more than L2 in total, so every step starts cold), one CUDA graph holds `copies` x `rounds`
    steps back to back, and each sample is one replay divided by the steps in it."""

    def __init__(self, batch, dev, copies=4, rounds=3):
        import torch
        self.preps = [Prepared(batch, dev) for _ in range(copies)]
        self.steps = copies * rounds
        torch.cuda.synchronize()
        for p in self.preps:
            p.step()
        torch.cuda.synchronize()
        self.graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(self.graph, capture_error_mode="thread_local"):
            for _ in range(rounds):
                for p in self.preps:
                    p.step()
        self.graph.replay()
        torch.cuda.synchronize()

    def samples(self, n):
        import torch
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
        for a, b in ev:
            a.record()
            self.graph.replay()
            b.record()
        torch.cuda.synchronize()
        self.preps[0].check_finite()
        return [a.elapsed_time(b) * 1e-3 / self.steps for a, b in ev]


def _c2_section(dev, peaks, args, W, reps, flush):
    """C2 (BASELINE configs[1]: Qwen3-4B shape, n_tok 2048, decode ctx 16, 512-token prompts — the paper's Fig. 1/2
    regime): per-r table, graph-replayed K(r), kappa with a bootstrap interval (N1), exclusive-vs-mixed (N3), fits, and
    the decode-context sweep (N2)."""
    import torch
    from paper_2606_00516_b200.synth import workloads
    preps = [Prepared(workloads.config2(r), dev) for r in R_GRID]
    out = {"table": [_point(p, peaks, reps, W, flush) for p in preps]}
    # ---- the cycle of 11 steps replayed from one CUDA graph (round 1's headline; launch-bound regime)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, capture_error_mode="thread_local"):
        for p in preps:
            p.step()
    g.replay()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(20):
        g.replay()
    e1.record()
    torch.cuda.synchronize()
    cyc = e0.elapsed_time(e1) * 1e-3 / 20
    out["graph_cycle"] = {"us_per_step": cyc / len(preps) * 1e6, "tokens_per_s": 2048 * len(preps) / cyc,
                          "note": "11-step r-cycle (22 launches) captured once and replayed 20 times; each batch has its own pools"}
    del g
    if args.quick:
        return out
    # ---- N1: K(r) from graph replays (>= 50 samples per r), kappa through pa_timer_kappa, bootstrap interval
    n_samp = 60
    Ks = []
    for p in preps:
        gt = GraphTimer(p.batch, dev)
        Ks.append(np.array(gt.samples(n_samp)))
        del gt
        torch.cuda.empty_cache()
    pa = preps[0].pa

    def kappa_of(vals):
        pa.timer_reset()
        for p, v in zip(preps, vals):
            pa.timer_record(round(p.batch.r, 3), p.batch.n_tok, float(v))
        return pa.timer_kappa(preps[0].batch.n_tok)
    (c0, c1, c2), kappa, npts = kappa_of([np.median(k) for k in Ks])
    rng = np.random.default_rng(11)
    boot = [kappa_of([np.median(rng.choice(k, len(k))) for k in Ks])[1] for _ in range(300)]
    k0, k1 = float(np.median(Ks[0])), float(np.median(Ks[-1]))
    kap = {"n_tok": 2048, "c0_us": c0 * 1e6, "c1_us": c1 * 1e6, "c2_us": c2 * 1e6, "kappa": kappa, "n_points": npts,
           "kappa_bootstrap_95": [float(np.percentile(boot, 2.5)), float(np.percentile(boot, 97.5))],
           "samples_per_r": n_samp, "method": "each r: 4 buffer sets x 3 rounds of (kv_append + attention) in one CUDA graph, "
           "60 replays, K(r) = median replay time / 12; kappa by pa_timer_kappa; interval from 300 bootstrap resamples",
           "note": "attention-only K(r) of one layer on B200 (paper: whole-model kappa -11.6 on RTX PRO 6000, -0.69 on H200, "
                   "PAPER.md:L547 — context, not comparable)", "per_r": []}
    # ---- N3 (first half): the same tokens as two exclusive launches vs the one mixed launch
    for p, ks in zip(preps, Ks):
        b = p.batch
        km = float(np.median(ks))
        row = {"r": round(b.r, 4), "K_mixed_us": km * 1e6, "K_linear_interp_us": ((1 - b.r) * k0 + b.r * k1) * 1e6,
               "gap_us": (km - ((1 - b.r) * k0 + b.r * k1)) * 1e6}
        t_excl = 0.0
        for part in _split_parts(b):
            if part is None:
                continue
            gt = GraphTimer(part, dev)
            t_excl += float(np.median(gt.samples(20)))
            del gt
            torch.cuda.empty_cache()
        row["K_exclusive_two_steps_us"] = t_excl * 1e6
        row["mixed_over_exclusive"] = km / t_excl if t_excl > 0 else None
        kap["per_r"].append(row)
    out["kappa"] = kap
    del preps
    torch.cuda.empty_cache()
    out["fits"] = _fit_sweep(dev, "c2", FIT_NTOK_C2, W, reps, flush, None, None)
    out["ctx_sweep"] = _ctx_sweep(dev)
    return out


def _ctx_sweep(dev):
    """N2 (Fig. 10 analogue): n_tok = 1024, decode ctx in {16, 64, 128, 256, 512},
    r = 0 ... 1, graph-replayed step times.  The paper's observations to check: time grows monotonically with ctx at
    every fixed r > 0, and the ctx curves meet at r = 0 ("no KV cache is accessed")."""
    import torch
    from paper_2606_00516_b200.synth import workloads
    out = {"n_tok": 1024, "ctx": [16, 64, 128, 256, 512], "r": [0.0, 0.2, 0.4, 0.6, 0.8, 1.0], "T_step_us": {}}
    for ctx in out["ctx"]:
        row = []
        for r in out["r"]:
            gt = GraphTimer(workloads.config2(r, n_tok=1024, ctx=ctx, num_blocks=40960), dev, copies=2, rounds=3)
            row.append(float(np.median(gt.samples(20))) * 1e6)
            del gt
            torch.cuda.empty_cache()
        out["T_step_us"][str(ctx)] = row
    cols = np.array([out["T_step_us"][str(c)] for c in out["ctx"]])
    d = np.diff(cols[:, 1:], axis=0)
    out["monotone_in_ctx_for_all_r_gt_0"] = bool((d > 0).all())
    out["monotone_violations"] = [{"r": out["r"][1 + int(j)], "ctx_from": out["ctx"][int(i)], "ctx_to": out["ctx"][int(i) + 1],
                                   "delta_us": float(d[i, j])} for i, j in zip(*np.where(d <= 0))]
    out["grows_with_r_at_ctx16"] = bool((np.diff(cols[0, 1:]) > 0).all())
    out["spread_at_r0_us"] = float(cols[:, 0].max() - cols[:, 0].min())
    return out


def _fit_sweep(dev, which, grid, W, reps, flush, pools, nb):
    """T = alpha + beta*n_tok per r over `grid` (medians), via pa_timer_* (PAPER.md:L21, L439); plan time beside alpha."""
    import torch
    from paper_2606_00516_b200.synth import workloads
    fits = []
    for r in R_GRID:
        timer_pa, plan_us = None, []
        for n in grid:
            batch = workloads.config2(r, n_tok=n) if which == "c2" else workloads.config4(r, n_tok=n, num_blocks=nb)
            p = Prepared(batch, dev, pools=pools, refill=pools is None or which == "c2")
            if which == "c2":
                pools = (p.db.k_pool, p.db.v_pool) if pools is None or p.db.k_pool.shape == pools[0].shape else None
            timer_pa = timer_pa or p.pa
            plan_us.append(p.plan_host_seconds * 1e6)
            fl = flush if batch.algorithmic_bytes() < (1 << 30) else None
            for _ in range(2):
                if fl:
                    fl.zero_()
                p.step()
            for _ in range(reps):
                if fl:
                    fl.zero_()
                timer_pa.timer_begin()
                p.step()
                timer_pa.timer_end(r, n)
            p.check_finite()
            del p
        a, b, r2, npts = timer_pa.timer_fit(r)
        fits.append({"r": r, "alpha_us": a * 1e6, "beta_ns_per_tok": b * 1e9, "r2": r2, "n_points": npts,
                     "n_tok_grid": grid, "plan_host_us": plan_us})
        if which == "c2":
            pools = None
    torch.cuda.synchronize()
    return fits


def _eq7_report(c4_fits, c2_fits):
    """N3 (second half; Prop. 3.4, Eq. 7; L117 beta_EB^w; L550-554 App. A.4): our fitted lines fed into
    the crossover condition.  alpha_p, beta_p = the r = 0 (prefill-only) fit; alpha_d, beta_d = the r = 1 (decode-only) fit;
    alpha_MB, beta_MB^e(r) = the mixed fit at r; beta_MB^e(r) additionally as the quadratic c0 + c1 r + c2 r^2 through the
    11 fitted betas.  (mu_L, mu_O) from Table 9; r_hat = mu_O / (mu_L + mu_O); theta0, zeta from Eq. 3 with p0 = 1/mu_O;
    k0* = floor(theta0 N).  Attention-only coefficients of ONE layer (DESIGN R17): a reporting exercise, not the paper's
    whole-model numbers.  All arithmetic by the library (pa_crossover_*, pa_timer_kappa's quadratic fit)."""
    from paper_2606_00516_b200 import binding
    from paper_2606_00516_b200.synth import workloads
    lib = binding.PagedAttention.__new__(binding.PagedAttention)
    lib.lib = binding.load_library()
    out = {}
    for name, fits in (("c4", c4_fits), ("c2", c2_fits)):
        if not fits:
            continue
        f = {round(x["r"], 1): x for x in fits}
        ap, bp = f[0.0]["alpha_us"] * 1e-6, f[0.0]["beta_ns_per_tok"] * 1e-9
        ad, bd = f[1.0]["alpha_us"] * 1e-6, f[1.0]["beta_ns_per_tok"] * 1e-9
        rs = np.array(sorted(f))
        betas = np.array([f[r]["beta_ns_per_tok"] * 1e-9 for r in rs])
        A = np.stack([np.ones_like(rs), rs, rs * rs], axis=1)
        c = np.linalg.lstsq(A, betas, rcond=None)[0]
        rows = []
        for wl, st in workloads.TABLE9.items():
            muL, muO = float(st["in_mean"]), float(st["out_mean"])
            r_hat = muO / (muL + muO)
            rk = min(f, key=lambda x: abs(x - r_hat))
            amb, bmb = f[rk]["alpha_us"] * 1e-6, f[rk]["beta_ns_per_tok"] * 1e-9
            if ap <= 0 or ad <= 0:
                rows.append({"workload": wl, "skipped": "non-positive fitted alpha_p or alpha_d"})
                continue
            theta0, zeta = lib.crossover_theta0((1.0 / muO) * ap / ad)
            for N in (256, 1024):
                k0 = max(1.0, float(np.floor(theta0 * N)))
                o = lib.crossover_eq7(ap, bp, ad, bd, amb, bmb, muL, muO, zeta, k0, N)
                rows.append({"workload": wl, "mu_L": muL, "mu_O": muO, "r_hat": r_hat, "r_fit_used": rk, "N": N,
                             "theta0": theta0, "zeta": zeta, "k0": k0, "beta_MB_e_s_per_tok": bmb,
                             "beta_MB_e_quadratic_s_per_tok": float(c[0] + c[1] * r_hat + c[2] * r_hat ** 2),
                             "beta_EB_w_s_per_tok": o["beta_eb_w"], "lhs": o["lhs"], "rhs": o["rhs"],
                             "mixed_wins": bool(o["lhs"] < o["rhs"]), "tp_eb": o["tp_eb"], "tp_mb": o["tp_mb"]})
        out[name] = {"alpha_p_s": ap, "beta_p_s_per_tok": bp, "alpha_d_s": ad, "beta_d_s_per_tok": bd,
                     "beta_MB_e_quadratic_c0_c1_c2_s_per_tok": [float(x) for x in c], "rows": rows}
    return out


def _other_configs(dev, peaks, args, W, flush):
    import torch
    from paper_2606_00516_b200.synth import workloads
    out = {}

    def run(key, make, reps, use_flush=True):
        try:
            p = Prepared(make(), dev)
            out[key] = _point(p, peaks, reps, 2, flush if use_flush else None)
            del p
        except Exception as e:  # noqa: BLE001 — report, do not hide (e.g. OOM on the 150 GB pool)
            out[key] = {"error": f"{type(e).__name__}: {e}"}
        torch.cuda.empty_cache()

    run("C3_gemma3_1b_decode", workloads.config3, args.reps)
    if not args.quick:
        # small batch, very long contexts: every (sequence, KV head) group is split over ~all decode streams
        run("long_context_4x131072", lambda: workloads.make_batch("long-4x131072", workloads.QWEN3_8B, 5, [1] * 4, [131072] * 4, 4),
            7, use_flush=False)
        for name in workloads.TABLE9:                       # N4: Table 9 length statistics
            for r in (0.5, 0.9):
                run(f"N4_{name}_r{r:.1f}", lambda name=name, r=r: workloads.table9_batch(name, r), 7)
    pool_blocks = int(150e9 // (32 * 1024))
    for v in ("r1.0", "r0.2", "r0.059"):
        run(f"C5_qwen3_30b_a3b_{v}", lambda v=v: workloads.config5(v, num_blocks=pool_blocks), 5, use_flush=False)
    return out


# ------------------------------------------------------------------------------------------------ reference arm
def run_reference(args):
    """The fp64 CPU oracle as the reference arm (no other implementation exists: DESIGN.md §9): each step a bounded
    sample of the headline workload's batch at r = (i mod 11)/10."""
    rank = int(os.environ.get("RANK", 0))
    if rank != 0:
        return
    K, W = args.steps, args.warmup
    cores = os.cpu_count() or 1
    samples = _oracle_samples()
    for i in range(W):
        _oracle_step(samples[i % len(samples)], cores)
    t0 = time.perf_counter()
    rows = sum(_oracle_step(samples[i % len(samples)], cores) for i in range(K))
    dt = time.perf_counter() - t0
    val = rows / dt
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": K,
                      "warmup": W, "ms_per_step": dt / K * 1e3, "higher_is_better": True, "scaling": "weak",
                      "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": "C4 Qwen3-8B-shaped attention layer, n_tok=8192/step, r cycled 0.0..1.0 "
                                             "(bounded sample of rows per step)", "n_tok": 8192, "r_grid": R_GRID},
                      "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": ORACLE_SAMPLE},
                      "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def run_only(args):
    """One configuration point by itself (used for the ncu captures in profiles/): c2:<r> | c3 | c4:<r> | c5:<variant>."""
    import torch
    from paper_2606_00516_b200.synth import workloads
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    kind, _, arg = args.only.partition(":")
    if kind == "c2":
        batch = workloads.config2(float(arg or 1.0))
    elif kind == "c3":
        batch = workloads.config3()
    elif kind == "c4":
        batch = workloads.config4(float(arg or 1.0), num_blocks=workloads.c4_pool_blocks())
    elif kind == "c5":
        batch = workloads.config5(arg or "r1.0", num_blocks=int(150e9 // (32 * 1024)))
    else:
        raise SystemExit("--only takes c2:<r> | c3 | c4:<r> | c5:<variant>")
    peaks = _peaks()
    peaks["read_probe_gbs"] = None
    big = batch.algorithmic_bytes() > (1 << 30)          # inputs larger than L2: no flush needed
    pt = _point(Prepared(batch, dev), peaks, args.reps, max(1, args.warmup), None if big else L2Flush(dev))
    print(json.dumps({"only": args.only, **pt}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=110)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--reps", type=int, default=20, help="timed repetitions per point of the per-r tables (R19)")
    ap.add_argument("--quick", action="store_true", help="headline, tables, C3 and C5 only (no fits, kappa, sweeps, N4)")
    ap.add_argument("--only", default=None, help="run one configuration point only: c2:<r> | c3 | c4:<r> | c5:<variant>")
    args = ap.parse_args()
    if args.only:
        run_only(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # replicas only: start one rank per GPU ourselves (the driver normally does this through torchrun)
        import socket
        with socket.socket() as s:
            s.bind(("127.0.0.1", 0))
            port = s.getsockname()[1]
        raise SystemExit(subprocess.call(replica_launch_command(args.gpus, sys.argv[1:], port)))
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
