#!/usr/bin/env python
"""bench.py — attention tokens/s and roofline fraction vs decode ratio r (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--extended]

Workload (N = 1): BASELINE.json configs[1] — Qwen3-4B-shaped attention layer (32 q heads / 8 KV heads,
head_dim 128, block 16), n_tok = 2048 per step, decode sequences with ctx 16, 512-token prompts,
decode ratio r swept 0.0 … 1.0 (Fig. 1 setup).  One *step* = kv_append +
batch_attention (SURVEY §8(a) a3–a7, planned by a1) over one synthetic batch; the K timed steps cycle
through the 11 r-batches (r_i = (i mod 11)/10), whose pools (11 × 1 GB) exceed L2, so every step
starts with cold inputs.  `value` = tokens / device time of those K steps (CUDA events, inputs resident
in HBM).  The same K steps are then repeated with an event pair around every attention launch: the live
per-launch durations behind `roofline` (kept out of the headline loop: an event between kv_append and
batch_attention would stop the attention CTAs from coming up under the append).
`e2e` = the same through the public binding from pinned HOST buffers (H2D of q/k_new/v_new
and the descriptors, pa_plan, kv_append, batch_attention, D2H of the output, per step).
Also reported: per-r table (tokens/s, achieved GB/s, roofline fraction, alpha/beta/R² of
T = alpha + beta·n_tok fitted through pa_timer_*), kappa and the mixed-vs-exclusive comparison
(SURVEY §8(f) N1/N3), the bandwidth-bound C3 (Gemma-3-1B decode) line, with --extended C4 (Qwen3-8B
mixed, n_tok 8192), N4 batches shaped by the paper's Table 9 length statistics and C5 (Qwen3-30B-A3B, 150 GB pool); the oracle timed on the host cores
(cpu_baseline).  Multi-GPU: the path has no exchange step ("replicas only"): each rank
runs the same workload on its GPU, value = Σ tokens / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "attention_tokens_per_s"
UNIT = "tokens/s"
R_GRID = [i / 10 for i in range(11)]
FIT_NTOK = [512, 1024, 2048, 4096]          # DESIGN R18
L2_FLUSH_BYTES = 512 << 20
# dram__bytes_read.sum + dram__bytes_write.sum per pa_attention_kernel launch, mean over the 11 r-batches of C2,
# from the ncu --set full capture summarised in profiles/ (None until that capture exists)
NCU_TRAFFIC_BYTES_PER_LAUNCH = 96011101.1
NCU_TRAFFIC_SOURCE = "profiles/r1g_c2_cycle.md (ncu --set full, 11 launches of one r-cycle)"


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


# ------------------------------------------------------------------------------------------------ ours
class Prepared:
    """A batch resident in HBM with its context and plan (inputs filled by the seeded device generator)."""

    def __init__(self, batch, dev, pools=None):
        import torch
        from paper_2606_00516_b200 import binding
        from paper_2606_00516_b200.synth import device as sdev
        self.batch = batch
        self.db = sdev.materialise(batch, dev, pools=pools)
        sh = batch.shape
        self.pa = binding.PagedAttention(sh.num_q_heads, sh.num_kv_heads, sh.head_dim, batch.num_blocks,
                                         max_seqs=batch.n_seq, max_tokens=batch.n_tok,
                                         max_blocks_per_seq=batch.max_blocks_per_seq, device=dev.index or 0)
        t0 = time.perf_counter()
        self.pa.plan(batch.cu_seqlens_q, batch.context_lens, batch.n_seq, batch.num_decode_seqs)
        torch.cuda.synchronize(dev)
        self.plan_seconds = time.perf_counter() - t0
        self.launches = 1 + self.pa.plan_info(5)

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
    """Cold-L2 statistics of one batch: T(append+attention), attention alone, roofline fraction."""
    b = prep.batch
    t_step = _timed_reps(prep.step, reps, warmup, flush)
    t_attn = _timed_reps(prep.attention, reps, warmup, flush)
    roof, bound = _roof_seconds(b, peaks)
    med_a = float(np.median(t_attn))
    return {"name": b.name, "r": round(b.r, 4), "n_tok": b.n_tok, "n_seq": b.n_seq,
            "T_step_us_median": float(np.median(t_step)) * 1e6, "T_step_us_min": float(np.min(t_step)) * 1e6,
            "T_attn_us_median": med_a * 1e6, "T_attn_us_min": float(np.min(t_attn)) * 1e6,
            "tokens_per_s": b.n_tok / float(np.median(t_step)),
            "alg_bytes": b.algorithmic_bytes(), "alg_flops": b.algorithmic_flops(),
            "achieved_GBps": b.algorithmic_bytes() / med_a / 1e9, "achieved_TFLOPs": b.algorithmic_flops() / med_a / 1e12,
            "roofline_us": roof * 1e6, "bound": bound, "roofline_frac": roof / med_a,
            "frac_of_nominal_8TBps": (b.algorithmic_bytes() / 8e12) / med_a if bound == "hbm" else None,
            "plan_us": prep.plan_seconds * 1e6, "launches_per_step": prep.launches,
            "decode_items": prep.pa.plan_info(0), "decode_bundles": prep.pa.plan_info(1),
            "split_items": prep.pa.plan_info(2), "prefill_tiles": prep.pa.plan_info(3)}


def _cpu_baseline(dev, seconds_budget=10.0):
    """The oracle, as it stands, on this host's cores: whole C2 steps (kv_append + attention of all 2048 rows),
    cycling r = 0.0, 0.1, ... like the timed region, until `seconds_budget` seconds of CPU work are done."""
    import torch
    import oracle
    from paper_2606_00516_b200.synth import device as sdev
    from paper_2606_00516_b200.synth import workloads
    cores = os.cpu_count() or 1
    hosts = []
    for r in R_GRID:
        batch = workloads.config2(r)
        db = sdev.materialise(batch, dev)
        torch.cuda.synchronize()
        sh = batch.shape
        osh = oracle.PagedShape(sh.num_q_heads, sh.num_kv_heads, sh.head_dim, sh.block_size)
        hosts.append((batch, osh, sdev.bits(db.q), sdev.bits(db.k_new), sdev.bits(db.v_new), sdev.bits(db.k_pool),
                      sdev.bits(db.v_pool)))
        del db
    torch.cuda.empty_cache()
    steps, tokens, dt = 0, 0, 0.0
    while dt < seconds_budget and steps < 2000:
        batch, osh, q, kn, vn, kp, vp = hosts[steps % len(hosts)]
        rows = np.arange(batch.n_tok, dtype=np.int64)
        t0 = time.perf_counter()
        oracle.kv_append(osh, kn, vn, kp, vp, batch.cu_seqlens_q, batch.context_lens, batch.block_tables)
        oracle.attention(osh, q, kp, vp, batch.cu_seqlens_q, batch.context_lens, batch.block_tables,
                         batch.softmax_scale, rows=rows, n_threads=cores)
        dt += time.perf_counter() - t0
        steps += 1
        tokens += batch.n_tok
    return {"value": tokens / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "seconds": dt, "steps": steps,
            "sample": f"{steps} whole C2 steps (kv_append + attention of all 2048 rows each, r cycled 0.0..1.0 as in the "
                      f"timed region; inputs resident in host memory), fp64 oracle, {cores} threads, {dt:.1f} s of CPU work"}


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
    flush = L2Flush(dev)

    sampler = ClockSampler(local)
    with sampler:
        # ---------------- headline: K steps cycling the 11 r-batches of C2 (each with its own pools)
        preps = [Prepared(workloads.config2(r), dev) for r in R_GRID]
        torch.cuda.synchronize()
        for i in range(W * len(preps)):
            preps[i % len(preps)].step()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        # The cycle of 11 steps (22 kernel launches through the C ABI) is captured once into a CUDA graph and replayed:
        # the library's calls only enqueue kernels on the caller's stream, so they capture as they are (the
        # programmatic dependency between kv_append and the attention launch included).  K mod 11 left-over steps
        # run eagerly.  Falls back to eager launches if capture is unavailable.
        n_cyc = len(preps)
        graph, launch_mode = None, "eager"
        try:
            graph = torch.cuda.CUDAGraph()
            # thread_local: the NCCL watchdog / NVML sampler threads neither break nor are broken by the capture
            with torch.cuda.graph(graph, capture_error_mode="thread_local"):
                for p in preps:
                    p.step()
            graph.replay()
            torch.cuda.synchronize()
            launch_mode = f"cuda graph of the {n_cyc}-step r-cycle, replayed"
        except Exception as exc:  # noqa: BLE001
            graph, launch_mode = None, f"eager (graph capture failed: {type(exc).__name__})"
            torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        launches = 0
        done = 0
        if graph is not None:
            for _ in range(K // n_cyc):
                graph.replay()
            done = (K // n_cyc) * n_cyc
            launches += sum(p.launches for p in preps) * (K // n_cyc)
        for i in range(done, K):
            p = preps[i % n_cyc]
            p.step()
            launches += p.launches
        e1.record()
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        sec = e0.elapsed_time(e1) * 1e-3
        tokens = sum(preps[i % len(preps)].batch.n_tok for i in range(K))
        # The same K steps once more, now with a CUDA event pair around every attention launch (same stream): the
        # dominant kernel's duration measured live for `roofline`.  Kept out of the headline loop because an event
        # between kv_append and batch_attention stops the attention CTAs from coming up under the append
        # (programmatic dependent launch), i.e. it would change the step being measured.
        kev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
        i0, i1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        i0.record()
        for i in range(K):
            p = preps[i % len(preps)]
            p.append()
            kev[i][0].record()
            p.attention()
            kev[i][1].record()
        i1.record()
        torch.cuda.synchronize()
        sec_instr = i0.elapsed_time(i1) * 1e-3
        attn_sec = [a.elapsed_time(b) * 1e-3 for a, b in kev]
        attn_bytes = [preps[i % len(preps)].batch.algorithmic_bytes() for i in range(K)]
        attn_roof = [_roof_seconds(preps[i % len(preps)].batch, peaks)[0] for i in range(K)]
        sec = max_over_ranks(sec, dev)

        # ---------------- e2e: host buffers in, host result out, through the public binding
        e2e = _e2e(preps, K, W, dev)
        e2e["seconds"] = max_over_ranks(e2e["seconds"], dev)
        e2e_value = job_throughput(tokens, e2e.pop("seconds"), world)

        sweep, fits, roofline, extra, cpu, kappa, ctx_sweep = [], [], None, {}, None, None, None
        if rank == 0:
            # ---------------- per-r table at the config's n_tok (cold L2 via flush), roofline fractions
            for p in preps:
                sweep.append(_point(p, peaks, args.reps, W, flush))
            # dominant kernel: pa_attention_kernel, the ONE launch of every batch_attention call (decode streams +
            # tcgen05 prefill units + merge).  achieved = algorithmic bytes per launch / average launch duration,
            # both averaged over the K timed steps; `traffic` = ncu dram bytes per launch, same average.
            mean_bytes, mean_sec = float(np.mean(attn_bytes)), float(np.mean(attn_sec))
            dec = sweep[-1]
            roofline = {"kernel": "pa::pa_attention_kernel<128, true> (single mixed launch per step; averaged over the "
                                  "K timed steps of the r cycle)",
                        "bound": "hbm", "achieved": mean_bytes / mean_sec / 1e9, "peak": peaks["hbm"], "unit": "GB/s",
                        "frac": mean_bytes / mean_sec / 1e9 / peaks["hbm"], "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH,
                        "traffic_source": NCU_TRAFFIC_SOURCE, "peak_source": peaks["src"] + " (burst copy figure)",
                        "alg_bytes_per_launch": mean_bytes, "launch_us": mean_sec * 1e6,
                        "kernel_share_of_step": sum(attn_sec) / sec_instr, "instrumented_ms_per_step": sec_instr / K * 1e3,
                        "roofline_time_frac": float(np.sum(attn_roof) / np.sum(attn_sec)),
                        "pure_decode_r1": {"achieved": dec["achieved_GBps"], "frac": dec["achieved_GBps"] / peaks["hbm"],
                                           "launch_us": dec["T_attn_us_median"], "note": "C2 r=1.0 alone, cold L2"}}
            # ---------------- N1 kappa / N3 exclusive-vs-mixed (post-processing of the sweep + two extra launches per r)
            kappa = _kappa_and_exclusive(preps, sweep, dev, W, max(3, args.reps // 2), flush)
            # ---------------- alpha/beta per r through the library's step timer (a8)
            if not args.no_fit:
                fits = _fit_sweep(dev, W, args.reps, flush)
                ctx_sweep = _ctx_sweep(dev, peaks, W, max(3, args.reps // 2), flush)
            # ---------------- bandwidth-bound decode (C3) and, with --extended, C4 / C5
            del preps
            torch.cuda.empty_cache()
            extra = _extra_configs(dev, peaks, args, W, flush)
            cpu = _cpu_baseline(dev)
    clocks = sampler.summary()

    if rank == 0:
        line = {"metric": METRIC, "value": job_throughput(tokens, sec, world), "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": sec / K * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "bf16", "data": "synthetic",
                "config": {"workload": "C2 Qwen3-4B-shaped attention layer (32/8/128, block 16), n_tok=2048/step, "
                                       "decode ctx 16, 512-token prompts, r cycled 0.0..1.0 over the K steps",
                           "n_tok": 2048, "r_grid": R_GRID, "l2": "inputs larger than L2: 11 batches x 0.5 GB pools "
                           "cycled; per-r table: L2 flushed between reps (512 MB write + 256 MB read)", "multi_gpu": "replicas only", "launch": launch_mode},
                "e2e": {"value": e2e_value, "unit": UNIT, **e2e},
                "gpu_launches": launches, "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu,
                "sweep": sweep, "fits": fits, "kappa": kappa, "ctx_sweep": ctx_sweep, "other_configs": extra, "peaks": peaks}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


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
        d, b = p.db, p.batch
        with torch.cuda.stream(s_in):
            if last_out[i % n] is not None:
                s_in.wait_event(last_out[i % n])        # inputs of this batch are being overwritten: its last step is done
            for k in ("q", "k_new", "v_new", "cu_seqlens_q", "context_lens", "block_tables"):
                getattr(d, k).copy_(h[k], non_blocking=True)
            e_in = torch.cuda.Event()
            e_in.record(s_in)
        with torch.cuda.stream(s_run):
            s_run.wait_event(e_in)
            p.pa.plan(b.cu_seqlens_q, b.context_lens, b.n_seq, b.num_decode_seqs)
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


def _kappa_and_exclusive(preps, sweep, dev, W, reps, flush):
    """N1: K(r) = c0 + c1 r + c2 r^2 and kappa = 2 c2/(c0+c1+c2) of OUR attention step time at n_tok = 2048
    (App. A.3, Eq. 9-11) through pa_timer_kappa; gap to the linear interpolation (Eq. 10).
    N3: the same tokens as two exclusive launches (decode-only step + prefill-only step) vs the one mixed step."""
    pa = preps[0].pa
    pa.timer_reset()
    for p, pt in zip(preps, sweep):
        pa.timer_record(round(p.batch.r, 3), p.batch.n_tok, pt["T_step_us_median"] * 1e-6)
    (c0, c1, c2), kappa, npts = pa.timer_kappa(preps[0].batch.n_tok)
    k0, k1 = sweep[0]["T_step_us_median"], sweep[-1]["T_step_us_median"]
    out = {"n_tok": preps[0].batch.n_tok, "c0_us": c0 * 1e6, "c1_us": c1 * 1e6, "c2_us": c2 * 1e6, "kappa": kappa,
           "n_points": npts, "note": "attention-only K(r) of one layer on B200 (paper: whole-model kappa -11.6 on "
           "RTX PRO 6000, -0.69 on H200, PAPER.md:L547 — context, not comparable)", "per_r": []}
    pools = None
    for p, pt in zip(preps, sweep):
        b = p.batch
        row = {"r": pt["r"], "K_mixed_us": pt["T_step_us_median"],
               "K_linear_interp_us": (1 - b.r) * k0 + b.r * k1,
               "gap_us": pt["T_step_us_median"] - ((1 - b.r) * k0 + b.r * k1)}
        dec, pre = _split_parts(b)
        t_excl = 0.0
        for part in (dec, pre):
            if part is None:
                continue
            pp = Prepared(part, dev, pools=(p.db.k_pool, p.db.v_pool))
            t_excl += float(np.median(_timed_reps(pp.step, reps, W, flush))) * 1e6
            del pp
        row["K_exclusive_two_steps_us"] = t_excl
        row["mixed_over_exclusive"] = pt["T_step_us_median"] / t_excl if t_excl > 0 else None
        out["per_r"].append(row)
    return out


def _ctx_sweep(dev, peaks, W, reps, flush):
    """N2 (Fig. 10 analogue): n_tok = 1024, decode ctx in {16, 64, 128, 256, 512},
    r = 0 ... 1.  The paper's observations to check: time grows monotonically with ctx at fixed r > 0, and the ctx
    curves meet at r = 0 ("no KV cache is accessed")."""
    from paper_2606_00516_b200.synth import workloads
    out = {"n_tok": 1024, "ctx": [16, 64, 128, 256, 512], "r": [0.0, 0.2, 0.4, 0.6, 0.8, 1.0], "T_step_us": {}}
    pools = None
    for ctx in out["ctx"]:
        row = []
        for r in out["r"]:
            b = workloads.config2(r, n_tok=1024, ctx=ctx, num_blocks=40960)
            p = Prepared(b, dev, pools=pools)
            pools = (p.db.k_pool, p.db.v_pool)
            row.append(float(np.median(_timed_reps(p.step, reps, W, flush))) * 1e6)
            del p
        out["T_step_us"][str(ctx)] = row
    cols = np.array([out["T_step_us"][str(c)] for c in out["ctx"]])
    out["monotone_in_ctx_for_r_ge_0.4"] = bool((np.diff(cols[:, 2:], axis=0) > -1.0).all())   # 1 us timing slack
    out["spread_at_r0_us"] = float(cols[:, 0].max() - cols[:, 0].min())
    return out


def _fit_sweep(dev, W, reps, flush):
    """T = alpha + beta*n_tok per r over n_tok in FIT_NTOK (medians), via pa_timer_* (PAPER.md:L21, L439)."""
    import torch
    from paper_2606_00516_b200.synth import workloads
    fits = []
    pools = None
    for r in R_GRID:
        timer_pa, T = None, {}
        for n in FIT_NTOK:
            p = Prepared(workloads.config2(r, n_tok=n), dev, pools=pools)
            pools = (p.db.k_pool, p.db.v_pool)
            timer_pa = timer_pa or p.pa
            for _ in range(W):
                flush.zero_()
                p.step()
            for _ in range(reps):
                flush.zero_()
                timer_pa.timer_begin()
                p.step()
                timer_pa.timer_end(r, n)
        a, b, r2, npts = timer_pa.timer_fit(r)
        fits.append({"r": r, "alpha_us": a * 1e6, "beta_ns_per_tok": b * 1e9, "r2": r2, "n_points": npts,
                     "n_tok_grid": FIT_NTOK})
    torch.cuda.synchronize()
    return fits


def _extra_configs(dev, peaks, args, W, flush):
    import torch
    from paper_2606_00516_b200.synth import workloads
    out = {}

    def run(key, batch, reps, use_flush=True):
        try:
            p = Prepared(batch, dev)
            out[key] = _point(p, peaks, reps, W, flush if use_flush else None)
            del p
        except Exception as e:  # noqa: BLE001 — report, do not hide (e.g. OOM on the 150 GB pool)
            out[key] = {"error": f"{type(e).__name__}: {e}"}
        torch.cuda.empty_cache()

    run("C3_gemma3_1b_decode", workloads.config3(), args.reps)
    if args.extended:
        for r in (0.0, 0.1, 0.5, 1.0):
            run(f"C4_qwen3_8b_r{r:.1f}", workloads.config4(r), 5, use_flush=False)
        # small batch, very long contexts: every (sequence, KV head) group is split over ~all decode streams
        run("long_context_4x131072", workloads.make_batch("long-4x131072", workloads.QWEN3_8B, 5, [1] * 4, [131072] * 4, 4),
            5, use_flush=False)
        for name in workloads.TABLE9:                       # N4: Table 9 length statistics
            for r in (0.5, 0.9):
                run(f"N4_{name}_r{r:.1f}", workloads.table9_batch(name, r), 5, use_flush=False)
        pool_blocks = int(150e9 // (32 * 1024))
        for v in ("r1.0", "r0.2", "r0.059"):
            run(f"C5_qwen3_30b_a3b_{v}", workloads.config5(v, num_blocks=pool_blocks), 3, use_flush=False)
    return out


# ------------------------------------------------------------------------------------------------ reference arm
def run_reference(args):
    """The fp64 CPU oracle as the reference arm (no other implementation exists: DESIGN.md §9)."""
    rank = int(os.environ.get("RANK", 0))
    if rank != 0:
        return
    import oracle
    from paper_2606_00516_b200.synth import gen, workloads
    K, W = args.steps, args.warmup
    cores = os.cpu_count() or 1
    # bounded sample per step: 64 rows (32 decode + 32 prefill) of a C2 batch, r cycled like our arm
    preps = []
    for r in R_GRID:
        b = workloads.config2(r)
        sh = b.shape
        osh = oracle.PagedShape(sh.num_q_heads, sh.num_kv_heads, sh.head_dim, sh.block_size)
        rng = np.random.default_rng(1000 + int(r * 10))
        nd = b.n_decode_tok
        rows = []
        if nd:
            rows += list(rng.choice(nd, min(32, nd), replace=False))
        if b.n_tok > nd:
            rows += list(nd + rng.choice(b.n_tok - nd, min(32, b.n_tok - nd), replace=False))
        rows = np.sort(np.array(rows, dtype=np.int64))
        # host inputs: q rows and the KV the sampled rows can see come from the seeded streams; the pool
        # is generated only for the blocks those sequences own
        q = b.q_bits()
        kn, vn = b.kv_new_bits()
        shape4 = (b.num_blocks, sh.num_kv_heads, sh.block_size, sh.head_dim)
        kp = np.zeros(shape4, dtype=np.uint16)
        vp = np.zeros(shape4, dtype=np.uint16)
        per_blk = sh.num_kv_heads * sh.block_size * sh.head_dim
        seqs = np.unique(np.searchsorted(b.cu_seqlens_q, rows, side="right") - 1)
        for s in seqs:
            for blk in b.block_tables[s][b.block_tables[s] >= 0]:
                kp[blk] = gen.bf16_normal(b.seed, gen.TENSOR_K_POOL, int(blk) * per_blk, per_blk).reshape(shape4[1:])
                vp[blk] = gen.bf16_normal(b.seed, gen.TENSOR_V_POOL, int(blk) * per_blk, per_blk).reshape(shape4[1:])
        oracle.kv_append(osh, kn, vn, kp, vp, b.cu_seqlens_q, b.context_lens, b.block_tables)
        preps.append((b, osh, q, kp, vp, rows))

    def step(i):
        b, osh, q, kp, vp, rows = preps[i % len(preps)]
        oracle.attention(osh, q, kp, vp, b.cu_seqlens_q, b.context_lens, b.block_tables, b.softmax_scale, rows=rows,
                         n_threads=cores)
        return len(rows)

    for i in range(W):
        step(i)
    t0 = time.perf_counter()
    tokens = sum(step(i) for i in range(K))
    dt = time.perf_counter() - t0
    val = tokens / dt
    sample = ("per step: attention of <=64 sampled token rows (32 decode + 32 prefill, seeded) of the C2 batch at "
              "r = (i mod 11)/10, all 32 q heads, fp64 oracle")
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": K,
                      "warmup": W, "ms_per_step": dt / K * 1e3, "higher_is_better": True, "scaling": "weak",
                      "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                      "config": {"workload": "C2 Qwen3-4B-shaped attention layer, n_tok=2048/step, r cycled 0.0..1.0 "
                                             "(bounded sample of rows per step)", "n_tok": 2048, "r_grid": R_GRID},
                      "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
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
        batch = workloads.config4(float(arg or 1.0))
    elif kind == "c5":
        batch = workloads.config5(arg or "r1.0", num_blocks=int(150e9 // (32 * 1024)))
    else:
        raise SystemExit("--only takes c2:<r> | c3 | c4:<r> | c5:<variant>")
    big = batch.algorithmic_bytes() > 4 * (126 << 20)          # inputs larger than L2: no flush needed
    pt = _point(Prepared(batch, dev), _peaks(), args.reps, max(1, args.warmup), None if big else L2Flush(dev))
    print(json.dumps({"only": args.only, **pt}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=110)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--reps", type=int, default=20, help="timed repetitions per point of the per-r tables (R19)")
    ap.add_argument("--extended", action="store_true", help="also run C4 (up to 92 GB pools) and C5 (150 GB pool)")
    ap.add_argument("--no-fit", action="store_true", help="skip the alpha/beta n_tok sweep")
    ap.add_argument("--only", default=None, help="run one configuration point only: c2:<r> | c3 | c4:<r> | c5:<variant>")
    args = ap.parse_args()
    if args.only:
        run_only(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
