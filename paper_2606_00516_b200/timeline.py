"""Developer tool: clock stamps of one CTA of the attention launch (the PA_TL / PA_TL_CTA macros of csrc/pa_common.cuh).

    python -m paper_2606_00516_b200.timeline --case c2:1.0            # 17-key decode items (paper Fig. 1/2 regime)
    python -m paper_2606_00516_b200.timeline --case c3 --bundles 2    # C3 with two queue-drawn bundles per stream

Builds an INSTRUMENTED copy of the library (`libpa_timeline_<cta>.so`, -DPA_TIMELINE=<cta>; the product library carries
no stamps), runs a few warm-up steps and one stamped step (kv_append + attention after an L2 flush) and prints
  - for stream 0 of the chosen CTA (decode role): per item, the consumer's and the producer lane's hand-off times in
    SM cycles since kernel entry, and the median duration of each phase of an item;
  - for every CTA: when it consumed its last K/V block and when it left the kernel (%globaltimer, ns).
The stamps live in the (otherwise idle) redo region of the workspace.  The numbers quoted in DESIGN.md §9b and
profiles/r2i_timelines.md come from this tool.  Not part of the product path; needs a B200.
"""
from __future__ import annotations

import argparse
import glob
import os
import subprocess

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)


def build(cta: int) -> str:
    lib = os.path.join(HERE, f"libpa_timeline_{cta}.so")
    srcs = sorted(glob.glob(os.path.join(HERE, "csrc", "*.cu")))
    deps = srcs + glob.glob(os.path.join(HERE, "csrc", "*.cuh")) + glob.glob(os.path.join(HERE, "csrc", "*.h"))
    if not os.path.exists(lib) or any(os.path.getmtime(s) > os.path.getmtime(lib) for s in deps):
        cmd = [os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc"), "-gencode", "arch=compute_100a,code=sm_100a", "-O3",
               "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-shared", "--expt-relaxed-constexpr",
               f"-DPA_TIMELINE={cta}", "-I", os.path.join(ROOT, "include"), "-o", lib, *srcs]
        print("+", " ".join(cmd), flush=True)
        subprocess.check_call(cmd)
    return lib


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--case", default="c2:1.0", help="c2:<r> | c3 | c4:<r>")
    ap.add_argument("--cta", type=int, default=100, help="CTA whose hand-offs are stamped (a decode CTA for --case c2:1.0 / c3)")
    ap.add_argument("--bundles", type=int, default=0, help="tune_bundles_per_stream (0 = planner's choice)")
    ap.add_argument("--build-only", action="store_true")
    args = ap.parse_args()
    lib = build(args.cta)
    if args.build_only:
        return
    import torch
    from paper_2606_00516_b200 import binding
    binding.LIB_PATH = lib
    from paper_2606_00516_b200.synth import device as sdev
    from paper_2606_00516_b200.synth import workloads as W

    kind, _, arg = args.case.partition(":")
    batch = {"c2": lambda: W.config2(float(arg or 1.0)), "c3": W.config3,
             "c4": lambda: W.config4(float(arg or 1.0))}[kind]()
    sh = batch.shape
    db = sdev.materialise(batch)
    stamp_bytes = 16 * 400 * 32 + 148 * 32
    # the stamps must fit the redo region (max_tokens * Hq * 8 bytes), or they would land in the split-KV partials
    max_tokens = max(batch.n_tok, -(-stamp_bytes // (sh.num_q_heads * 8)))
    pa = binding.PagedAttention(sh.num_q_heads, sh.num_kv_heads, sh.head_dim, batch.num_blocks, max_seqs=batch.n_seq,
                                max_tokens=max_tokens, max_blocks_per_seq=batch.max_blocks_per_seq,
                                tune_bundles_per_stream=args.bundles)
    pa.plan(batch.cu_seqlens_q, batch.context_lens, batch.n_seq, batch.num_decode_seqs)
    flush_w = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
    flush_r = torch.zeros(64 << 20, dtype=torch.int32, device="cuda")

    def step():
        flush_w.zero_()
        flush_r.sum()
        pa.kv_append(db.k_new, db.v_new, db.k_pool, db.v_pool, db.cu_seqlens_q, db.context_lens, db.block_tables,
                     batch.n_seq, batch.n_tok)
        pa.batch_attention(db.q, db.k_pool, db.v_pool, db.cu_seqlens_q, db.context_lens, db.block_tables,
                           batch.softmax_scale, db.out)

    for _ in range(4):
        step()
    torch.cuda.synchronize()
    off, nbytes = pa.plan_info(100), stamp_bytes
    pa.workspace[off:off + nbytes].zero_()
    step()
    torch.cuda.synchronize()
    raw = pa.workspace[off:off + nbytes].cpu().numpy().view(np.int64)
    tl, cta = raw[:16 * 400 * 4].reshape(16, 400, 4), raw[16 * 400 * 4:].reshape(148, 4)
    print(f"case {batch.name}: decode items {pa.plan_info(0)}, bundles {pa.plan_info(1)}, split items {pa.plan_info(2)}, "
          f"prefill tiles {pa.plan_info(3)}, CTAs {pa.plan_info(4)} (prefill role: {pa.plan_info(6)}); stamped CTA {args.cta}")
    t0 = tl[15, 399, 0]

    def rel(x):
        return np.where(x > 0, x - t0, -1)

    print(f"kernel entry -> roles start: {int(rel(tl[15, 399, 1]))} cycles; role passes end at {rel(tl[15, 397:399, 0]).tolist()}")
    n = int((tl[0, :, 3] > 0).sum())
    if n:
        print(f"stream 0 of CTA {args.cta}: {n} items.  cycles since kernel entry:")
        print("  item | consumer: wait for item, got it, blocks done, item end | K ready, S done, softmax done, V ready | "
              "epilogue: start, stmatrix done, stores done, fence done | producer: fifo wait, got slot, Q issued, K/V issued")
        for i in range(min(n, 12)):
            print(f"  {i:4d} | {rel(tl[0, i]).tolist()} | {rel(tl[2, i]).tolist()} | {rel(tl[5, i]).tolist()} | {rel(tl[1, i]).tolist()}")
    if n > 3:
        def seg(a, b):
            d = (b - a)[1:n]
            d = d[(a[1:n] > 0) & (b[1:n] > 0)]
            return float(np.median(d)) if len(d) else float("nan")

        print(f"  item period (median over items 1..{n - 1}): {float(np.median(np.diff(tl[0, 1:n, 3]))):.0f} cycles")
        print("  consumer phases (median cycles): " + ", ".join(f"{k} {v:.0f}" for k, v in [
            ("wait for item", seg(tl[0, :, 0], tl[0, :, 1])), ("wait for K", seg(tl[0, :, 1], tl[2, :, 0])),
            ("S", seg(tl[2, :, 0], tl[2, :, 1])), ("softmax", seg(tl[2, :, 1], tl[2, :, 2])),
            ("wait for V", seg(tl[2, :, 2], tl[2, :, 3])), ("dead-row zero fill", seg(tl[2, :, 3], tl[3, :, 0])),
            ("PV", seg(tl[3, :, 0], tl[0, :, 2])), ("row-sum reduction", seg(tl[0, :, 2], tl[5, :, 0])),
            ("stmatrix", seg(tl[5, :, 0], tl[5, :, 1])), ("output stores", seg(tl[5, :, 1], tl[5, :, 2])),
            ("fence", seg(tl[5, :, 2], tl[5, :, 3])), ("hand-back", seg(tl[5, :, 3], tl[0, :, 3]))]))
        print("  producer lane (median cycles): " + ", ".join(f"{k} {v:.0f}" for k, v in [
            ("fifo wait", seg(tl[1, :, 0], tl[1, :, 1])), ("descriptor + Q loads", seg(tl[1, :, 1], tl[1, :, 2])),
            ("K/V loads of the item", seg(tl[1, :, 2], tl[1, :, 3])), ("period", float(np.median(np.diff(tl[1, 1:n, 0]))))]))
    ok = cta[:, 0] > 0
    g = cta[ok, 0].min()
    ends = (cta[:, 1:3].max(axis=1) - g)[ok]
    q = lambda a: [int(np.min(a)), int(np.percentile(a, 10)), int(np.median(a)), int(np.percentile(a, 90)), int(np.max(a))]
    print(f"CTA leaves the kernel (ns after the first CTA's entry): min / p10 / median / p90 / max = {q(ends)}")
    if (cta[ok, 3] > 0).any():
        last_blk = (cta[:, 3] - g)[ok]
        print(f"CTA's last K/V block consumed (ns): {q(last_blk)}; from there to the CTA's end: {q(ends - last_blk)}")


if __name__ == "__main__":
    main()
