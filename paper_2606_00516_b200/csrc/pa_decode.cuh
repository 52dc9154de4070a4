// a5 + a6: bandwidth-bound split-KV decode attention with in-launch flash-decoding merge.
//
// Design.  The decode role of a CTA runs 8 independent *streams*.  A stream is a
// private ring of 4 KB shared-memory slots plus a 2-entry item fifo, filled by a producer lane and
// drained by one consumer warp; streams never synchronise with each other, only producer <-> consumer
// through mbarriers, so HBM requests of a stream keep flowing across item and bundle boundaries.
//   producer (warps 0-3, two lanes each, one stream per lane): walks the planner's bundles — runs of the
//     block stream of all (decode sequence, KV head) groups — and derives the (sequence, KV head, block
//     range) items from the bundle descriptor and context_lens; per item it writes the item descriptor
//     into the fifo and fetches the G query rows of that KV head with one TMA box per 64 columns; per block it
//     looks up the block table and issues TMA tensor loads (cp.async.bulk.tensor, 128B swizzle) of the
//     16-token K tile and V tile.  All of this runs ahead of the math by the ring depth, so block-table
//     and descriptor latencies are off the consumers' critical path;
//   consumer (warps 4-11): S^T = K·Q^T with warp-level mma.sync m16n8k16 (M = 16 tokens of the block,
//     N = the <= 8 q heads that share the KV head, K = head_dim), so K and V are read ONCE per KV head
//     and the G = Hq/Hkv FMAs per loaded element run on the tensor pipe, not the fp32 lanes;
//     online softmax over tokens with warp shuffles (xor 4, 8, 16); P^T re-laid-out for the second MMA
//     with movmatrix; O^T = V^T·P^T accumulates in registers;
//   an item that covers a whole (seq, head) writes its output rows directly; split groups write
//     (m, l, o) partials and the LAST arriving consumer merges them (m = max m_i, l = Σ l_i 2^{m_i-m},
//     o = Σ o_i 2^{m_i-m} / l) — one launch, no separate merge kernel.
// HBM-bound: algorithmic bytes per decode token = kv_len·kvb + 2·qb + 4·ceil(kv_len/16).
#pragma once
#include "pa_common.cuh"
#include "pa_internal.h"
#include "pa_launch.h"

namespace pa {

struct AttnParams {
    const __nv_bfloat16* q;       // [n_tok, Hq, D]
    __nv_bfloat16* out;           // [n_tok, Hq, D]
    const __nv_bfloat16* k_pool;  // pools as plain pointers: the plain row loop (debug kernel, overflow redo) reads them
    const __nv_bfloat16* v_pool;  //   directly; the decode and prefill roles see them through tensor maps only
    const int32_t* cu_seqlens_q;  // dev [n_seq+1]
    const int32_t* context_lens;  // dev [n_seq]
    const int32_t* block_tables;  // dev [n_seq, max_blocks_per_seq]
    int32_t max_blocks_per_seq;
    int32_t Hq, Hkv, G;
    float scale_log2;             // softmax_scale * log2(e)
    PlanView plan;
    int32_t decode_workers;       // decode streams with a statically assigned first bundle (= initial decode CTAs x 8)
    int32_t prefill_ctas;         // CTAs [0, prefill_ctas) start in the prefill role (first unit = blockIdx.x)
};

template <int D>
struct DecodeCfg {
    static constexpr int kUnit = 4096;                    // ring slot: 16 tokens x 128 columns (two 64-column TMA boxes)
    static constexpr int kHalves = D / 128;               // units per K (or V) tile of one block-head
    static constexpr int kRing = (D == 128) ? 6 : 5;      // slots per stream
    static constexpr int kFifo = 2;                       // items in flight per stream (descriptor + Q rows)
    static constexpr int kQSlot = (D / 64) * 1024;        // Q rows of one item: D/64 boxes of 8 rows x 128 B
    static constexpr int kStreamBytes = kRing * kUnit + kFifo * kQSlot;   // 28 KB
    // per-stream scratch: full[kRing], empty[kRing], ffull[kFifo], fempty[kFifo] mbarriers, then the descriptors
    static constexpr int kOffEmpty = 8 * kRing, kOffFFull = 16 * kRing, kOffFEmpty = 16 * kRing + 8 * kFifo;
    static constexpr int kOffDesc = 128;
    static constexpr int kAuxBytes = 192;
    static_assert(kOffFEmpty + 8 * kFifo <= kOffDesc && kOffDesc + kFifo * 32 <= kAuxBytes, "decode scratch layout");
    static_assert(kStreamBytes == 28 * 1024, "decode stream bytes");
};
constexpr int kDecodeProducerWarps = 4;                              // warps 0-3
constexpr int kStreamsPerProducer = kDecodeWarps / kDecodeProducerWarps;

// one thread per stream, once per CTA, before the roles start
template <int D>
__device__ __forceinline__ void decode_init_barriers(uint8_t* dec_aux, int s) {
    using Cfg = DecodeCfg<D>;
    const uint32_t a = smem_u32(dec_aux + s * Cfg::kAuxBytes);
    for (int i = 0; i < 2 * Cfg::kRing + 2 * Cfg::kFifo; ++i) mbar_init(a + 8 * i, 1);
}

// ------------------------------------------------------------------------------------------------
// Producer lane of one stream.  first_bundle: the statically assigned first bundle, or -1 for a stream
// that joins late (its CTA finished the prefill role) and takes every bundle from the queue.
// ------------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void decode_producer(const AttnParams& p, const CUtensorMap* tmQd, const CUtensorMap* tmK,
                                                const CUtensorMap* tmV, const TailMaps* tails, uint8_t* stream_mem,
                                                uint8_t* aux, int first_bundle) {
    using Cfg = DecodeCfg<D>;
    constexpr int R = Cfg::kRing, FQ = Cfg::kFifo, H = Cfg::kHalves;
    const PlanView& pl = p.plan;
    const uint32_t ring_u32 = smem_u32(stream_mem);
    const uint32_t q_u32 = ring_u32 + R * Cfg::kUnit;
    const uint32_t bar = smem_u32(aux);
    const uint32_t q_bytes = (uint32_t)p.G * D * 2;
    const uint64_t pol = policy_evict_first();

    uint32_t u_iss = 0, i_iss = 0;
    // ---- bundle walk.  The stream's first bundle is static (or queue-drawn for a late joiner); every further one
    // comes from the queue.  The queue index is requested two bundles ahead and the 32-byte descriptor one bundle
    // ahead of their use, so neither the atomic nor the descriptor load is waited on where it is issued.
    const int4* bundles = reinterpret_cast<const int4*>(pl.bundles);
    // tickets: level-major (PlanView::n_levels); ticket -> (level, bundle)
    const int n_tickets = pl.n_bundles * pl.n_levels;
    auto ticket_bundle = [&](int ticket, int& level) -> int {
        level = 0;
        if (pl.n_levels > 1) { level = ticket / pl.n_bundles; ticket -= level * pl.n_bundles; }
        return ticket;
    };
    auto level_cum = [&](int l) -> int { return l == 0 ? 0 : (int)((pl.level_cum >> (8 * (l - 1))) & 0xffu) + (l == pl.n_levels ? 1 : 0); };
    int b_next = first_bundle;
    if (b_next < 0) b_next = p.decode_workers + atomicAdd(&pl.queue[0], 1);
    int4 nd0 = make_int4(0, 0, -1, 0), nd1 = nd0;        // descriptor of the bundle of ticket b_next
    int lvl_next = 0;
    bool have_next = b_next < n_tickets;
    if (have_next) {
        const int bb = ticket_bundle(b_next, lvl_next);
        nd0 = __ldg(bundles + 2 * bb); nd1 = __ldg(bundles + 2 * bb + 1);
    }
    // no ticket beyond the statically assigned ones (pure decode with one bundle per stream): no queue traffic at all —
    // 1184 lanes hitting one counter at kernel start cost the first item ~1.5 us
    const bool dynamic = n_tickets > p.decode_workers;
    int b_after = (have_next && dynamic) ? p.decode_workers + atomicAdd(&pl.queue[0], 1) : n_tickets;
    int4 d0 = make_int4(0, 0, -1, 0), d1 = d0;           // current bundle: {grp_begin, blk_begin, grp_end, blk_end}, parts
    int grp = 0, grp_last = -1;
    // A group of the walk, with its context length in flight: {seq, kv head, blk_begin, blk_end or -1}, {ctx, part_base, part}
    auto next_group = [&](int4& ga, int4& gb, int& gn) -> bool {
        while (grp > grp_last) {
            if (!have_next) return false;
            d0 = nd0; d1 = nd1;
            const int lvl = lvl_next;
            have_next = b_after < n_tickets;
            if (have_next) {
                const int bb = ticket_bundle(b_after, lvl_next);
                nd0 = __ldg(bundles + 2 * bb); nd1 = __ldg(bundles + 2 * bb + 1);
                b_after = p.decode_workers + atomicAdd(&pl.queue[0], 1);
            }
            if (pl.n_levels > 1) {
                const int n = d0.z - d0.x + 1;           // groups of the bundle; this ticket takes its piece `lvl`
                grp = d0.x + ((n * level_cum(lvl)) >> 8);
                grp_last = d0.x + ((n * level_cum(lvl + 1)) >> 8) - 1;      // empty piece: try the next ticket
            } else {
                grp = d0.x; grp_last = d0.z;
            }
        }
        const int seq = grp / p.Hkv, kvh = grp - seq * p.Hkv;
        const bool first = grp == d0.x, last = grp == d0.z;
        ga = make_int4(seq, kvh, first ? d0.y : 0, last ? d0.w : -1);
        // the ids of the group's first two blocks are requested together with its context length (their addresses do
        // not depend on it; the second entry is inside the table row and never dereferenced unless the block exists)
        const int32_t* bt0 = p.block_tables + (int64_t)seq * p.max_blocks_per_seq + ga.z;
        gb = make_int4(__ldg(p.context_lens + seq), first ? d1.x : (last ? d1.z : -1), first ? d1.y : (last ? d1.w : 1), __ldg(bt0));
        gn = (ga.z + 1 < p.max_blocks_per_seq) ? __ldg(bt0 + 1) : 0;
        ++grp;
        return true;
    };
    // turns a fetched group into the item descriptor (DecItem layout) once its context length has arrived
    auto resolve = [&](int4& ga, int4& gb, int& first_id) {
        const int kv_len = gb.x + 1, nblk = (kv_len + kBlock - 1) / kBlock;
        if (ga.w < 0) ga.w = nblk;
        const int part = gb.z;
        first_id = gb.w;
        gb = make_int4(kv_len, gb.y, gb.y < 0 ? 0 : (part >> 16), gb.y < 0 ? 1 : (part & 0xffff));
    };
    // Two-deep software pipeline over items so that no load is waited on where it is issued:
    //   stage 2: context length and first block ids of item i+2 in flight;  stage 1: item i+1 resolved.
    int4 a1 = make_int4(0, 0, 0, 0), b1 = a1, a2 = a1, b2 = a1;
    int blkid1 = 0, blkid1n = 0, n2 = 0;      // ids of the first two blocks of the stage-1 item; second id of stage 2
    if (threadIdx.x == 0) PA_TL(4, 0, 2);
    bool v2 = next_group(a2, b2, n2);
    bool v1 = v2;
    if (threadIdx.x == 0) PA_TL(4, 0, 3);
    if (v1) {
        a1 = a2; b1 = b2; blkid1n = n2;
        resolve(a1, b1, blkid1);
        if (threadIdx.x == 0) PA_TL(4, 1, 0);
        v2 = next_group(a2, b2, n2);
        if (threadIdx.x == 0) PA_TL(4, 1, 1);
    }
    while (v1) {
        const int4 a = a1, b = b1;
        int blkid = blkid1, blkid_n = blkid1n;
        // ---- advance the pipeline
        v1 = v2;
        if (v1) {
            a1 = a2; b1 = b2; blkid1n = n2;
            resolve(a1, b1, blkid1);
            v2 = next_group(a2, b2, n2);
        }
        // ---- open the item: descriptor + Q rows into the fifo entry
        const int seq = a.x, kvh = a.y, blk_end = a.w, kv_len = b.x;
        int blk = a.z;
        const int32_t* bt = p.block_tables + (int64_t)seq * p.max_blocks_per_seq;
        {
            const uint32_t fs = i_iss % FQ;
            if (threadIdx.x == 0) PA_TL(1, (int)i_iss, 0);
            mbar_wait(bar + Cfg::kOffFEmpty + 8 * fs, ((i_iss / FQ) & 1u) ^ 1u);
            if (threadIdx.x == 0) PA_TL(1, (int)i_iss, 1);
            const uint32_t d = smem_u32(aux + Cfg::kOffDesc + 32 * fs);
            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(d), "r"(a.x), "r"(a.y), "r"(a.z), "r"(a.w) : "memory");
            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(d + 16), "r"(b.x), "r"(b.y), "r"(b.z), "r"(b.w) : "memory");
            const uint32_t ff = bar + Cfg::kOffFFull + 8 * fs;
            mbar_expect_tx(ff, q_bytes);
            // decode sequences come first with q_len == 1 (R11), so the packed query row of sequence s is s
            const int qrow = seq * p.Hq + kvh * p.G;
#pragma unroll
            for (int c = 0; c < D / 64; ++c) tma_load_2d(q_u32 + fs * Cfg::kQSlot + c * 1024, tmQd, ff, c * 64, qrow);
            ++i_iss;
            if (threadIdx.x == 0) PA_TL(1, (int)i_iss - 1, 2);
        }
        // ---- stream the K and V tiles of the item's blocks
        while (blk < blk_end) {
            const int cur = blkid;
            const int nvalid = min(kBlock, kv_len - blk * kBlock);   // filled rows of this block
            ++blk;
            blkid = blkid_n;
            if (blk + 1 < blk_end) blkid_n = __ldg(bt + blk + 1);   // block ids are fetched two blocks ahead of their use
#pragma unroll
            for (int isV = 0; isV < 2; ++isV) {
#pragma unroll
                for (int h = 0; h < H; ++h) {
                    const uint32_t slot = u_iss % R;
                    mbar_wait(bar + Cfg::kOffEmpty + 8 * slot, ((u_iss / R) & 1u) ^ 1u);
                    const uint32_t full = bar + 8 * slot, dst = ring_u32 + slot * Cfg::kUnit;
                    if (nvalid == kBlock) {
                        mbar_expect_tx(full, Cfg::kUnit);
                        tma_load_5d_hint(dst, isV ? &tails->v[0] : &tails->k[0], full, 0, 0, 2 * h, kvh, cur, pol);
                    } else {
                        // partly filled last block: rows [0, nvalid) as 8 + 4 + 2 + 1 row boxes of ONE column plane each
                        // (a short two-plane box would put plane 1 at rows·128 B, not at the slot's 2048 B plane offset;
                        // the 128B swizzle pattern depends on the shared-memory address only, rows are 128 B apart)
                        mbar_expect_tx(full, nvalid * 256);
                        int r0 = 0;
#pragma unroll
                        for (int i = 1; i < 5; ++i) {
                            if (nvalid & (16 >> i)) {
                                const CUtensorMap* tm = isV ? &tails->v[i] : &tails->k[i];
                                tma_load_5d_hint(dst + r0 * 128, tm, full, 0, r0, 2 * h, kvh, cur, pol);
                                tma_load_5d_hint(dst + 2048 + r0 * 128, tm, full, 0, r0, 2 * h + 1, kvh, cur, pol);
                                r0 += 16 >> i;
                            }
                        }
                    }
                    ++u_iss;
                }
            }
        }
        if (threadIdx.x == 0) PA_TL(1, (int)i_iss - 1, 3);
    }
    // ---- sentinel item: tells the consumer that the stream is finished
    {
        const uint32_t fs = i_iss % FQ;
        mbar_wait(bar + Cfg::kOffFEmpty + 8 * fs, ((i_iss / FQ) & 1u) ^ 1u);
        const uint32_t d = smem_u32(aux + Cfg::kOffDesc + 32 * fs);
        asm volatile("st.shared.b32 [%0], %1;" ::"r"(d), "r"(-1) : "memory");
        mbar_arrive(bar + Cfg::kOffFFull + 8 * fs);
    }
}

// ------------------------------------------------------------------------------------------------
// a6 merge of one split (sequence, KV head) group by one warp: m = max m_i, l = Σ l_i 2^{m_i-m},
// o = Σ o_i 2^{m_i-m} / l.  Lane (i, h) = (lane / 8, lane % 8) owns the (m, l) of part c0 + i, head h, so the
// statistics of four parts arrive with ONE coalesced load and reduce with two shuffles; the partial outputs
// of those four parts are then fetched for all heads at once (loads of heads >= G are clamped duplicates, so
// that no load waits on a branch) — the merge costs a few L2 round trips, not a few per head.
// ------------------------------------------------------------------------------------------------
template <int D, int GG>
__device__ __forceinline__ void decode_merge(const AttnParams& p, const DecItem& ci, int q_row, int h0, int lane) {
    constexpr int VPL = D / 32;                  // floats per lane
    const PlanView& pl = p.plan;
    const int G = p.G, np = ci.n_parts;
    const int pi = lane >> 3, hl = lane & 7;
    const float2* ml_base = pl.part_ml + (int64_t)ci.part_base * kMaxGroup;
    float M = -INFINITY;
    for (int c0 = 0; c0 < np; c0 += 4)
        if (c0 + pi < np) M = fmaxf(M, __ldcg(ml_base + (c0 + pi) * kMaxGroup + hl).x);
    M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, 8));
    M = fmaxf(M, __shfl_xor_sync(0xffffffffu, M, 16));          // max of head hl over all parts, on every lane
    float L = 0.f, acc[GG][VPL];
#pragma unroll
    for (int h = 0; h < GG; ++h)
#pragma unroll
        for (int k = 0; k < VPL; ++k) acc[h][k] = 0.f;
    // PB parts' partial outputs are fetched together (as many as the register budget allows) and the (m, l) of
    // the next four parts are already in flight, so a group of n parts costs ~n/PB + n/4 L2 round trips
    // the accumulators of the item are dead by now, so 64 registers can hold partial outputs in flight:
    // a group of many parts (a few long sequences split over every stream) is merged by ONE warp at the very end of the
    // launch, and its time is the number of L2 round trips
    constexpr int PB = (GG * VPL <= 16) ? 4 : ((GG * VPL <= 32) ? 2 : 1);
    float2 ml_next = make_float2(-INFINITY, 0.f);
    if (pi < np) ml_next = __ldcg(ml_base + pi * kMaxGroup + hl);
    for (int c0 = 0; c0 < np; c0 += 4) {
        const float2 ml = ml_next;
        if (c0 + 4 + pi < np) ml_next = __ldcg(ml_base + (c0 + 4 + pi) * kMaxGroup + hl);
        float w = 0.f;
        if (c0 + pi < np) {
            w = fast_exp2(ml.x - M);
            L += ml.y * w;
        }
        const int nk = min(4, np - c0);
#pragma unroll
        for (int k0 = 0; k0 < 4; k0 += PB) {
            if (k0 < nk) {
                float4 v[PB][GG][VPL / 4];
#pragma unroll
                for (int kk = 0; kk < PB; ++kk) {
                    const int part = ci.part_base + c0 + min(k0 + kk, nk - 1);      // clamped duplicate past the end
                    const float* src = pl.part_o + (int64_t)part * G * D + lane * VPL;
#pragma unroll
                    for (int h = 0; h < GG; ++h)
#pragma unroll
                        for (int x = 0; x < VPL / 4; ++x)
                            v[kk][h][x] = __ldcg(reinterpret_cast<const float4*>(src + min(h, G - 1) * D) + x);
                }
#pragma unroll
                for (int kk = 0; kk < PB; ++kk) {
#pragma unroll
                    for (int h = 0; h < GG; ++h) {
                        float wk = __shfl_sync(0xffffffffu, w, (k0 + kk) * 8 + h);
                        if (k0 + kk >= nk) wk = 0.f;
#pragma unroll
                        for (int x = 0; x < VPL / 4; ++x) {
                            acc[h][4 * x] += wk * v[kk][h][x].x; acc[h][4 * x + 1] += wk * v[kk][h][x].y;
                            acc[h][4 * x + 2] += wk * v[kk][h][x].z; acc[h][4 * x + 3] += wk * v[kk][h][x].w;
                        }
                    }
                }
            }
        }
    }
    L += __shfl_xor_sync(0xffffffffu, L, 8);
    L += __shfl_xor_sync(0xffffffffu, L, 16);
#pragma unroll
    for (int h = 0; h < GG; ++h) {
        const float inv = 1.f / __shfl_sync(0xffffffffu, L, h);
        if (h < G) {
            uint32_t packed[VPL / 2];
#pragma unroll
            for (int k = 0; k < VPL / 2; ++k) packed[k] = pack_bf16x2(acc[h][2 * k] * inv, acc[h][2 * k + 1] * inv);
            uint32_t* dst = reinterpret_cast<uint32_t*>(p.out + ((int64_t)q_row * p.Hq + h0 + h) * D + lane * VPL);
            if constexpr (VPL == 4) *reinterpret_cast<uint2*>(dst) = make_uint2(packed[0], packed[1]);
            else *reinterpret_cast<uint4*>(dst) = make_uint4(packed[0], packed[1], packed[2], packed[3]);
        }
    }
}

// The filled rows of a partly filled last block are fetched (8/4/2/1-row boxes); the other rows of the V slot keep
// whatever the slot held.  P of those rows is exactly 0, but 0 x NaN would poison O, so they are cleared: the slot is
// [plane][row][128 B] = 256 consecutive 16-byte chunks, lane l owns chunks l + 32k (row = (l / 8 + 4k) mod 16).
__device__ __forceinline__ void decode_zero_dead_rows(uint32_t tile, int nvalid, int lane) {
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const int row = ((lane >> 3) + 4 * k) & 15;
        if (row >= nvalid)
            asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(tile + (uint32_t)(lane + 32 * k) * 16u), "r"(0u) : "memory");
    }
    __syncwarp();
}

// ------------------------------------------------------------------------------------------------
// Consumer warp of one stream.
// ------------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void decode_consumer(const AttnParams& p, uint8_t* stream_mem, uint8_t* aux) {
    using Cfg = DecodeCfg<D>;
    constexpr int R = Cfg::kRing, FQ = Cfg::kFifo, H = Cfg::kHalves, KS = D / 16;
    const int lane = lane_id(), g = lane >> 2, t = lane & 3;
    const uint32_t ring_u32 = smem_u32(stream_mem);
    const uint32_t q_u32 = ring_u32 + R * Cfg::kUnit;
    const uint32_t bar = smem_u32(aux);
    const PlanView& pl = p.plan;
    const int G = p.G;
    const uint32_t mi = lane >> 3, r8 = lane & 7;

    uint32_t u_con = 0, i_con = 0;
    for (;;) {
        const uint32_t fs = i_con % FQ;
        if (threadIdx.x == 128) PA_TL(0, (int)i_con, 0);
        mbar_wait(bar + Cfg::kOffFFull + 8 * fs, (i_con / FQ) & 1u);
        if (threadIdx.x == 128) PA_TL(0, (int)i_con, 1);
        const DecItem ci = *reinterpret_cast<const DecItem*>(aux + Cfg::kOffDesc + 32 * fs);
        if (ci.seq < 0) break;
        const uint32_t qs = q_u32 + fs * Cfg::kQSlot;
        const int q_row = ci.seq, h0 = ci.kv_head * G;
        float m0 = -INFINITY, m1 = -INFINITY, l0 = 0.f, l1 = 0.f;
        float o[KS][4];
#pragma unroll
        for (int i = 0; i < KS; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;

        int blk = ci.blk_begin;
        if constexpr (H == 1) {
            // ---- two blocks per iteration (D = 128: K, V, K, V of the pair fit the ring).  Both score tiles are computed
            // first, ONE online-softmax update serves the 32 tokens (half the shuffles, exponentials of the correction
            // and rescale multiplies per block), then both PV products: a lone in-order warp hides the latencies of the
            // four MMA chains in each other.  Only the second block of a pair can be a partly filled last block.
            for (; blk + 1 < ci.blk_end; blk += 2) {
                const int nvalidB = min(16, ci.kv_len - (blk + 1) * kBlock);
                const uint32_t sKA = u_con % R, sVA = (u_con + 1) % R, sKB = (u_con + 2) % R, sVB = (u_con + 3) % R;
                const uint32_t phKA = (u_con / R) & 1u, phVA = ((u_con + 1) / R) & 1u, phKB = ((u_con + 2) / R) & 1u,
                               phVB = ((u_con + 3) / R) & 1u;
                float sA0[4] = {0.f, 0.f, 0.f, 0.f}, sA1[4] = {0.f, 0.f, 0.f, 0.f};
                float sB0[4] = {0.f, 0.f, 0.f, 0.f}, sB1[4] = {0.f, 0.f, 0.f, 0.f};
                const uint32_t tKA = ring_u32 + sKA * Cfg::kUnit, tKB = ring_u32 + sKB * Cfg::kUnit;
                const uint32_t rowk = r8 + 8 * (mi & 1);
                mbar_wait(bar + 8 * sKA, phKA);
                mbar_wait(bar + 8 * sKB, phKB);
                if (threadIdx.x == 128) PA_TL(2, (int)i_con, 0);
#pragma unroll
                for (int k2 = 0; k2 < 4; ++k2) {
                    uint32_t qf[4];
                    const uint32_t cq = 4 * k2 + mi;
                    ldmatrix_x4(qf, qs + (cq >> 3) * 1024 + swz128(r8, cq & 7));
#pragma unroll
                    for (int kk = 0; kk < 2; ++kk) {
                        const uint32_t chunk = 2 * (2 * k2 + kk) + (mi >> 1);
                        const uint32_t off = (chunk >> 3) * 2048 + swz128(rowk, chunk & 7);
                        uint32_t a[4], b[4];
                        ldmatrix_x4(a, tKA + off);
                        ldmatrix_x4(b, tKB + off);
                        if (kk) { mma_bf16_16816(sA1, a, qf[2], qf[3]); mma_bf16_16816(sB1, b, qf[2], qf[3]); }
                        else    { mma_bf16_16816(sA0, a, qf[0], qf[1]); mma_bf16_16816(sB0, b, qf[0], qf[1]); }
                    }
                }
                __syncwarp();
                if (lane == 0) { mbar_arrive(bar + Cfg::kOffEmpty + 8 * sKA); mbar_arrive(bar + Cfg::kOffEmpty + 8 * sKB); }
                if (threadIdx.x == 128) PA_TL(2, (int)i_con, 1);
                // tokens g, g + 8 of block A (s0..s3) and of block B (s4..s7), heads 2t / 2t + 1
                float s0 = (sA0[0] + sA1[0]) * p.scale_log2, s1 = (sA0[1] + sA1[1]) * p.scale_log2;
                float s2 = (sA0[2] + sA1[2]) * p.scale_log2, s3 = (sA0[3] + sA1[3]) * p.scale_log2;
                float s4 = (sB0[0] + sB1[0]) * p.scale_log2, s5 = (sB0[1] + sB1[1]) * p.scale_log2;
                float s6 = (sB0[2] + sB1[2]) * p.scale_log2, s7 = (sB0[3] + sB1[3]) * p.scale_log2;
                if (g >= nvalidB) { s4 = -INFINITY; s5 = -INFINITY; }
                if (g + 8 >= nvalidB) { s6 = -INFINITY; s7 = -INFINITY; }
                float mx0 = fmaxf(fmaxf(s0, s2), fmaxf(s4, s6)), mx1 = fmaxf(fmaxf(s1, s3), fmaxf(s5, s7));
#pragma unroll
                for (int off = 4; off <= 16; off <<= 1) {
                    mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, off));
                    mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, off));
                }
                const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);
                const float c0 = fast_exp2(m0 - mn0), c1 = fast_exp2(m1 - mn1);
                const float p0 = fast_exp2(s0 - mn0), p1 = fast_exp2(s1 - mn1), p2 = fast_exp2(s2 - mn0), p3 = fast_exp2(s3 - mn1);
                const float p4 = fast_exp2(s4 - mn0), p5 = fast_exp2(s5 - mn1), p6 = fast_exp2(s6 - mn0), p7 = fast_exp2(s7 - mn1);
                m0 = mn0; m1 = mn1;
                l0 = l0 * c0 + (p0 + p2) + (p4 + p6);
                l1 = l1 * c1 + (p1 + p3) + (p5 + p7);
                if (__any_sync(0xffffffffu, c0 != 1.f || c1 != 1.f)) {     // the running max of long contexts rarely moves
#pragma unroll
                    for (int i = 0; i < KS; ++i) { o[i][0] *= c0; o[i][1] *= c1; o[i][2] *= c0; o[i][3] *= c1; }
                }
                const uint32_t pA0 = movmatrix_trans(pack_bf16x2(p0, p1)), pA1 = movmatrix_trans(pack_bf16x2(p2, p3));
                const uint32_t pB0 = movmatrix_trans(pack_bf16x2(p4, p5)), pB1 = movmatrix_trans(pack_bf16x2(p6, p7));
                const uint32_t tVA = ring_u32 + sVA * Cfg::kUnit, tVB = ring_u32 + sVB * Cfg::kUnit;
                const uint32_t rowv = r8 + 8 * (mi >> 1);
                if (threadIdx.x == 128) PA_TL(2, (int)i_con, 2);
                mbar_wait(bar + 8 * sVA, phVA);
                mbar_wait(bar + 8 * sVB, phVB);
                if (threadIdx.x == 128) PA_TL(2, (int)i_con, 3);
                if (nvalidB < 16) decode_zero_dead_rows(tVB, nvalidB, lane);
                if (threadIdx.x == 128) PA_TL(3, (int)i_con, 0);
#pragma unroll
                for (int i = 0; i < 8; ++i) {      // block A first, then block B: dependent MMAs of o[i] are eight apart
                    const uint32_t chunk = 2 * i + (mi & 1);
                    uint32_t a[4];
                    ldmatrix_x4_trans(a, tVA + (chunk >> 3) * 2048 + swz128(rowv, chunk & 7));
                    mma_bf16_16816(o[i], a, pA0, pA1);
                }
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const uint32_t chunk = 2 * i + (mi & 1);
                    uint32_t b[4];
                    ldmatrix_x4_trans(b, tVB + (chunk >> 3) * 2048 + swz128(rowv, chunk & 7));
                    mma_bf16_16816(o[i], b, pB0, pB1);
                }
                if (nvalidB < 16) fence_proxy_async();   // generic-proxy zero fill before the slot's next TMA write
                __syncwarp();
                if (lane == 0) { mbar_arrive(bar + Cfg::kOffEmpty + 8 * sVA); mbar_arrive(bar + Cfg::kOffEmpty + 8 * sVB); }
                u_con += 4;
            }
        }
        for (; blk < ci.blk_end; ++blk) {
            const int nvalid = min(16, ci.kv_len - blk * kBlock);
            // ---- S^T[16 tok x 8 heads] = K[16 x D] · Q^T[D x 8]
            float sa[4] = {0.f, 0.f, 0.f, 0.f}, sb[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int h = 0; h < H; ++h) {
                const uint32_t slot = u_con % R;
                mbar_wait(bar + 8 * slot, (u_con / R) & 1u);
                const uint32_t tile = ring_u32 + slot * Cfg::kUnit;
                const uint32_t row = r8 + 8 * (mi & 1);
#pragma unroll
                for (int k2 = 0; k2 < 4; ++k2) {     // pairs of k-steps within the 128-column unit
                    uint32_t qf[4];
                    {   // B fragments of k-steps 2k2, 2k2+1: matrices = 16-byte chunks 4k2 + mi of the q rows
                        const uint32_t cq = h * 16 + 4 * k2 + mi;
                        ldmatrix_x4(qf, qs + (cq >> 3) * 1024 + swz128(r8, cq & 7));
                    }
#pragma unroll
                    for (int kk = 0; kk < 2; ++kk) {
                        const uint32_t chunk = 2 * (2 * k2 + kk) + (mi >> 1);     // 16-byte chunk along d within the unit
                        uint32_t a[4];
                        ldmatrix_x4(a, tile + (chunk >> 3) * 2048 + swz128(row, chunk & 7));
                        if (kk) mma_bf16_16816(sb, a, qf[2], qf[3]);
                        else    mma_bf16_16816(sa, a, qf[0], qf[1]);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(bar + Cfg::kOffEmpty + 8 * slot);
                ++u_con;
            }
            // thread holds tokens g (s0,s1) and g+8 (s2,s3) for heads 2t (s0,s2) and 2t+1 (s1,s3)
            float s0 = (sa[0] + sb[0]) * p.scale_log2, s1 = (sa[1] + sb[1]) * p.scale_log2;
            float s2 = (sa[2] + sb[2]) * p.scale_log2, s3 = (sa[3] + sb[3]) * p.scale_log2;
            if (g >= nvalid) { s0 = -INFINITY; s1 = -INFINITY; }
            if (g + 8 >= nvalid) { s2 = -INFINITY; s3 = -INFINITY; }
            float mx0 = fmaxf(s0, s2), mx1 = fmaxf(s1, s3);
#pragma unroll
            for (int off = 4; off <= 16; off <<= 1) {
                mx0 = fmaxf(mx0, __shfl_xor_sync(0xffffffffu, mx0, off));
                mx1 = fmaxf(mx1, __shfl_xor_sync(0xffffffffu, mx1, off));
            }
            const float mn0 = fmaxf(m0, mx0), mn1 = fmaxf(m1, mx1);
            const float c0 = fast_exp2(m0 - mn0), c1 = fast_exp2(m1 - mn1);
            const float p0 = fast_exp2(s0 - mn0), p1 = fast_exp2(s1 - mn1);
            const float p2 = fast_exp2(s2 - mn0), p3 = fast_exp2(s3 - mn1);
            m0 = mn0; m1 = mn1;
            l0 = l0 * c0 + p0 + p2;       // per-lane partial sums; reduced over g at item end
            l1 = l1 * c1 + p1 + p3;
#pragma unroll
            for (int i = 0; i < KS; ++i) { o[i][0] *= c0; o[i][1] *= c1; o[i][2] *= c0; o[i][3] *= c1; }
            // P^T as the B operand of the second MMA (k = token, n = head): transpose the two 8x8 tiles
            const uint32_t pb0 = movmatrix_trans(pack_bf16x2(p0, p1));
            const uint32_t pb1 = movmatrix_trans(pack_bf16x2(p2, p3));
            // ---- O^T[D x 8 heads] += V^T[D x 16 tok] · P^T[16 tok x 8]
#pragma unroll
            for (int h = 0; h < H; ++h) {
                const uint32_t slot = u_con % R;
                mbar_wait(bar + 8 * slot, (u_con / R) & 1u);
                const uint32_t tile = ring_u32 + slot * Cfg::kUnit;
                if (nvalid < 16) decode_zero_dead_rows(tile, nvalid, lane);
                const uint32_t row = r8 + 8 * (mi >> 1);               // token
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const uint32_t chunk = 2 * i + (mi & 1);
                    uint32_t a[4];
                    ldmatrix_x4_trans(a, tile + (chunk >> 3) * 2048 + swz128(row, chunk & 7));
                    mma_bf16_16816(o[h * 8 + i], a, pb0, pb1);
                }
                if (nvalid < 16) fence_proxy_async();   // generic-proxy zero fill before the slot's next TMA write
                __syncwarp();
                if (lane == 0) mbar_arrive(bar + Cfg::kOffEmpty + 8 * slot);
                ++u_con;
            }
        }
        // ---------------- item finished
        if (threadIdx.x == 128) PA_TL(0, (int)i_con, 2);
        if (lane == 0) PA_TL_CTA(3);        // (instrumented build only) the CTA's latest "blocks of an item consumed"
        ++i_con;
#pragma unroll
        for (int off = 4; off <= 16; off <<= 1) {
            l0 += __shfl_xor_sync(0xffffffffu, l0, off);
            l1 += __shfl_xor_sync(0xffffffffu, l1, off);
        }
        const int ha = 2 * t, hb = 2 * t + 1;
        if (ci.n_parts == 1) {
            // O^T fragments (row d, columns head 2t / 2t+1) -> out[q_row][h0 .. h0+G)[:], G·D·2 contiguous bytes: the 8x8
            // matrices are stored TRANSPOSED (stmatrix.trans) into the item's (now idle) Q slot as [head][d] rows, 16-byte
            // chunks XOR-swizzled by head, and leave as whole 16-byte vectors, consecutive lanes on consecutive addresses
            const float i0 = 1.f / l0, i1 = 1.f / l1;
            __syncwarp();                                   // every lane is done with the Q rows of the slot
            if (threadIdx.x == 128) PA_TL(5, (int)i_con - 1, 0);
#pragma unroll
            for (int i = 0; i < KS; i += 2) {
                const uint32_t mm = (uint32_t)lane >> 3, hh = (uint32_t)lane & 7u;     // matrix (i + mm/2, half mm%2), head row hh
                const uint32_t cc = (uint32_t)(2 * (i + (int)(mm >> 1))) + (mm & 1u);  // 16-byte chunk = 8 consecutive d
                const uint32_t addr = qs + hh * (uint32_t)(2 * D) + (((cc ^ hh) & (uint32_t)(D / 8 - 1))) * 16u;
                asm volatile("stmatrix.sync.aligned.m8n8.x4.trans.shared.b16 [%0], {%1, %2, %3, %4};"
                             ::"r"(addr), "r"(pack_bf16x2(o[i][0] * i0, o[i][1] * i1)), "r"(pack_bf16x2(o[i][2] * i0, o[i][3] * i1)),
                               "r"(pack_bf16x2(o[i + 1][0] * i0, o[i + 1][1] * i1)), "r"(pack_bf16x2(o[i + 1][2] * i0, o[i + 1][3] * i1))
                             : "memory");
            }
            __syncwarp();
            if (threadIdx.x == 128) PA_TL(5, (int)i_con - 1, 1);
            uint4* dst = reinterpret_cast<uint4*>(p.out + ((int64_t)q_row * p.Hq + h0) * D);
            for (int q = lane; q < G * (D / 8); q += 32) {
                const uint32_t hh = (uint32_t)q / (uint32_t)(D / 8), cc = (uint32_t)q % (uint32_t)(D / 8);
                uint4 v;
                asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                             : "r"(qs + hh * (uint32_t)(2 * D) + ((cc ^ hh) & (uint32_t)(D / 8 - 1)) * 16u));
                dst[q] = v;
            }
            __syncwarp();
            if (threadIdx.x == 128) PA_TL(5, (int)i_con - 1, 2);
            fence_proxy_async();                            // generic-proxy writes before the slot's next TMA fill
            if (threadIdx.x == 128) PA_TL(5, (int)i_con - 1, 3);
            if (lane == 0) mbar_arrive(bar + Cfg::kOffFEmpty + 8 * fs);    // Q slot and descriptor may be refilled
        } else {
            __syncwarp();
            if (lane == 0) mbar_arrive(bar + Cfg::kOffFEmpty + 8 * fs);    // Q rows and descriptor are no longer needed
            const int ps = ci.part_base + ci.part_idx;
            if (g == 0) {
                if (ha < G) pl.part_ml[ps * kMaxGroup + ha] = make_float2(m0, l0);
                if (hb < G) pl.part_ml[ps * kMaxGroup + hb] = make_float2(m1, l1);
            }
            float* pa_ = pl.part_o + ((int64_t)ps * G + ha) * D + g;
            float* pb_ = pa_ + D;
#pragma unroll
            for (int i = 0; i < KS; ++i) {
                if (ha < G) { pa_[16 * i] = o[i][0]; pa_[16 * i + 8] = o[i][2]; }
                if (hb < G) { pb_[16 * i] = o[i][1]; pb_[16 * i + 8] = o[i][3]; }
            }
            __threadfence();
            __syncwarp();
            int last = 0;
            int32_t* ctr = pl.group_counters + ci.seq * p.Hkv + ci.kv_head;
            if (lane == 0) last = (atomicAdd(ctr, 1) == ci.n_parts - 1);
            last = __shfl_sync(0xffffffffu, last, 0);
            if (last) {
                // ---------------- a6 merge by the last-arriving consumer
                __threadfence();
                if (G <= 4) decode_merge<D, 4>(p, ci, q_row, h0, lane);
                else decode_merge<D, 8>(p, ci, q_row, h0, lane);
                if (lane == 0) *ctr = 0;                      // self-reset for the next launch
            }
        }
        if (threadIdx.x == 128) PA_TL(0, (int)i_con - 1, 3);
    }
}

// The decode role of one CTA (12 warps): warps 0-3 produce (lanes 0,1 -> streams 2w, 2w+1), warps 4-11 consume.
// dec_rank >= 0: rank among the CTAs that START in the decode role (static first bundles, interleaved so that
// the first bundles land on distinct SMs); dec_rank < 0: late joiner, every bundle comes from the queue.
template <int D>
__device__ __forceinline__ void decode_role(const AttnParams& p, const CUtensorMap* tmQd, const CUtensorMap* tmK,
                                            const CUtensorMap* tmV, const TailMaps* tails, uint8_t* tiles, uint8_t* dec_aux,
                                            int dec_rank) {
    using Cfg = DecodeCfg<D>;
    const int warp = threadIdx.x >> 5, lane = lane_id();
    [[maybe_unused]] const PlanView& pl = p.plan;
    if (warp < kDecodeProducerWarps) {
        if (lane < kStreamsPerProducer) {
            const int s = warp * kStreamsPerProducer + lane;
            const int dec_ctas = p.decode_workers / kDecodeWarps;
            decode_producer<D>(p, tmQd, tmK, tmV, tails, tiles + s * Cfg::kStreamBytes, dec_aux + s * Cfg::kAuxBytes,
                               dec_rank >= 0 ? s * dec_ctas + dec_rank : -1);
        }
    } else {
        const int s = warp - kDecodeProducerWarps;
        decode_consumer<D>(p, tiles + s * Cfg::kStreamBytes, dec_aux + s * Cfg::kAuxBytes);
    }
    // The producer warps ran with two lanes in their own control flow: reconverge every warp before the caller's
    // __syncthreads().  A warp that reaches a CTA barrier in two pieces is counted twice, and the barrier would
    // release while consumer warps are still reading the ring (measured: thread 0 passed it ~7 us early).
    __syncwarp();
}

}  // namespace pa
