// a5 + a6: bandwidth-bound split-KV decode attention with in-launch flash-decoding merge.
//
// Design.  Every warp is an independent persistent worker that streams whole KV
// blocks of (decode sequence, KV head) items through its own ring of shared-memory slots:
//   * one elected lane issues TMA tensor loads (cp.async.bulk.tensor, 128B swizzle) of the 16-token
//     K tile and V tile of each block, addressed through the block table, running up to kRing-1
//     tiles ahead of the math — across item and bundle boundaries — so HBM requests never drain;
//   * S^T = K·Q^T is computed with warp-level mma.sync m16n8k16 (M = 16 tokens of the block, N = the
//     <= 8 q heads that share the KV head, K = head_dim), so K and V are read ONCE per KV head and the
//     G = Hq/Hkv FMAs per loaded element run on the tensor pipe, not the fp32 lanes;
//   * online softmax over tokens uses warp shuffles (xor 4, 8, 16); P^T is re-laid-out for the second
//     MMA with movmatrix; O^T = V^T·P^T accumulates in registers;
//   * an item that covers a whole (seq, head) writes its output row directly; split groups write
//     (m, l, o) partials and the LAST arriving worker merges them (m = max m_i, l = Σ l_i 2^{m_i-m},
//     o = Σ o_i 2^{m_i-m} / l) — one launch, no separate merge kernel.
// HBM-bound: algorithmic bytes per decode token = kv_len·kvb + 2·qb + 4·ceil(kv_len/16).
#pragma once
#include "pa_common.cuh"
#include "pa_internal.h"

namespace pa {

struct AttnParams {
    const __nv_bfloat16* q;       // [n_tok, Hq, D]
    __nv_bfloat16* out;           // [n_tok, Hq, D]
    const int32_t* cu_seqlens_q;  // dev [n_seq+1]
    const int32_t* context_lens;  // dev [n_seq]
    const int32_t* block_tables;  // dev [n_seq, max_blocks_per_seq]
    int32_t max_blocks_per_seq;
    int32_t Hq, Hkv, G;
    float scale_log2;             // softmax_scale * log2(e)
    PlanView plan;
    int32_t decode_workers;       // decode warps with a statically assigned first bundle (= initial decode CTAs x 8)
    int32_t prefill_ctas;         // CTAs [0, prefill_ctas) start in the prefill role (first unit = blockIdx.x)
};

template <int D>
struct DecodeCfg {
    static constexpr int kUnit = kBlock * D * 2;          // bytes of one K (or V) tile of one block-head
    static constexpr int kRingBytes = 24576;              // per warp
    static constexpr int kRing = kRingBytes / kUnit;      // 6 slots (D=128) / 3 slots (D=256)
    static constexpr int kKSteps = D / 16;                // k-steps of QK^T == m-tiles of O^T
    static constexpr int kBoxes = D / 64;                 // 64-column TMA boxes per tile
    static constexpr int kFifo = 4;                       // opened-but-unfinished items per warp
    static constexpr int kAuxBytes = 192;                 // per warp: kRing mbarriers (<= 48 B, at +0) + fifo (128 B, at +64)
    static constexpr int kWarpBytes = kRingBytes + kAuxBytes;
    static constexpr int kSmemBytes = kDecodeWarps * kRingBytes + kDecodeWarps * kAuxBytes + 1024;  // + align slack
};

// One persistent decode worker (a full warp).  ring: this warp's slot ring (1024-byte aligned);
// aux: this warp's 192-byte scratch (mbarriers, item fifo).  first_bundle: the statically assigned first
// bundle, or -1 for a worker that joins late (its CTA finished the prefill role) and takes every bundle
// from the queue.
template <int D>
__device__ __forceinline__ void decode_worker(const AttnParams& p, const CUtensorMap* tmK, const CUtensorMap* tmV,
                                              uint8_t* ring, uint8_t* aux, int first_bundle) {
    using Cfg = DecodeCfg<D>;
    constexpr int R = Cfg::kRing, UNIT = Cfg::kUnit, KS = Cfg::kKSteps, FQ = Cfg::kFifo;
    const int lane = lane_id(), g = lane >> 2, t = lane & 3;
    const uint32_t ring_u32 = smem_u32(ring);
    const uint32_t bar_u32 = smem_u32(aux);                       // kRing x 8 bytes
    DecItem* fifo = reinterpret_cast<DecItem*>(aux + 64);         // FQ x 32 bytes
    const PlanView& pl = p.plan;
    const int G = p.G;

    if (lane == 0) {
        for (int i = 0; i < R; ++i) mbar_init(bar_u32 + 8 * i, 1);
        fence_mbar_init();
        fence_proxy_async();
    }
    __syncwarp();

    uint32_t u_iss = 0, u_con = 0;
    // ---- issue cursor (warp-uniform except iss_blkid / nb_l0 which live in lane 0)
    int iss_item = 0, iss_item_end = 0;
    bool iss_open = false, iss_isV = false, queue_done = false;
    int iss_seq = 0, iss_kvh = 0, iss_blk = 0, iss_blk_end = 0, iss_blkid = 0;
    int next_bundle = first_bundle, nb_l0 = 0;
    bool have_prefetched = false;
    if (first_bundle < 0) {
        if (lane == 0) nb_l0 = p.decode_workers + atomicAdd(&pl.queue[0], 1);
        have_prefetched = true;
    }
    int f_head = 0, f_tail = 0;
    // ---- consume cursor
    bool con_open = false, con_isV = false;
    DecItem ci = {};
    int con_blk = 0, nvalid = 16, q_row = 0, h0 = 0;
    float m0 = 0.f, m1 = 0.f, l0 = 0.f, l1 = 0.f;
    float o[KS][4];
    uint32_t qf[KS][2];
    uint32_t pb0 = 0, pb1 = 0;

    for (;;) {
        // =============================== issue side: keep the ring full
        while (u_iss - u_con < (uint32_t)R) {
            if (!iss_open) {
                if (iss_item >= iss_item_end) {
                    if (queue_done) break;
                    if (have_prefetched) next_bundle = __shfl_sync(0xffffffffu, nb_l0, 0);
                    if (next_bundle >= pl.n_bundles) { queue_done = true; break; }
                    iss_item = pl.bundle_start[next_bundle];
                    iss_item_end = pl.bundle_start[next_bundle + 1];
                    if (lane == 0) nb_l0 = p.decode_workers + atomicAdd(&pl.queue[0], 1);  // consumed at the next bundle
                    have_prefetched = true;
                }
                if (f_tail - f_head >= FQ) break;
                const int4* src = reinterpret_cast<const int4*>(pl.items + iss_item);
                int4 a = __ldg(src), b = __ldg(src + 1);
                if (lane == 0) {
                    int4* dst = reinterpret_cast<int4*>(fifo + (f_tail % FQ));
                    dst[0] = a;
                    dst[1] = b;
                }
                ++f_tail;
                ++iss_item;
                iss_seq = a.x; iss_kvh = a.y; iss_blk = a.z; iss_blk_end = a.w;
                iss_open = true; iss_isV = false;
            }
            if (lane == 0) {
                if (!iss_isV) iss_blkid = __ldg(p.block_tables + (int64_t)iss_seq * p.max_blocks_per_seq + iss_blk);
                const uint32_t slot = u_iss % R;
                const uint32_t bar = bar_u32 + 8 * slot, dst = ring_u32 + slot * UNIT;
                mbar_expect_tx(bar, UNIT);
                const CUtensorMap* tm = iss_isV ? tmV : tmK;
#pragma unroll
                for (int qd = 0; qd < Cfg::kBoxes; ++qd) tma_load_4d(dst + qd * 2048, tm, bar, qd * 64, 0, iss_kvh, iss_blkid);
            }
            ++u_iss;
            if (iss_isV) {
                ++iss_blk;
                if (iss_blk == iss_blk_end) iss_open = false;
            }
            iss_isV = !iss_isV;
        }
        if (u_con == u_iss) {
            if (queue_done) break;
            continue;
        }

        // =============================== consume side: one tile per iteration
        const uint32_t slot = u_con % R, parity = (u_con / R) & 1u;
        const uint32_t tile = ring_u32 + slot * UNIT;
        if (!con_open) {
            __syncwarp();
            ci = fifo[f_head % FQ];
            con_blk = ci.blk_begin;
            con_isV = false;
            q_row = __ldg(p.cu_seqlens_q + ci.seq);
            h0 = ci.kv_head * G;
            const uint32_t* qp = reinterpret_cast<const uint32_t*>(p.q + ((int64_t)q_row * p.Hq + h0 + g) * D) + t;
#pragma unroll
            for (int ks = 0; ks < KS; ++ks) {
                qf[ks][0] = (g < G) ? __ldg(qp + ks * 8) : 0u;      // d = 16ks + 2t, +1
                qf[ks][1] = (g < G) ? __ldg(qp + ks * 8 + 4) : 0u;  // d = 16ks + 8 + 2t, +1
            }
            m0 = m1 = -INFINITY;
            l0 = l1 = 0.f;
#pragma unroll
            for (int i = 0; i < KS; ++i) o[i][0] = o[i][1] = o[i][2] = o[i][3] = 0.f;
            con_open = true;
        }
        mbar_wait(bar_u32 + 8 * slot, parity);

        if (!con_isV) {
            // ---- S^T[16 tok x 8 heads] = K[16 x D] · Q^T[D x 8]
            nvalid = min(16, ci.kv_len - con_blk * kBlock);
            float sa[4] = {0.f, 0.f, 0.f, 0.f}, sb[4] = {0.f, 0.f, 0.f, 0.f};
            const uint32_t mi = lane >> 3, r8 = lane & 7;
            const uint32_t row = r8 + 8 * (mi & 1);
#pragma unroll
            for (int ks = 0; ks < KS; ++ks) {
                const uint32_t chunk = 2 * ks + (mi >> 1);          // 16-byte chunk along d
                uint32_t a[4];
                ldmatrix_x4(a, tile + (chunk >> 3) * 2048 + swz128(row, chunk & 7));
                if (ks & 1) mma_bf16_16816(sb, a, qf[ks][0], qf[ks][1]);
                else        mma_bf16_16816(sa, a, qf[ks][0], qf[ks][1]);
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
            pb0 = movmatrix_trans(pack_bf16x2(p0, p1));
            pb1 = movmatrix_trans(pack_bf16x2(p2, p3));
            con_isV = true;
        } else {
            // ---- O^T[D x 8 heads] += V^T[D x 16 tok] · P^T[16 tok x 8]
            if (nvalid < 16) {   // last, partly filled block: unused V rows may hold anything (NaN): zero them
                const int nz = (16 - nvalid) * 8;                    // 16-byte chunks per 64-column box
#pragma unroll
                for (int qd = 0; qd < Cfg::kBoxes; ++qd)
                    for (int idx = lane; idx < nz; idx += 32)
                        asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(tile + qd * 2048 + nvalid * 128 + idx * 16), "r"(0u) : "memory");
                __syncwarp();
            }
            const uint32_t mi = lane >> 3, r8 = lane & 7;
            const uint32_t row = r8 + 8 * (mi >> 1);               // token
#pragma unroll
            for (int i = 0; i < KS; ++i) {
                const uint32_t chunk = 2 * i + (mi & 1);
                uint32_t a[4];
                ldmatrix_x4_trans(a, tile + (chunk >> 3) * 2048 + swz128(row, chunk & 7));
                mma_bf16_16816(o[i], a, pb0, pb1);
            }
            con_isV = false;
            ++con_blk;
            if (con_blk == ci.blk_end) {
                // ---------------- item finished
#pragma unroll
                for (int off = 4; off <= 16; off <<= 1) {
                    l0 += __shfl_xor_sync(0xffffffffu, l0, off);
                    l1 += __shfl_xor_sync(0xffffffffu, l1, off);
                }
                const int ha = 2 * t, hb = 2 * t + 1;
                if (ci.n_parts == 1) {
                    const float i0 = 1.f / l0, i1 = 1.f / l1;
                    __nv_bfloat16* oa = p.out + ((int64_t)q_row * p.Hq + h0 + ha) * D + g;
                    __nv_bfloat16* ob = oa + D;
#pragma unroll
                    for (int i = 0; i < KS; ++i) {
                        if (ha < G) { oa[16 * i] = __float2bfloat16_rn(o[i][0] * i0); oa[16 * i + 8] = __float2bfloat16_rn(o[i][2] * i0); }
                        if (hb < G) { ob[16 * i] = __float2bfloat16_rn(o[i][1] * i1); ob[16 * i + 8] = __float2bfloat16_rn(o[i][3] * i1); }
                    }
                } else {
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
                        // ---------------- a6 merge by the last-arriving worker
                        __threadfence();
                        constexpr int VPL = D / 32;                  // floats per lane
                        for (int hh = 0; hh < G; ++hh) {
                            float M = -INFINITY;
                            for (int i = 0; i < ci.n_parts; ++i)
                                M = fmaxf(M, __ldcg(&pl.part_ml[(ci.part_base + i) * kMaxGroup + hh]).x);
                            float L = 0.f, acc[VPL];
#pragma unroll
                            for (int k = 0; k < VPL; ++k) acc[k] = 0.f;
                            for (int i = 0; i < ci.n_parts; ++i) {
                                const float2 ml = __ldcg(&pl.part_ml[(ci.part_base + i) * kMaxGroup + hh]);
                                const float w = fast_exp2(ml.x - M);
                                L += ml.y * w;
                                const float4* src = reinterpret_cast<const float4*>(
                                    pl.part_o + ((int64_t)(ci.part_base + i) * G + hh) * D + lane * VPL);
#pragma unroll
                                for (int k = 0; k < VPL / 4; ++k) {
                                    const float4 v = __ldcg(src + k);
                                    acc[4 * k] += w * v.x; acc[4 * k + 1] += w * v.y;
                                    acc[4 * k + 2] += w * v.z; acc[4 * k + 3] += w * v.w;
                                }
                            }
                            const float inv = 1.f / L;
                            uint32_t packed[VPL / 2];
#pragma unroll
                            for (int k = 0; k < VPL / 2; ++k) packed[k] = pack_bf16x2(acc[2 * k] * inv, acc[2 * k + 1] * inv);
                            uint32_t* dst = reinterpret_cast<uint32_t*>(p.out + ((int64_t)q_row * p.Hq + h0 + hh) * D + lane * VPL);
                            if constexpr (VPL == 4) *reinterpret_cast<uint2*>(dst) = make_uint2(packed[0], packed[1]);
                            else *reinterpret_cast<uint4*>(dst) = make_uint4(packed[0], packed[1], packed[2], packed[3]);
                        }
                        if (lane == 0) *ctr = 0;                      // self-reset for the next launch
                    }
                }
                con_open = false;
                ++f_head;
            }
        }
        __syncwarp();   // every lane is done with this slot before lane 0 re-arms it
        ++u_con;
    }

}

}  // namespace pa
