// a4: prefill / chunked-prefill attention on the 5th-generation tensor cores (tcgen05 + TMEM), fed by TMA.
//
// "Prefill is compute-bound" (§1); a chunk of new tokens attends to the prompt's earlier
// KV (§2, L437 App. A.1): S = Q·K^T and O = P·V over a chunk are dense contractions, so this
// is the one part of the path that belongs on the tensor pipe (SURVEY §8(a) a4, §8(d) "Which roofline").
//
// Design.  One work unit = (128-row query tile of one chunk, KV head, group of NQ q heads
// that share that KV head).  The NQ q-head tiles of a unit stream the SAME K/V tiles (GQA: K/V are read
// once per KV head, not once per q head) and ping-pong on the tensor pipe, so the softmax of one tile
// overlaps the MMAs of the other:
//   warp 0      TMA producer: Q tiles once per unit; K and V tiles of KT keys through a ring of kStages
//               shared-memory stages (128B-swizzled boxes of one 16-token block x 64 columns, addressed
//               through the block table; lane b issues the boxes of block b)
//   warp 1      MMA issuer (one elected lane): S_t = Q_t·K^T (SS, K-major x K-major) into TMEM, then
//               O_t += P_t·V (P from TMEM [TS] or shared memory [SS], V MN-major), order
//               PV_0(j) S_0(j+1) PV_1(j) S_1(j+1) so each softmax group has two MMAs of cover
//   warp 2      TMEM allocation (512 columns: O_t at t·D, S_t at NQ·D + t·KT; P_t overlays S_t)
//   warps 4-7   softmax of tile 0, warps 8-11 softmax of tile 1: one query row per thread
//               (tcgen05.ld), causal mask (bottom-right aligned, DESIGN R3), online max with lazy
//               rescale of O (only when the running max grew by more than 2^8), exp2 with the scale
//               folded, P -> bf16, row sums in fp32; epilogue O/l -> bf16 -> global.
// All hand-offs are mbarriers (TMA complete_tx, tcgen05.commit, thread arrivals); no __syncthreads in
// the steady state.  Tensor-core-bound: algorithmic FLOPs = 4·D·Hq·Σ(q·ctx + q(q+1)/2).
#pragma once
#include "pa_common.cuh"
#include "pa_internal.h"
#include "pa_decode.cuh"

namespace pa {

constexpr int kAttnThreads = 384;   // 12 warps: control warpgroup + two softmax warpgroups
template <int D, bool kPinTmem>
struct PrefillCfg {
    static constexpr int NQ = (D == 128) ? 2 : 1;              // q-head tiles per unit
    static constexpr int KT = (D == 128) ? 128 : 64;           // keys per KV tile
    static constexpr int kQBytes = kQTile * D * 2;             // one Q tile
    static constexpr int kStageBytes = KT * D * 2;             // one K (or V) tile = 32 KB
    static constexpr int kPBytes = kPinTmem ? 0 : kQTile * KT * 2;
    static constexpr int kStages = kPinTmem ? 5 : (D == 128 ? 3 : 4);
    static constexpr int kOffQ = 0;
    static constexpr int kOffP = NQ * kQBytes;
    static constexpr int kOffRing = kOffP + NQ * kPBytes;
    static constexpr int kTileBytes = kOffRing + kStages * kStageBytes;   // <= 224 KB
    static constexpr int kColO = 0;                             // TMEM columns
    static constexpr int kColS = NQ * D;
    static constexpr int kTmemCols = 512;
    static constexpr int kBlocksPerTile = KT / kBlock;
    static_assert(kTileBytes <= 224 * 1024, "prefill shared memory budget");
    static_assert(kColS + NQ * KT <= 512, "TMEM budget");
};

// control block (after the tile region): mbarriers + TMEM base + unit mailbox
struct PrefillCtrl {
    uint64_t q_full, q_empty;
    uint64_t kv_full[5], kv_empty[5];
    uint64_t s_full[2], p_full[2], o_full[2];
    uint32_t tmem_base;
    int32_t unit[2];
};
static_assert(sizeof(PrefillCtrl) <= 256, "PrefillCtrl size");

__device__ __forceinline__ void prefill_init_barriers(PrefillCtrl* c) {   // one thread, once per CTA
    mbar_init(smem_u32(&c->q_full), 1);
    mbar_init(smem_u32(&c->q_empty), 1);
    for (int i = 0; i < 5; ++i) { mbar_init(smem_u32(&c->kv_full[i]), 1); mbar_init(smem_u32(&c->kv_empty[i]), 1); }
    for (int t = 0; t < 2; ++t) {
        mbar_init(smem_u32(&c->s_full[t]), 1);
        mbar_init(smem_u32(&c->p_full[t]), 128);
        mbar_init(smem_u32(&c->o_full[t]), 1);
    }
}

// The prefill role of one CTA.  `tiles` = 1024-byte aligned tile region; `first_unit` = statically assigned
// first unit, or -1 to take every unit from the queue (CTA that joins after finishing its decode role).
template <int D, bool kPinTmem>
__device__ void prefill_role(const AttnParams& p, const CUtensorMap* tmQ, const CUtensorMap* tmK, const CUtensorMap* tmV,
                             uint8_t* tiles, PrefillCtrl* ctrl, int first_unit) {
    using Cfg = PrefillCfg<D, kPinTmem>;
    constexpr int NQ = Cfg::NQ, KT = Cfg::KT, ST = Cfg::kStages;
    const int warp = (int)__reduce_max_sync(0xffffffffu, threadIdx.x >> 5), lane = lane_id();
    const PlanView& pl = p.plan;
    const uint32_t tiles_u32 = smem_u32(tiles);

    // ---- TMEM allocation (warp 2), published through shared memory
    if (warp == 2) {
        tmem_alloc(smem_u32(&ctrl->tmem_base), Cfg::kTmemCols);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = ctrl->tmem_base;

    // pipeline state that persists across units (each role advances its own copy identically)
    uint32_t ring = 0;          // K/V ring entries produced (warp 0) / consumed (warp 1)
    uint32_t n_unit = 0;        // units processed (parity of q_full / q_empty)
    uint32_t sph = 0, oph = 0;  // softmax groups: s_full / o_full parity
    uint32_t pph0 = 0, pph1 = 0;  // MMA warp: p_full parity per tile

    int unit = first_unit;
    for (uint32_t it = 0;; ++it) {
        // ---------------- unit hand-out: one atomic per unit, broadcast through a 2-slot mailbox
        if (threadIdx.x == 0) {
            int u = unit;
            if (it > 0 || u < 0) u = p.prefill_ctas + atomicAdd(&pl.queue[2], 1);
            ctrl->unit[it & 1] = u;
        }
        __syncthreads();
        unit = __reduce_max_sync(0xffffffffu, ctrl->unit[it & 1]);   // the same for all threads; a warp reduction lands in a uniform register, so the compiler knows it
        if (unit >= pl.n_units) break;

        const int per_tile = p.Hkv * pl.head_groups;
        const int ti = unit / per_tile, rem = unit - ti * per_tile;
        const int kvh = rem / pl.head_groups, hg = rem - kvh * pl.head_groups;
        const PreTile tile = pl.tiles[ti];
        const int h_first = kvh * p.G + hg * NQ;
        const int nact = min(NQ, p.G - hg * NQ);                     // active q-head tiles of this unit
        const int kv_total = tile.ctx + tile.q_begin + tile.q_rows;  // keys any row of the tile can see
        const int n_kv = (kv_total + KT - 1) / KT;

        if (warp == 0) {
            // ======================================================== TMA producer
            if (lane == 0) {
                mbar_wait(smem_u32(&ctrl->q_empty), (n_unit & 1u) ^ 1u);
                mbar_expect_tx(smem_u32(&ctrl->q_full), nact * Cfg::kQBytes);
                for (int t = 0; t < nact; ++t)
#pragma unroll
                    for (int c = 0; c < D / 64; ++c)
                        tma_load_3d(tiles_u32 + Cfg::kOffQ + t * Cfg::kQBytes + c * (kQTile * 128), tmQ, smem_u32(&ctrl->q_full),
                                    c * 64, h_first + t, tile.row0 + tile.q_begin);
            }
            // K/V tiles: every lane runs the same loop on warp-uniform values (lane-0 shuffles make that provable, so
            // the box addresses stay in the uniform datapath); lane b fetches the id of block b, the ids are broadcast
            // one by one and the elected lane issues the boxes.
            const uint32_t ring_base = tiles_u32 + Cfg::kOffRing;
            const int nkv_u = __reduce_max_sync(0xffffffffu, n_kv), kvt_u = __reduce_max_sync(0xffffffffu, kv_total);
            const int kvh_u = __reduce_max_sync(0xffffffffu, kvh);
            const int32_t* bt = p.block_tables + (int64_t)tile.seq * p.max_blocks_per_seq;
            for (int j = 0; j < nkv_u; ++j) {
                const int keys = min(KT, kvt_u - j * KT);
                const int nb = (keys + kBlock - 1) / kBlock;
                const int blk = (lane < nb) ? __ldg(bt + j * Cfg::kBlocksPerTile + lane) : 0;
                int ids[Cfg::kBlocksPerTile];
#pragma unroll
                for (int bb = 0; bb < Cfg::kBlocksPerTile; ++bb) ids[bb] = __shfl_sync(0xffffffffu, blk, bb);
#pragma unroll
                for (int isV = 0; isV < 2; ++isV) {
                    const uint32_t stage = ring % ST, ph = (ring / ST) & 1u;
                    const uint32_t full = smem_u32(&ctrl->kv_full[stage]);
                    mbar_wait(smem_u32(&ctrl->kv_empty[stage]), ph ^ 1u);
                    if (elect_one()) {
                        mbar_expect_tx(full, nb * (kBlock * D * 2));
                        const uint32_t dst = ring_base + stage * Cfg::kStageBytes;
#pragma unroll
                        for (int bb = 0; bb < Cfg::kBlocksPerTile; ++bb) {
                            if (bb < nb) {
#pragma unroll
                                for (int c = 0; c < D / 64; ++c)
                                    tma_load_4d(dst + bb * 2048 + c * (KT * 128), isV ? tmV : tmK, full, c * 64, 0, kvh_u, ids[bb]);
                            }
                        }
                    }
                    __syncwarp();
                    ++ring;
                }
            }
        } else if (warp == 1) {
            // ======================================================== MMA issuer
            // Warp-uniform control flow; tcgen05.mma / tcgen05.commit are predicated on the elected lane and their
            // descriptors advance by compile-time constants, so issuing an MMA costs a few uniform instructions
            // (the issue rate of this one warp bounds the tensor pipe: 32 MMAs per KV tile).
            constexpr uint32_t idescS = umma_idesc_bf16(128, KT, 0);
            constexpr uint32_t idescO = umma_idesc_bf16(128, D, 1);
            const uint32_t tm = __reduce_max_sync(0xffffffffu, tmem);
            const uint32_t sbase = tiles_u32;
            const int nkv_u = __reduce_max_sync(0xffffffffu, n_kv), kvt_u = __reduce_max_sync(0xffffffffu, kv_total);
            const int kvl_u = __reduce_max_sync(0xffffffffu, tile.kv_len), nact_u = __reduce_max_sync(0xffffffffu, nact);
            auto issue_S = [&](int t, uint32_t kstage) {      // S_t = Q_t · K^T   (D/16 k-steps)
                if (elect_one()) {
                    const uint64_t da0 = umma_desc_sw128(sbase + Cfg::kOffQ + t * Cfg::kQBytes, 16, 1024);
                    const uint64_t db0 = umma_desc_sw128(sbase + Cfg::kOffRing + kstage * Cfg::kStageBytes, 16, 1024);
#pragma unroll
                    for (int ks = 0; ks < D / 16; ++ks) {
                        const uint32_t oa = (uint32_t)(((ks >> 2) * (kQTile * 128) + (ks & 3) * 32) >> 4);
                        const uint32_t ob = (uint32_t)(((ks >> 2) * (KT * 128) + (ks & 3) * 32) >> 4);
                        umma_ss(tm + Cfg::kColS + t * KT, da0 + oa, db0 + ob, idescS, ks > 0);
                    }
                    umma_commit(smem_u32(&ctrl->s_full[t]));
                }
                __syncwarp();
            };
            auto issue_PV = [&](int t, uint32_t vb, int ks, uint32_t acc) {   // O_t += P_t[:, 16 ks..] · V[16 ks.., :]
                const uint64_t db = umma_desc_sw128(vb, KT * 128, 1024) + (uint64_t)(ks * (2048 >> 4));
                if constexpr (kPinTmem) {
                    umma_ts(tm + Cfg::kColO + t * D, tm + Cfg::kColS + t * KT + ks * 8, db, idescO, acc);
                } else {
                    const uint64_t da = umma_desc_sw128(sbase + Cfg::kOffP + t * Cfg::kPBytes, 16, 1024) +
                                        (uint64_t)(((ks >> 2) * (kQTile * 128) + (ks & 3) * 32) >> 4);
                    umma_ss(tm + Cfg::kColO + t * D, da, db, idescO, acc);
                }
            };
            mbar_wait(smem_u32(&ctrl->q_full), n_unit & 1u);
            {   // S(0)
                const uint32_t stage = ring % ST, ph = (ring / ST) & 1u;
                mbar_wait(smem_u32(&ctrl->kv_full[stage]), ph);
                tc_fence_after();
                for (int t = 0; t < nact_u; ++t) issue_S(t, stage);
                umma_commit_p(smem_u32(&ctrl->kv_empty[stage]));
                ++ring;
            }
            for (int j = 0; j < nkv_u; ++j) {
                const uint32_t sv = ring % ST, phv = (ring / ST) & 1u;
                ++ring;
                mbar_wait(smem_u32(&ctrl->kv_full[sv]), phv);
                const int keys = min(KT, kvt_u - j * KT);
                const int nks = (keys + kBlock - 1) / kBlock;            // PV k-steps = loaded blocks
                const uint32_t vb = sbase + Cfg::kOffRing + sv * Cfg::kStageBytes;
                const int first_dead = kvl_u - j * KT;                   // rows >= this hold no token (R8)
                if (first_dead < nks * kBlock) {
                    // zero them: masked P is exactly 0, but 0 x NaN (sentinel / garbage) would poison O
                    const int nrows = nks * kBlock - first_dead;
                    for (int idx = lane; idx < nrows * 8 * (D / 64); idx += 32) {
                        const int c = idx / (nrows * 8), rr = idx - c * (nrows * 8);
                        asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};"
                                     ::"r"(vb + c * (KT * 128) + first_dead * 128 + rr * 16), "r"(0u) : "memory");
                    }
                    fence_proxy_async();
                    __syncwarp();
                }
                uint32_t sk = 0;
                for (int t = 0; t < nact_u; ++t) {
                    mbar_wait(smem_u32(&ctrl->p_full[t]), t == 0 ? pph0 : pph1);
                    tc_fence_after();
                    if (elect_one()) {
                        if (nks == KT / kBlock) {
#pragma unroll
                            for (int ks = 0; ks < KT / kBlock; ++ks) issue_PV(t, vb, ks, (j > 0 || ks > 0) ? 1u : 0u);
                        } else {
                            for (int ks = 0; ks < nks; ++ks) issue_PV(t, vb, ks, (j > 0 || ks > 0) ? 1u : 0u);
                        }
                        if (t == nact_u - 1) umma_commit(smem_u32(&ctrl->kv_empty[sv]));
                        if (j == nkv_u - 1) umma_commit(smem_u32(&ctrl->o_full[t]));
                    }
                    __syncwarp();
                    if (j + 1 < nkv_u) {
                        if (t == 0) {
                            sk = ring % ST;
                            const uint32_t phk = (ring / ST) & 1u;
                            ++ring;
                            mbar_wait(smem_u32(&ctrl->kv_full[sk]), phk);
                            tc_fence_after();
                        }
                        issue_S(t, sk);
                        if (t == nact_u - 1) umma_commit_p(smem_u32(&ctrl->kv_empty[sk]));
                    }
                }
                pph0 ^= 1u;
                if (nact_u > 1) pph1 ^= 1u;
            }
            umma_commit_p(smem_u32(&ctrl->q_empty));
        } else if (warp >= 4) {
            // ======================================================== softmax + correction + epilogue
            const int t = (warp - 4) >> 2;
            if (t < nact) {
                const int row = ((warp & 3) << 5) + lane;               // TMEM lane == query row of the tile
                const uint32_t lane_addr = (uint32_t)((warp & 3) << 5) << 16;
                const uint32_t tS = tmem + lane_addr + Cfg::kColS + t * KT;
                const uint32_t tO = tmem + lane_addr + Cfg::kColO + t * D;
                const int limit = tile.ctx + tile.q_begin + row;        // keys 0 .. limit are visible (R3)
                const float sl = p.scale_log2;
                const float NEG_INF = -INFINITY;
                // m_ref: the reference max the exponentials of a tile are taken against; m_run: max of all scores seen.
                // Only the first tile needs its own max before exponentiating (two passes over S); later tiles use the
                // reference left by their predecessors and fold the max into the same pass, so S is read from TMEM
                // once.  The reference is moved (l and the O row rescaled) at the start of a tile, and only when the
                // running max outgrew it by more than 2^8; within a tile P may therefore exceed 1 by the growth of
                // that one tile, which floating point absorbs (P <= 2^64 is left alone; beyond it the row is fixed up
                // exactly, see below).
                float m_ref = NEG_INF, m_run = NEG_INF, l = 0.f;
                for (int j = 0; j < n_kv; ++j) {
                    mbar_wait(smem_u32(&ctrl->s_full[t]), sph);
                    sph ^= 1u;
                    tc_fence_after();
                    const int kbase = j * KT;
                    const bool need_mask = kbase + KT - 1 > tile.ctx + tile.q_begin;
                    auto rescale_o = [&](float alpha) {
#pragma unroll
                        for (int c = 0; c < D / 32; ++c) {
                            uint32_t r[32];
                            tmem_ld32(tO + c * 32, r);
                            tmem_wait_ld();
#pragma unroll
                            for (int i = 0; i < 32; ++i) r[i] = __float_as_uint(__uint_as_float(r[i]) * alpha);
                            tmem_st32(tO + c * 32, r);
                        }
                        tmem_wait_st();
                    };
                    if (j == 0) {
                        // ---- first tile: row maximum of the raw scores
                        float mx = NEG_INF;
#pragma unroll
                        for (int c = 0; c < KT / 32; ++c) {
                            uint32_t r[32];
                            tmem_ld32(tS + c * 32, r);
                            tmem_wait_ld();
                            if (need_mask) {
#pragma unroll
                                for (int i = 0; i < 32; ++i)
                                    mx = fmaxf(mx, (kbase + c * 32 + i <= limit) ? __uint_as_float(r[i]) : NEG_INF);
                            } else {
#pragma unroll
                                for (int i = 0; i < 32; ++i) mx = fmaxf(mx, __uint_as_float(r[i]));
                            }
                        }
                        m_ref = m_run = mx;
                    } else if (__any_sync(0xffffffffu, (m_run - m_ref) * sl > 8.f)) {
                        // lazy correction: O holds the tiles before this one (their PV MMAs completed before s_full)
                        const float alpha = fast_exp2((m_ref - m_run) * sl);
                        l *= alpha;
                        m_ref = m_run;
                        rescale_o(alpha);
                    }
                    const float neg = -m_ref * sl;
                    // ---- P = exp2(s*sl - m_ref*sl) -> bf16 (TMEM over S, or swizzled shared memory) and the tile max,
                    // one pass, packed f32x2 math; the TMEM load of chunk c+1 is in flight while chunk c is processed.
                    const uint64_t sl2 = pack_f2(sl, sl), neg2 = pack_f2(neg, neg);
                    uint64_t lsum = pack_f2(0.f, 0.f);
                    float mx = NEG_INF;
                    uint32_t rbuf[2][32];
                    tmem_ld32(tS, rbuf[0]);
#pragma unroll
                    for (int c = 0; c < KT / 32; ++c) {
                        uint32_t (&r)[32] = rbuf[c & 1];
                        tmem_wait_ld();
                        if (c + 1 < KT / 32) tmem_ld32(tS + (c + 1) * 32, rbuf[(c + 1) & 1]);
                        uint32_t pk[16];
#pragma unroll
                        for (int i = 0; i < 32; i += 2) {
                            float s0 = __uint_as_float(r[i]), s1 = __uint_as_float(r[i + 1]);
                            if (need_mask) {
                                if (kbase + c * 32 + i > limit) s0 = NEG_INF;
                                if (kbase + c * 32 + i + 1 > limit) s1 = NEG_INF;
                            }
                            mx = fmaxf(mx, fmaxf(s0, s1));
                            const uint64_t x = ffma2(pack_f2(s0, s1), sl2, neg2);
                            float x0, x1, p0, p1;
                            unpack_f2(x, x0, x1);
                            p0 = fast_exp2(x0);
                            p1 = fast_exp2(x1);
                            lsum = fadd2(lsum, pack_f2(p0, p1));
                            pk[i >> 1] = pack_bf16x2(p0, p1);
                        }
                        if constexpr (kPinTmem) {
                            tmem_st16(tS + c * 16, pk);
                        } else {
                            const uint32_t pbase = tiles_u32 + Cfg::kOffP + t * Cfg::kPBytes;
#pragma unroll
                            for (int q4 = 0; q4 < 4; ++q4) {
                                const uint32_t cc = c * 4 + q4;             // 16-byte chunk (8 keys) of the row
                                asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};"
                                             ::"r"(pbase + (cc >> 3) * (kQTile * 128) + swz128(row, cc & 7)),
                                               "r"(pk[q4 * 4]), "r"(pk[q4 * 4 + 1]), "r"(pk[q4 * 4 + 2]), "r"(pk[q4 * 4 + 3])
                                             : "memory");
                            }
                        }
                    }
                    {
                        float la, lb;
                        unpack_f2(lsum, la, lb);
                        l += la + lb;
                    }
                    m_run = fmaxf(m_run, mx);
                    if (j > 0 && __any_sync(0xffffffffu, (mx - m_ref) * sl > 64.f)) {
                        // rare: this tile outgrew the reference by more than 2^64.  Its P (finite up to 2^127) is scaled
                        // down by the exact power of two alpha, together with l and the O row, and the reference moves.
                        const bool mine = (mx - m_ref) * sl > 64.f;
                        const float alpha = mine ? fast_exp2(floorf((m_ref - mx) * sl)) : 1.f;
                        if (mine) m_ref += -floorf((m_ref - mx) * sl) / sl;
                        l *= alpha;
                        if constexpr (kPinTmem) {
                            tmem_wait_st();
#pragma unroll
                            for (int c = 0; c < KT / 64; ++c) {
                                uint32_t r[32];
                                tmem_ld32(tS + c * 32, r);
                                tmem_wait_ld();
#pragma unroll
                                for (int i = 0; i < 32; ++i)
                                    r[i] = pack_bf16x2(__uint_as_float(r[i] << 16) * alpha, __uint_as_float(r[i] & 0xffff0000u) * alpha);
                                tmem_st32(tS + c * 32, r);
                            }
                        } else {
                            const uint32_t pbase = tiles_u32 + Cfg::kOffP + t * Cfg::kPBytes;
                            for (int cc = 0; cc < KT / 8; ++cc) {
                                const uint32_t addr = pbase + (cc >> 3) * (kQTile * 128) + swz128(row, cc & 7);
                                uint32_t v[4];
                                asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]) : "r"(addr) : "memory");
#pragma unroll
                                for (int i = 0; i < 4; ++i)
                                    v[i] = pack_bf16x2(__uint_as_float(v[i] << 16) * alpha, __uint_as_float(v[i] & 0xffff0000u) * alpha);
                                asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]) : "memory");
                            }
                        }
                        rescale_o(alpha);
                    }
                    if constexpr (kPinTmem) tmem_wait_st();
                    else fence_proxy_async();
                    tc_fence_before();
                    mbar_arrive(smem_u32(&ctrl->p_full[t]));
                }
                // ---- epilogue: O / l -> bf16 -> out[row0 + q_begin + row][h][:]
                mbar_wait(smem_u32(&ctrl->o_full[t]), oph);
                oph ^= 1u;
                tc_fence_after();
                const float inv = 1.f / l;
                bool valid = row < tile.q_rows;
                if (valid && !(l <= 3.0e38f)) {
                    // the one-pass softmax overflowed (a tile outgrew everything before it by > 2^127): hand the row
                    // to the plain loop that the last CTA of the launch runs (include/pa.h, "Range")
                    pl.redo[atomicAdd(&pl.queue[3], 1)] = make_int2(ti, (row << 8) | (h_first + t));
                    __threadfence();
                    valid = false;
                }
                uint4* dst = reinterpret_cast<uint4*>(p.out + ((int64_t)(tile.row0 + tile.q_begin + row) * p.Hq + h_first + t) * D);
#pragma unroll
                for (int c = 0; c < D / 32; ++c) {
                    uint32_t r[32];
                    tmem_ld32(tO + c * 32, r);
                    tmem_wait_ld();
                    if (valid) {
#pragma unroll
                        for (int q4 = 0; q4 < 4; ++q4) {
                            uint4 v;
                            v.x = pack_bf16x2(__uint_as_float(r[q4 * 8 + 0]) * inv, __uint_as_float(r[q4 * 8 + 1]) * inv);
                            v.y = pack_bf16x2(__uint_as_float(r[q4 * 8 + 2]) * inv, __uint_as_float(r[q4 * 8 + 3]) * inv);
                            v.z = pack_bf16x2(__uint_as_float(r[q4 * 8 + 4]) * inv, __uint_as_float(r[q4 * 8 + 5]) * inv);
                            v.w = pack_bf16x2(__uint_as_float(r[q4 * 8 + 6]) * inv, __uint_as_float(r[q4 * 8 + 7]) * inv);
                            dst[c * 4 + q4] = v;
                        }
                    }
                }
                tc_fence_before();
            }
        }
        ++n_unit;
    }

    // ---- teardown: every tcgen05 op of this CTA has completed (the softmax groups waited on o_full)
    tc_fence_before();
    __syncthreads();
    if (warp == 2) tmem_dealloc(tmem, Cfg::kTmemCols);
}

}  // namespace pa
