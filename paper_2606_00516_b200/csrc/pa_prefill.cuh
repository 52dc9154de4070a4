// a4: prefill / chunked-prefill attention on the 5th-generation tensor cores (tcgen05 + TMEM), fed by TMA.
//
// "Prefill is compute-bound" (§1); a chunk of new tokens attends to the prompt's earlier
// KV (§2, L437 App. A.1): S = Q·K^T and O = P·V over a chunk are dense contractions, so this
// is the one part of the path that belongs on the tensor pipe (SURVEY §8(a) a4, §8(d) "Which roofline").
//
// Design.  One work unit = (128-row query tile of one chunk, KV head, group of NQ q heads
// that share that KV head).  The NQ q-head tiles of a unit stream the SAME K/V tiles (GQA: K/V are read
// once per KV head, not once per q head).  The keys are processed in steps of HT = 64; the scores of a
// q-head tile live in TWO TMEM buffers (step j in buffer j & 1), so the MMA issuer computes S(j+1) and S(j+2)
// while the softmax group still works on step j: neither side waits for the other in the steady state
// (with one buffer, S(j+1) cannot start before PV(j) has read the P that overlays S(j), and the chain
// S -> softmax -> PV -> S leaves the tensor pipe idle half of the time).
//   warp 9      unit hand-out + TMA producer: takes unit ids from the queue (one atomic per unit, requested a
//               unit ahead) and publishes them through a 4-slot mailbox; Q tiles once per unit; K and V tiles of
//               KT keys through a ring of kStages shared-memory stages (128B-swizzled boxes of one 16-token
//               block x 64 columns, addressed through the block table)
//   warps 10,11 MMA issuer of q-head tile 0 / 1 (one elected lane each): S_t(j) = Q_t·K(j)^T (SS, K-major x K-major, N = 64) into TMEM
//               buffer j & 1, O_t += P_t(j)·V(j) (P from TMEM [TS] or shared memory [SS], V MN-major); issue
//               order per step and tile: PV_t(j) S_t(j+2); the two issuers take strict turns on the tensor pipe
//   warp 8      TMEM allocation (512 columns: O_t at t·D, S_t buffer b at NQ·D + (2t+b)·64; P overlays S)
//   warps 0-3   softmax of tile 0, warps 4-7 softmax of tile 1: one query row per thread
//               (tcgen05.ld), causal mask (bottom-right aligned, DESIGN R3), online max with lazy
//               rescale of O (only when the running max grew by more than 2^8), exp2 with the scale
//               folded, P -> bf16, row sums in fp32; epilogue O/l -> bf16 -> global.
// All hand-offs are mbarriers (TMA complete_tx, tcgen05.commit, thread arrivals); the roles of a CTA run
// decoupled across units (the producer and the MMA issuers start the next unit while the softmax groups are in
// the epilogue of the current one).  Tensor-core-bound: algorithmic FLOPs = 4·D·Hq·Σ(q·ctx + q(q+1)/2).
#pragma once
#include "pa_common.cuh"
#include "pa_internal.h"
#include "pa_decode.cuh"
#include <type_traits>

namespace pa {

constexpr int kAttnThreads = 384;   // 12 warps: two softmax warpgroups + control warpgroup
// Warp roles of the prefill role.  The warp scheduler of an SM sub-partition favours the highest warp id among its
// eligible warps (B300_MICROARCH.md "Multi-warp arbiter"), so the warps every other warp waits for — the MMA
// issuers and the TMA producer — take the highest ids and the softmax groups the lowest.
constexpr int kWarpAlloc = 8, kWarpLoad = 9, kWarpMma0 = 10;     // MMA issuers: warps 10 (tile 0) and 11 (tile 1)
template <int D, bool kPinTmem>
struct PrefillCfg {
    static constexpr int NQ = (D == 128) ? 2 : 1;              // q-head tiles per unit
    static constexpr int KT = (D == 128) ? 128 : 64;           // keys per K/V ring stage (one TMA tile)
    static constexpr int HT = 64;                              // keys per MMA / softmax step
    static constexpr int HPT = KT / HT;                        // steps per ring stage
    static constexpr int kQBytes = kQTile * D * 2;             // one Q tile
    static constexpr int kStageBytes = KT * D * 2;             // one K (or V) tile = 32 KB
    static constexpr int kPBytes = kPinTmem ? 0 : kQTile * HT * 2;   // one P buffer (2 per q-head tile)
    static constexpr int kStages = kPinTmem ? 4 : (D == 128 ? 3 : 4);
    static constexpr int kOffQ = 0;
    static constexpr int kOffP = NQ * kQBytes;
    static constexpr int kOffRing = kOffP + NQ * 2 * kPBytes;
    // epilogue staging, 4 KB per softmax warp: its own area behind the ring, or (P in shared memory) the tile's P buffers,
    // which are idle once the last PV MMA of a unit has completed; a warp only ever touches its own 32 rows of either
    static constexpr int kOffStage = kPinTmem ? kOffRing + kStages * kStageBytes : kOffP;
    static constexpr int kStageStride = kPinTmem ? 4 * 4096 : 2 * kPBytes;
    static constexpr int kTileBytes = kOffRing + kStages * kStageBytes + (kPinTmem ? NQ * 4 * 4096 : 0);   // <= 224 KB
    static constexpr int kColO = 0;                             // TMEM columns
    static constexpr int kColS = NQ * D;
    static constexpr int kTmemCols = 512;
    static constexpr int kBlocksPerTile = KT / kBlock;
    static_assert(kTileBytes <= 224 * 1024, "prefill shared memory budget");
    static_assert(kColS + NQ * 2 * HT <= 512, "TMEM budget");
};

// control block (after the tile region): mbarriers + TMEM base + unit mailbox
struct PrefillCtrl {
    uint64_t q_full, q_empty;
    uint64_t kv_full[5], kv_empty[5];
    uint64_t s_full[2][2], p_full[2][2];    // [q-head tile][score buffer]
    uint64_t o_full[2], pv_done[2];
    uint64_t unit_full[4];
    uint64_t turn[2];       // the two MMA issuers take turns on the tensor pipe (prefill_role)
    uint32_t tmem_base;
    int32_t unit[4];        // mailbox: unit id ...
    int32_t pad_[3];
    PreTile tile[4];        // ... and its tile descriptor (fetched once, by the producer)
};
static_assert(sizeof(PrefillCtrl) <= 512, "PrefillCtrl size");

__device__ __forceinline__ void prefill_init_barriers(PrefillCtrl* c, int nq) {   // one thread, once per CTA; nq = q-head tiles per unit
    mbar_init(smem_u32(&c->q_full), 1);
    mbar_init(smem_u32(&c->q_empty), nq);            // one arrival per MMA issuer
    for (int i = 0; i < 5; ++i) { mbar_init(smem_u32(&c->kv_full[i]), 1); mbar_init(smem_u32(&c->kv_empty[i]), nq); }
    for (int t = 0; t < 2; ++t) {
        for (int b = 0; b < 2; ++b) {
            mbar_init(smem_u32(&c->s_full[t][b]), 1);
            mbar_init(smem_u32(&c->p_full[t][b]), 128);
        }
        mbar_init(smem_u32(&c->o_full[t]), 1);
        mbar_init(smem_u32(&c->pv_done[t]), 1);
    }
    for (int i = 0; i < 4; ++i) mbar_init(smem_u32(&c->unit_full[i]), 1);
    mbar_init(smem_u32(&c->turn[0]), 1);
    mbar_init(smem_u32(&c->turn[1]), 1);
    mbar_arrive(smem_u32(&c->turn[0]));       // tile 0 goes first
}

// exp2 of two finite floats on the FMA / integer pipes: x = n + f with n = round(x), f in [-0.5, 0.5];
// 2^f by a cubic (near-minimax, relative error 7.5e-5: below the bf16 rounding of P by a factor of 25), 2^n by adding
// n to the exponent field.  x is clamped at -126 (result 2^-126, which rounds P to ~1e-38: nothing in fp32 sums).
#ifndef PA_POLY_PAIRS
#define PA_POLY_PAIRS 3
#endif
constexpr int kPolyPairs = PA_POLY_PAIRS;       // of every 16 pairs of an unmasked softmax pass
__device__ __forceinline__ void exp2_poly_pair(float x0, float x1, float& p0, float& p1) {
    constexpr float kMagic = 12582912.f;        // 1.5 * 2^23: x + kMagic holds round(x) in its low mantissa bits
    x0 = fmaxf(x0, -126.f);
    x1 = fmaxf(x1, -126.f);
    const uint64_t x = pack_f2(x0, x1);
    const uint64_t t = fadd2(x, pack_f2(kMagic, kMagic));
    const uint64_t n = fadd2(t, pack_f2(-kMagic, -kMagic));
    const uint64_t f = ffma2(n, pack_f2(-1.f, -1.f), x);
    uint64_t p = ffma2(pack_f2(0.05517157167196274f, 0.05517157167196274f), f, pack_f2(0.2426111102104187f, 0.2426111102104187f));
    p = ffma2(p, f, pack_f2(0.6932610273361206f, 0.6932610273361206f));
    p = ffma2(p, f, pack_f2(0.9999280571937561f, 0.9999280571937561f));
    float q0, q1, t0, t1;
    unpack_f2(p, q0, q1);
    unpack_f2(t, t0, t1);
    p0 = __int_as_float(__float_as_int(q0) + (__float_as_int(t0) << 23));
    p1 = __int_as_float(__float_as_int(q1) + (__float_as_int(t1) << 23));
}

// what every role derives from a unit id
struct PrefillUnit {
    PreTile tile;
    int ti, kvh, h_first, nact, kv_total, n_kv, n_step;
};
// tile_src: null = fetch the tile descriptor from the plan (the producer), else the mailbox copy in shared memory
template <int NQ, int KT, int HT>
__device__ __forceinline__ PrefillUnit prefill_decode_unit(const AttnParams& p, int unit, const PreTile* tile_src = nullptr) {
    const PlanView& pl = p.plan;
    PrefillUnit u;
    const int per_tile = p.Hkv * pl.head_groups;
    u.ti = unit / per_tile;
    const int rem = unit - u.ti * per_tile;
    u.kvh = rem / pl.head_groups;
    const int hg = rem - u.kvh * pl.head_groups;
    u.tile = tile_src ? *tile_src : pl.tiles[u.ti];
    u.h_first = u.kvh * p.G + hg * NQ;
    u.nact = min(NQ, p.G - hg * NQ);                              // active q-head tiles of this unit
    u.kv_total = u.tile.ctx + u.tile.q_begin + u.tile.q_rows;     // keys any row of the tile can see
    u.n_kv = (u.kv_total + KT - 1) / KT;
    u.n_step = (u.kv_total + HT - 1) / HT;
    return u;
}

// The prefill role of one CTA.  `tiles` = 1024-byte aligned tile region; `first_unit` = statically assigned
// first unit, or -1 to take every unit from the queue (CTA that joins after finishing its decode role).
template <int D, bool kPinTmem>
__device__ void prefill_role(const AttnParams& p, const CUtensorMap* tmQ, const CUtensorMap* tmK, const CUtensorMap* tmV,
                             uint8_t* tiles, PrefillCtrl* ctrl, int first_unit) {
    using Cfg = PrefillCfg<D, kPinTmem>;
    constexpr int NQ = Cfg::NQ, KT = Cfg::KT, HT = Cfg::HT, HPT = Cfg::HPT, ST = Cfg::kStages;
    const int warp = (int)__reduce_max_sync(0xffffffffu, threadIdx.x >> 5), lane = lane_id();
    const PlanView& pl = p.plan;
    const uint32_t tiles_u32 = smem_u32(tiles);

    // ---- TMEM allocation (warp 2), published through shared memory
    if (warp == kWarpAlloc) {
        tmem_alloc(smem_u32(&ctrl->tmem_base), Cfg::kTmemCols);
        tmem_relinquish();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = ctrl->tmem_base;
    if (threadIdx.x == 0) PA_TL(15, 399, 2);
    // A role call starts with fresh barriers phases only the first time: the barriers persist across the two passes of
    // the kernel, but a CTA runs the prefill role at most once (pa_attention_kernel), so every phase starts at 0.

    if (warp == kWarpLoad) {
        // ======================================================== unit hand-out + TMA producer
        uint32_t ring = 0;          // K/V ring entries produced
        int unit = first_unit;
        if (unit < 0) {
            if (lane == 0) unit = p.prefill_ctas + atomicAdd(&pl.queue[2], 1);
            unit = __shfl_sync(0xffffffffu, unit, 0);
        }
        for (uint32_t it = 0;; ++it) {
            // the id of the next unit is requested now and read at the end of this unit's loads
            int unit_next = 0;
            if (lane == 0 && unit < pl.n_units) unit_next = p.prefill_ctas + atomicAdd(&pl.queue[2], 1);
            PrefillUnit u{};
            if (unit < pl.n_units) u = prefill_decode_unit<NQ, KT, HT>(p, unit);
            if (lane == 0) {
                ctrl->unit[it & 3] = unit;
                ctrl->tile[it & 3] = u.tile;
                mbar_arrive(smem_u32(&ctrl->unit_full[it & 3]));
            }
            __syncwarp();
            if (unit >= pl.n_units) break;
            const PreTile& tile = u.tile;
            if (lane == 0) {
                mbar_wait(smem_u32(&ctrl->q_empty), (it & 1u) ^ 1u);
                mbar_expect_tx(smem_u32(&ctrl->q_full), u.nact * Cfg::kQBytes);
                for (int t = 0; t < u.nact; ++t)
#pragma unroll
                    for (int c = 0; c < D / 64; ++c)
                        tma_load_3d(tiles_u32 + Cfg::kOffQ + t * Cfg::kQBytes + c * (kQTile * 128), tmQ, smem_u32(&ctrl->q_full),
                                    c * 64, u.h_first + t, tile.row0 + tile.q_begin);
            }
            // K/V tiles: every lane runs the same loop on warp-uniform values (lane-0 shuffles make that provable, so
            // the box addresses stay in the uniform datapath); lane b fetches the id of block b, the ids are broadcast
            // one by one and the elected lane issues the boxes.
            const uint32_t ring_base = tiles_u32 + Cfg::kOffRing;
            const int nkv_u = __reduce_max_sync(0xffffffffu, u.n_kv), kvt_u = __reduce_max_sync(0xffffffffu, u.kv_total);
            const int kvh_u = __reduce_max_sync(0xffffffffu, u.kvh);
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
            unit = __shfl_sync(0xffffffffu, unit_next, 0);
        }
    } else if (warp >= kWarpMma0 && warp - kWarpMma0 < NQ) {
        // ======================================================== MMA issuers: warp kWarpMma0 + t issues for q-head tile t
        // tcgen05.mma enters the tensor pipe through a queue only a few instructions deep: the issuing warp runs in
        // lock-step with the pipe, and whatever it does between two bursts (barrier waits, descriptor arithmetic) is
        // idle pipe time.  With one issuer per q-head tile the gaps of one warp are covered by the burst of the other.
        // Warp-uniform control flow; tcgen05.mma / tcgen05.commit are predicated on the elected lane.
        const int t = warp - kWarpMma0;
        constexpr uint32_t idescS = umma_idesc_bf16(128, HT, 0);
        constexpr uint32_t idescO = umma_idesc_bf16(128, D, 1);
        const uint32_t tm = __reduce_max_sync(0xffffffffu, tmem);
        const uint32_t sbase = tiles_u32;
        const uint32_t ocol = tm + Cfg::kColO + t * D;              // O_t
        const uint32_t scol0 = tm + Cfg::kColS + 2 * t * HT;        // score buffer 0 of tile t (buffer 1 follows)
        const uint64_t dq = umma_desc_sw128(sbase + Cfg::kOffQ + t * Cfg::kQBytes, 16, 1024);
        uint32_t ring0 = 0;                    // ring entries of the units before this one: K(i) = ring0 + 2i, V(i) = ring0 + 2i + 1
        uint32_t pph = 0;                      // p_full parity, bit b per score buffer
        [[maybe_unused]] int tl_step = 0;
        auto stage_wait = [&](uint32_t e) {
            mbar_wait(smem_u32(&ctrl->kv_full[e % ST]), (e / ST) & 1u);
            tc_fence_after();
        };
        // The tensor pipe interleaves the MMAs of two issuing warps one by one, so two bursts issued at the same time
        // both finish after the sum of their lengths, the two softmax groups get their scores together, compete for the
        // MUFU/FMA pipes together and hand back P together: everything waits for everything.  The issuers therefore
        // take strict turns, one burst (PV(j) + S(j+2)) per turn, through a pair of mbarriers (a sleeping wait, no
        // polling traffic): each group gets its scores after ONE burst length and the groups settle half a step apart.
        uint32_t turns = 0;                    // turns taken by this warp
        auto turn_take = [&](bool both) {
            if (NQ > 1 && both) mbar_wait(smem_u32(&ctrl->turn[t]), turns & 1u);
        };
        auto turn_pass = [&](bool both) {
            if (NQ > 1 && both) {
                __syncwarp();
                if (lane == 0) mbar_arrive(smem_u32(&ctrl->turn[t ^ 1]));
                ++turns;
            }
        };
        // S_t(js) = Q_t · K(js)^T into score buffer js & 1 (D/16 k-steps, N = HT keys), with the ring bookkeeping of the
        // K stage; an inactive tile (t >= nact) only takes part in the stage / Q hand-back
        auto step_S = [&](int js, bool active, int nstep_u) {
            const uint32_t e = ring0 + 2 * (uint32_t)(js / HPT);
            if (js % HPT == 0) stage_wait(e);
            if (elect_one()) {
                if (active) {
                    const uint64_t db0 = umma_desc_sw128(sbase + Cfg::kOffRing + (e % ST) * Cfg::kStageBytes + (js % HPT) * (HT * 128), 16, 1024);
#pragma unroll
                    for (int ks = 0; ks < D / 16; ++ks) {
                        const uint32_t oa = (uint32_t)(((ks >> 2) * (kQTile * 128) + (ks & 3) * 32) >> 4);
                        const uint32_t ob = (uint32_t)(((ks >> 2) * (KT * 128) + (ks & 3) * 32) >> 4);
                        umma_ss(scol0 + (js & 1) * HT, dq + oa, db0 + ob, idescS, ks > 0);
                    }
                    umma_commit(smem_u32(&ctrl->s_full[t][js & 1]));
                }
                if (js % HPT == HPT - 1 || js == nstep_u - 1) umma_commit(smem_u32(&ctrl->kv_empty[e % ST]));
                if (js == nstep_u - 1) umma_commit(smem_u32(&ctrl->q_empty));     // Q is read by the S MMAs only
            }
            __syncwarp();
        };
        for (uint32_t it = 0;; ++it) {
            mbar_wait(smem_u32(&ctrl->unit_full[it & 3]), (it >> 2) & 1u);
            const int unit = __reduce_max_sync(0xffffffffu, ctrl->unit[it & 3]);
            if (unit >= pl.n_units) break;
            const PrefillUnit u = prefill_decode_unit<NQ, KT, HT>(p, unit, &ctrl->tile[it & 3]);
            const int nstep_u = __reduce_max_sync(0xffffffffu, u.n_step), kvt_u = __reduce_max_sync(0xffffffffu, u.kv_total);
            const int kvl_u = __reduce_max_sync(0xffffffffu, u.tile.kv_len);
            const int nkv_u = __reduce_max_sync(0xffffffffu, u.n_kv);
            const int nact_u = (int)__reduce_max_sync(0xffffffffu, u.nact);
            const bool active = t < nact_u, both = nact_u == NQ;
            mbar_wait(smem_u32(&ctrl->q_full), it & 1u);
            tc_fence_after();
            for (int js = 0; js < min(2, nstep_u); ++js) step_S(js, active, nstep_u);
            int j = 0;
            if constexpr (HPT == 2) {
                // ---- steady state, one K/V tile (two steps) per iteration, everything but the ring position a
                // compile-time constant.  Covers the tiles whose PV steps are full (64 keys) and whose look-ahead S
                // steps are not the unit's last.
                const int n_fast = active ? max(0, (nstep_u - 3) / 2) : 0;      // tiles i with 2i + 3 <= nstep_u - 2
                uint32_t ek = ring0 + 2, ev = ring0 + 1;               // ring entries: K tile i + 1, V tile i
                uint32_t kst = ek % ST, kph = (ek / ST) & 1u, vst = ev % ST, vph = (ev / ST) & 1u;
                // Every wait sits BEHIND a burst of MMAs (its latency, ~100 cycles even when the barrier has long
                // completed, is covered by the backlog of the pipe), and the descriptors of the next ring stages are
                // computed at the end of an iteration, not between a wait and the MMAs that depend on it.
                auto desc_v = [&](uint32_t st) { return umma_desc_sw128(sbase + Cfg::kOffRing + st * Cfg::kStageBytes, KT * 128, 1024); };
                auto desc_k = [&](uint32_t st) { return umma_desc_sw128(sbase + Cfg::kOffRing + st * Cfg::kStageBytes, 16, 1024); };
                uint64_t dbv = desc_v(vst), dbk = desc_k(kst);
                uint64_t dp[2] = {0, 0};
                if constexpr (!kPinTmem) {
                    dp[0] = umma_desc_sw128(sbase + Cfg::kOffP + (2 * t) * Cfg::kPBytes, 16, 1024);
                    dp[1] = umma_desc_sw128(sbase + Cfg::kOffP + (2 * t + 1) * Cfg::kPBytes, 16, 1024);
                }
                auto pv_burst = [&](int hf, bool first) {
#pragma unroll
                    for (int ks = 0; ks < HT / kBlock; ++ks) {
                        const uint64_t db = dbv + (uint64_t)((hf * (HT / kBlock) + ks) * (2048 >> 4));
                        const uint32_t acc = (!first || ks > 0) ? 1u : 0u;
                        if constexpr (kPinTmem) umma_ts(ocol, scol0 + hf * HT + ks * 8, db, idescO, acc);
                        else umma_ss(ocol, dp[hf] + (uint64_t)((ks * 32) >> 4), db, idescO, acc);
                    }
                    umma_commit(smem_u32(&ctrl->pv_done[t]));
                };
                auto s_burst = [&](int hf) {
#pragma unroll
                    for (int ks = 0; ks < D / 16; ++ks) {
                        const uint32_t oa = (uint32_t)(((ks >> 2) * (kQTile * 128) + (ks & 3) * 32) >> 4);
                        const uint32_t ob = (uint32_t)(((ks >> 2) * (KT * 128) + (ks & 3) * 32 + hf * (HT * 128)) >> 4);
                        umma_ss(scol0 + hf * HT, dq + oa, dbk + ob, idescS, ks > 0);
                    }
                    umma_commit(smem_u32(&ctrl->s_full[t][hf]));
                };
                if (n_fast > 0) mbar_wait(smem_u32(&ctrl->kv_full[vst]), vph);       // V tile 0
                for (int i = 0; i < n_fast; ++i) {
                    // ---- step 2i: PV(2i), then S(2i + 2) on the first half of K tile i + 1
                    if (lane == 0) PA_TL(2 + t, tl_step, 0);
                    mbar_wait(smem_u32(&ctrl->p_full[t][0]), pph & 1u);
                    turn_take(both);
                    tc_fence_after();
                    if (lane == 0) PA_TL(2 + t, tl_step, 1);
                    if (elect_one()) pv_burst(0, i == 0);
                    __syncwarp();
                    mbar_wait(smem_u32(&ctrl->kv_full[kst]), kph);                   // K tile i + 1
                    tc_fence_after();
                    if (elect_one()) s_burst(0);
                    __syncwarp();
                    turn_pass(both);
                    if (lane == 0) PA_TL(2 + t, tl_step, 2);
                    // ---- step 2i + 1: PV(2i + 1), then S(2i + 3) on the second half of K tile i + 1
                    if (lane == 0) PA_TL(2 + t, tl_step + 1, 0);
                    mbar_wait(smem_u32(&ctrl->p_full[t][1]), (pph >> 1) & 1u);
                    turn_take(both);
                    tc_fence_after();
                    if (lane == 0) PA_TL(2 + t, tl_step + 1, 1);
                    if (elect_one()) {
                        pv_burst(1, false);
                        umma_commit(smem_u32(&ctrl->kv_empty[vst]));
                    }
                    __syncwarp();
                    vst += 2; if (vst >= ST) { vst -= ST; vph ^= 1u; }
                    mbar_wait(smem_u32(&ctrl->kv_full[vst]), vph);                   // V tile i + 1 (it exists: >= 3 steps follow)
                    tc_fence_after();
                    if (elect_one()) {
                        s_burst(1);
                        umma_commit(smem_u32(&ctrl->kv_empty[kst]));
                    }
                    __syncwarp();
                    turn_pass(both);
                    if (lane == 0) PA_TL(2 + t, tl_step + 1, 2);
#ifdef PA_TIMELINE
                    tl_step += 2;
#endif
                    pph ^= 0x3u;
                    kst += 2; if (kst >= ST) { kst -= ST; kph ^= 1u; }
                    dbv = desc_v(vst);
                    dbk = desc_k(kst);
                    asm volatile("" : "+l"(dbv), "+l"(dbk));                        // materialised here, behind the S burst
                }
                j = 2 * n_fast;
            } else {
                // ---- steady state for one-step K/V tiles (D = 256: KT = HT = 64): two steps per iteration so that the
                // score buffer is a compile-time constant; per step PV(j) on V tile j, then S(j + 2) on K tile j + 2.
                const int n_fast = active ? max(0, (nstep_u - 3) / 2) : 0;      // pairs (2i, 2i + 1) with 2i + 3 <= nstep_u - 2
                uint32_t ek = ring0 + 4, ev = ring0 + 1;               // ring entries: K tile j + 2, V tile j
                uint32_t kst = ek % ST, kph = (ek / ST) & 1u, vst = ev % ST, vph = (ev / ST) & 1u;
                auto desc_v = [&](uint32_t st) { return umma_desc_sw128(sbase + Cfg::kOffRing + st * Cfg::kStageBytes, KT * 128, 1024); };
                auto desc_k = [&](uint32_t st) { return umma_desc_sw128(sbase + Cfg::kOffRing + st * Cfg::kStageBytes, 16, 1024); };
                uint64_t dbv = desc_v(vst), dbk = desc_k(kst);
                uint64_t dp[2] = {0, 0};
                if constexpr (!kPinTmem) {
                    dp[0] = umma_desc_sw128(sbase + Cfg::kOffP + (2 * t) * Cfg::kPBytes, 16, 1024);
                    dp[1] = umma_desc_sw128(sbase + Cfg::kOffP + (2 * t + 1) * Cfg::kPBytes, 16, 1024);
                }
                if (n_fast > 0) mbar_wait(smem_u32(&ctrl->kv_full[vst]), vph);       // V tile 0
                for (int i = 0; i < n_fast; ++i) {
#pragma unroll
                    for (int b = 0; b < 2; ++b) {
                        mbar_wait(smem_u32(&ctrl->p_full[t][b]), (pph >> b) & 1u);
                        tc_fence_after();
                        if (elect_one()) {
#pragma unroll
                            for (int ks = 0; ks < HT / kBlock; ++ks) {
                                const uint64_t db = dbv + (uint64_t)(ks * (2048 >> 4));
                                const uint32_t acc = (i > 0 || b > 0 || ks > 0) ? 1u : 0u;
                                if constexpr (kPinTmem) umma_ts(ocol, scol0 + b * HT + ks * 8, db, idescO, acc);
                                else umma_ss(ocol, dp[b] + (uint64_t)((ks * 32) >> 4), db, idescO, acc);
                            }
                            umma_commit(smem_u32(&ctrl->pv_done[t]));
                            umma_commit(smem_u32(&ctrl->kv_empty[vst]));
                        }
                        __syncwarp();
                        mbar_wait(smem_u32(&ctrl->kv_full[kst]), kph);               // K tile j + 2
                        tc_fence_after();
                        if (elect_one()) {
#pragma unroll
                            for (int ks = 0; ks < D / 16; ++ks) {
                                const uint32_t oa = (uint32_t)(((ks >> 2) * (kQTile * 128) + (ks & 3) * 32) >> 4);
                                const uint32_t ob = (uint32_t)(((ks >> 2) * (KT * 128) + (ks & 3) * 32) >> 4);
                                umma_ss(scol0 + b * HT, dq + oa, dbk + ob, idescS, ks > 0);
                            }
                            umma_commit(smem_u32(&ctrl->s_full[t][b]));
                            umma_commit(smem_u32(&ctrl->kv_empty[kst]));
                        }
                        __syncwarp();
                        kst += 2; if (kst >= ST) { kst -= ST; kph ^= 1u; }
                        vst += 2; if (vst >= ST) { vst -= ST; vph ^= 1u; }
                        mbar_wait(smem_u32(&ctrl->kv_full[vst]), vph);               // V tile j + 1 (it exists: >= 3 steps follow)
                        dbv = desc_v(vst);
                        dbk = desc_k(kst);
                        asm volatile("" : "+l"(dbv), "+l"(dbk));
                    }
                    pph ^= 0x3u;
                }
                j = 2 * n_fast;
            }
            for (; j < nstep_u; ++j) {
                const int i = j / HPT, hf = j % HPT, b = j & 1;
                const uint32_t ev = ring0 + 2 * (uint32_t)i + 1;
                const uint32_t vb = sbase + Cfg::kOffRing + (ev % ST) * Cfg::kStageBytes;
                if (hf == 0) {
                    stage_wait(ev);
                    const int tkeys = min(KT, kvt_u - i * KT);
                    const int loaded = ((tkeys + kBlock - 1) / kBlock) * kBlock;   // rows the producer fetched
                    const int first_dead = kvl_u - i * KT;                          // rows >= this hold no token (R8)
                    if (active && first_dead < loaded) {
                        // zero them: masked P is exactly 0, but 0 x NaN (sentinel / garbage) would poison O.  Both
                        // issuers write the same zeros (a benign race) and each fences its own writes.
                        const int nrows = loaded - first_dead;
                        for (int idx = lane; idx < nrows * 8 * (D / 64); idx += 32) {
                            const int c = idx / (nrows * 8), rr = idx - c * (nrows * 8);
                            asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};"
                                         ::"r"(vb + c * (KT * 128) + first_dead * 128 + rr * 16), "r"(0u) : "memory");
                        }
                        fence_proxy_async();
                        __syncwarp();
                    }
                }
                const int keys = min(HT, kvt_u - j * HT);
                const int nks = (keys + kBlock - 1) / kBlock;            // PV k-steps = loaded blocks of this step
                if (active) {
                    if (lane == 0) PA_TL(2 + t, tl_step, 0);
                    mbar_wait(smem_u32(&ctrl->p_full[t][b]), (pph >> b) & 1u);
                    pph ^= 1u << b;
                    turn_take(both);
                    tc_fence_after();
                    if (lane == 0) PA_TL(2 + t, tl_step, 1);
                }
                if (elect_one()) {
                    if (active) {
                        const uint64_t db0 = umma_desc_sw128(vb, KT * 128, 1024) + (uint64_t)(hf * (HT / kBlock) * (2048 >> 4));
                        const uint32_t pcol = scol0 + b * HT;
                        const uint64_t da0 = kPinTmem ? 0ull : umma_desc_sw128(sbase + Cfg::kOffP + (2 * t + b) * Cfg::kPBytes, 16, 1024);
                        auto pv = [&](int ks) {
                            const uint32_t acc = (j > 0 || ks > 0) ? 1u : 0u;
                            if constexpr (kPinTmem) umma_ts(ocol, pcol + ks * 8, db0 + (uint64_t)(ks * (2048 >> 4)), idescO, acc);
                            else umma_ss(ocol, da0 + (uint64_t)((ks * 32) >> 4), db0 + (uint64_t)(ks * (2048 >> 4)), idescO, acc);
                        };
                        if (nks == HT / kBlock) {
#pragma unroll
                            for (int ks = 0; ks < HT / kBlock; ++ks) pv(ks);
                        } else {
                            for (int ks = 0; ks < nks; ++ks) pv(ks);
                        }
                        umma_commit(smem_u32(&ctrl->pv_done[t]));
                    }
                    if (hf == HPT - 1 || j == nstep_u - 1) umma_commit(smem_u32(&ctrl->kv_empty[ev % ST]));
                    if (active && j == nstep_u - 1) umma_commit(smem_u32(&ctrl->o_full[t]));
                }
                __syncwarp();
                if (j + 2 < nstep_u) step_S(j + 2, active, nstep_u);
                if (active) turn_pass(both);
                if (lane == 0) PA_TL(2 + t, tl_step, 2);
#ifdef PA_TIMELINE
                ++tl_step;
#endif
            }
            ring0 += 2 * (uint32_t)nkv_u;
        }
    } else if (warp < 8) {
        // ======================================================== softmax + correction + epilogue
        const int t = warp >> 2;
        const int row = ((warp & 3) << 5) + lane;               // TMEM lane == query row of the tile
        const uint32_t lane_addr = (uint32_t)((warp & 3) << 5) << 16;
        const uint32_t tO = tmem + lane_addr + Cfg::kColO + t * D;
        const float sl = p.scale_log2;
        const float NEG_INF = -INFINITY;
        uint32_t sph = 0;           // s_full parity, bit b per score buffer
        uint32_t oph = 0;           // o_full parity
        uint32_t pv_base = 0;       // PV commits of this tile before the current unit
        [[maybe_unused]] int tl_step = 0;
        [[maybe_unused]] const bool tl_me = (warp & 3) == 0 && lane == 0;
        for (uint32_t it = 0;; ++it) {
            mbar_wait(smem_u32(&ctrl->unit_full[it & 3]), (it >> 2) & 1u);
            const int unit = ctrl->unit[it & 3];
            if (unit >= pl.n_units) break;
            const PrefillUnit u = prefill_decode_unit<NQ, KT, HT>(p, unit, &ctrl->tile[it & 3]);
            if (t >= u.nact) continue;
            const PreTile& tile = u.tile;
            if (tl_me) PA_TL(12 + t, (int)it, 3);
            const int limit = tile.ctx + tile.q_begin + row;        // keys 0 .. limit are visible (R3)
            // m_ref: the reference max the exponentials of a step are taken against; m_run: max of all scores seen.
            // Only the first step needs its own max before exponentiating (two passes over S); later steps use the
            // reference left by their predecessors and fold the max into the same pass, so S is read from TMEM
            // once.  The reference is moved (l and the O row rescaled) at the start of a step, and only when the
            // running max outgrew it by more than 2^8; within a step P may therefore exceed 1 by the growth of
            // that one step, which floating point absorbs (P <= 2^64 is left alone; beyond it the row is fixed up
            // exactly, see below).
            float m_ref = NEG_INF, m_run = NEG_INF, l = 0.f;
            bool grew = false;
            // O_t may be touched only when every PV issued so far has completed.  PV(j-1) is the last one issued when
            // step j is being processed (PV(j) needs this step's P), and PV(j-2) has completed (s_full of step j was
            // committed behind it), so the commit count of pv_done is pv_base + j - 1 or pv_base + j: waiting for the
            // parity of phase pv_base + j - 1 is unambiguous.
            auto wait_pv = [&](int j) {
                if (j > 0) mbar_wait(smem_u32(&ctrl->pv_done[t]), (pv_base + (uint32_t)j - 1u) & 1u);
                tc_fence_after();
            };
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
            for (int j = 0; j < u.n_step; ++j) {
                const int b = j & 1;
                const uint32_t tS = tmem + lane_addr + Cfg::kColS + (2 * t + b) * HT;
                if (tl_me) PA_TL(t, tl_step, 0);
                mbar_wait(smem_u32(&ctrl->s_full[t][b]), (sph >> b) & 1u);
                sph ^= 1u << b;
                tc_fence_after();
                if (tl_me) PA_TL(t, tl_step, 1);
                if (lane == 0) PA_TL(4 + warp, tl_step, 1);
                const int kbase = j * HT;
                const bool need_mask = kbase + HT - 1 > tile.ctx + tile.q_begin;
                if (j == 0) {
                    // ---- first step: row maximum of the raw scores
                    float mx = NEG_INF;
                    const int rel0 = limit - kbase;
#pragma unroll
                    for (int c = 0; c < HT / 32; ++c) {
                        uint32_t r[32];
                        tmem_ld32(tS + c * 32, r);
                        tmem_wait_ld();
                        if (need_mask) {
#pragma unroll
                            for (int i = 0; i < 32; ++i)
                                mx = fmaxf(mx, (c * 32 + i <= rel0) ? __uint_as_float(r[i]) : NEG_INF);
                        } else {
#pragma unroll
                            for (int i = 0; i < 32; ++i) mx = fmaxf(mx, __uint_as_float(r[i]));
                        }
                    }
                    m_ref = m_run = mx;
                } else if (grew) {
                    // lazy correction of the O row and l
                    const float alpha = fast_exp2((m_ref - m_run) * sl);
                    l *= alpha;
                    m_ref = m_run;
                    wait_pv(j);
                    rescale_o(alpha);
                }
                const float neg = -m_ref * sl;
                // ---- P = exp2(s*sl - m_ref*sl) -> bf16 (TMEM over S, or swizzled shared memory) and the step max,
                // one pass, packed f32x2 math; the TMEM load of chunk c+1 is in flight while chunk c is processed.
                const uint64_t sl2 = pack_f2(sl, sl), neg2 = pack_f2(neg, neg);
                // four row-sum and two max accumulators: a lone in-order warp would otherwise wait out the latency of a
                // 32-deep dependent FADD2 / FMNMX3 chain
                uint64_t lsum4[4] = {pack_f2(0.f, 0.f), pack_f2(0.f, 0.f), pack_f2(0.f, 0.f), pack_f2(0.f, 0.f)};
                float mx2[2] = {NEG_INF, NEG_INF};
                // Two copies of the pass: only the steps that straddle the diagonal pay for the mask (as one predicated
                // pass the compare + select pair of every element ran on every step: a third of all instructions).
                const int rel = limit - kbase;          // columns 0 .. rel of this step are visible to this row
                auto pass = [&](auto masked) {
                    constexpr bool kMask = decltype(masked)::value;
                    uint32_t rbuf[2][32];
                    tmem_ld32(tS, rbuf[0]);
#pragma unroll
                    for (int c = 0; c < HT / 32; ++c) {
                        uint32_t (&r)[32] = rbuf[c & 1];
                        tmem_wait_ld();
                        if (lane == 0) PA_TL(4 + warp, tl_step, c == 0 ? 0 : 3);
                        if (c + 1 < HT / 32) tmem_ld32(tS + (c + 1) * 32, rbuf[(c + 1) & 1]);
                        uint32_t pk[16];
#pragma unroll
                        for (int i = 0; i < 32; i += 2) {
                            float s0 = __uint_as_float(r[i]), s1 = __uint_as_float(r[i + 1]);
                            if constexpr (kMask) {
                                if (c * 32 + i > rel) s0 = NEG_INF;
                                if (c * 32 + i + 1 > rel) s1 = NEG_INF;
                            }
                            mx2[(i >> 1) & 1] = fmaxf(mx2[(i >> 1) & 1], fmaxf(s0, s1));
                            const uint64_t x = ffma2(pack_f2(s0, s1), sl2, neg2);
                            float x0, x1, p0, p1;
                            unpack_f2(x, x0, x1);
                            if (!kMask && (((i >> 1) * kPolyPairs) % 16) < kPolyPairs) {     // folded at compile time (unrolled loop)
                                // exp2 on the FMA pipe for kPolyPairs of every 16 pairs: the MUFU unit (16 exp2 per clock and
                                // SM) would otherwise bound the pass; Cody-Waite split + cubic, relative error 7.5e-5
                                exp2_poly_pair(x0, x1, p0, p1);
                            } else {
                                p0 = fast_exp2(x0);
                                p1 = fast_exp2(x1);
                            }
                            lsum4[(i >> 1) & 3] = fadd2(lsum4[(i >> 1) & 3], pack_f2(p0, p1));
                            pk[i >> 1] = pack_bf16x2(p0, p1);
                        }
                        if constexpr (kPinTmem) {
                            tmem_st16(tS + c * 16, pk);
                        } else {
                            const uint32_t pbase = tiles_u32 + Cfg::kOffP + (2 * t + b) * Cfg::kPBytes;
#pragma unroll
                            for (int q4 = 0; q4 < 4; ++q4) {
                                const uint32_t cc = c * 4 + q4;             // 16-byte chunk (8 keys) of the row
                                asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};"
                                             ::"r"(pbase + swz128(row, cc)),
                                               "r"(pk[q4 * 4]), "r"(pk[q4 * 4 + 1]), "r"(pk[q4 * 4 + 2]), "r"(pk[q4 * 4 + 3])
                                             : "memory");
                            }
                        }
                    }
                };
                if (need_mask) pass(std::true_type{});
                else pass(std::false_type{});
                const float mx = fmaxf(mx2[0], mx2[1]);
                {
                    float la, lb;
                    unpack_f2(fadd2(fadd2(lsum4[0], lsum4[1]), fadd2(lsum4[2], lsum4[3])), la, lb);
                    l += la + lb;
                }
                m_run = fmaxf(m_run, mx);
                // one vote per step: did any row's running max outgrow its reference by more than 2^8?  (the next step then
                // moves the reference; a step that outgrew it by more than 2^64 is a subset and fixed up right here)
                grew = __any_sync(0xffffffffu, (m_run - m_ref) * sl > 8.f);
                if (grew && j > 0 && __any_sync(0xffffffffu, (mx - m_ref) * sl > 64.f)) {
                    // rare: this step outgrew the reference by more than 2^64.  Its P (finite up to 2^127) is scaled
                    // down by the exact power of two alpha, together with l and the O row, and the reference moves.
                    const bool mine = (mx - m_ref) * sl > 64.f;
                    const float alpha = mine ? fast_exp2(floorf((m_ref - mx) * sl)) : 1.f;
                    if (mine) m_ref += -floorf((m_ref - mx) * sl) / sl;
                    l *= alpha;
                    if constexpr (kPinTmem) {
                        tmem_wait_st();
                        uint32_t r[32];
                        tmem_ld32(tS, r);
                        tmem_wait_ld();
#pragma unroll
                        for (int i = 0; i < 32; ++i)
                            r[i] = pack_bf16x2(__uint_as_float(r[i] << 16) * alpha, __uint_as_float(r[i] & 0xffff0000u) * alpha);
                        tmem_st32(tS, r);
                    } else {
                        const uint32_t pbase = tiles_u32 + Cfg::kOffP + (2 * t + b) * Cfg::kPBytes;
                        for (int cc = 0; cc < HT / 8; ++cc) {
                            const uint32_t addr = pbase + swz128(row, cc);
                            uint32_t v[4];
                            asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]) : "r"(addr) : "memory");
#pragma unroll
                            for (int i = 0; i < 4; ++i)
                                v[i] = pack_bf16x2(__uint_as_float(v[i] << 16) * alpha, __uint_as_float(v[i] & 0xffff0000u) * alpha);
                            asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]) : "memory");
                        }
                    }
                    wait_pv(j);
                    rescale_o(alpha);
                    grew = __any_sync(0xffffffffu, (m_run - m_ref) * sl > 8.f);
                }
                if (tl_me) PA_TL(t, tl_step, 2);
                if (lane == 0) PA_TL(4 + warp, tl_step, 2);
                if constexpr (kPinTmem) tmem_wait_st();
                else fence_proxy_async();
                tc_fence_before();
                mbar_arrive(smem_u32(&ctrl->p_full[t][b]));
                if (tl_me) PA_TL(t, tl_step, 3);
#ifdef PA_TIMELINE
                ++tl_step;
#endif
            }
            pv_base += (uint32_t)u.n_step;
            // ---- epilogue: O / l -> bf16 -> out[row0 + q_begin + row][h][:]
            if (tl_me) PA_TL(12 + t, (int)it, 0);
            mbar_wait(smem_u32(&ctrl->o_full[t]), oph);
            oph ^= 1u;
            tc_fence_after();
            if (tl_me) PA_TL(12 + t, (int)it, 1);
            const float inv = 1.f / l;
            bool valid = row < tile.q_rows;
            if (valid && !(l <= 3.0e38f)) {
                // the one-pass softmax overflowed (a step outgrew everything before it by > 2^127): hand the row
                // to the plain loop that the last CTA of the launch runs (include/pa.h, "Range")
                pl.redo[atomicAdd(&pl.queue[3], 1)] = make_int2(u.ti, (row << 8) | (u.h_first + t));
                __threadfence();
                valid = false;
            }
            // A thread owns a row, and rows are Hq·D·2 bytes apart in `out`: stored straight from the registers, every
            // 16-byte store of a warp would touch 32 different lines (32 L1 wavefronts per instruction, ~2.7 us per
            // unit).  The warp's 32 rows x 64 columns go through a 4 KB staging area (16-byte pieces XOR-swizzled by
            // row) and leave as whole 128-byte lines, four rows per instruction.
            const uint32_t stg = tiles_u32 + Cfg::kOffStage + t * Cfg::kStageStride + (uint32_t)(warp & 3) * 4096u;
            const uint32_t vmask = __ballot_sync(0xffffffffu, valid);
            __nv_bfloat16* out0 = p.out + ((int64_t)(tile.row0 + tile.q_begin + ((warp & 3) << 5)) * p.Hq + u.h_first + t) * D;
#pragma unroll
            for (int hh = 0; hh < D / 64; ++hh) {
                uint32_t r[2][32];
                tmem_ld32(tO + hh * 64, r[0]);
                tmem_ld32(tO + hh * 64 + 32, r[1]);
                tmem_wait_ld();
                if (tl_me && hh == 0) PA_TL(14 + t, (int)it, 0);
#pragma unroll
                for (int pc = 0; pc < 8; ++pc) {
                    const uint32_t* x = &r[pc >> 2][(pc & 3) * 8];
                    uint4 v;
                    v.x = pack_bf16x2(__uint_as_float(x[0]) * inv, __uint_as_float(x[1]) * inv);
                    v.y = pack_bf16x2(__uint_as_float(x[2]) * inv, __uint_as_float(x[3]) * inv);
                    v.z = pack_bf16x2(__uint_as_float(x[4]) * inv, __uint_as_float(x[5]) * inv);
                    v.w = pack_bf16x2(__uint_as_float(x[6]) * inv, __uint_as_float(x[7]) * inv);
                    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(stg + (uint32_t)(lane * 128 + ((pc ^ (lane & 7)) << 4))),
                                 "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
                }
                __syncwarp();
                if (tl_me && hh == 0) PA_TL(14 + t, (int)it, 1);
                uint4 w[8];
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int rr = 4 * i + (lane >> 3), pc = lane & 7;
                    // volatile (ordered behind the stores and the warp barrier) but no memory clobber: the eight loads and
                    // the global stores that consume them are scheduled freely
                    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(w[i].x), "=r"(w[i].y), "=r"(w[i].z), "=r"(w[i].w)
                                 : "r"(stg + (uint32_t)(rr * 128 + ((pc ^ (rr & 7)) << 4))));
                }
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const int rr = 4 * i + (lane >> 3), pc = lane & 7;
                    if ((vmask >> rr) & 1u)
                        *reinterpret_cast<uint4*>(out0 + (int64_t)rr * p.Hq * D + hh * 64 + pc * 8) = w[i];
                }
                __syncwarp();
                if (tl_me && hh == 0) PA_TL(14 + t, (int)it, 2);
            }
            tc_fence_before();
            if (tl_me) PA_TL(12 + t, (int)it, 2);
        }
    }

    // ---- teardown: every tcgen05 op of this CTA has completed (the softmax groups waited on o_full)
    tc_fence_before();
    __syncthreads();
    if (warp == kWarpAlloc) tmem_dealloc(tmem, Cfg::kTmemCols);
}

}  // namespace pa
