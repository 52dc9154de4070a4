// Kernels of libpa_b200.so (sm_100a) and their launch wrappers.
#include "pa_launch.h"
#include "pa_common.cuh"
#include "pa_decode.cuh"
#include "pa_prefill.cuh"
#include "pa_simple.cuh"

namespace pa {

// ------------------------------------------------------------------------------------------------
// a3 kv_append: one warp per new token; 16-byte vector copies of the token's K and V rows into
// slot(s, ctx_s + j) = (block_tables[s][(ctx_s+j)/16], (ctx_s+j)%16) of pool[block][kv head][slot][d].
// HBM-bound: 2·n_tok·kvb algorithmic bytes (read new + write pool), SURVEY §8(a) a3.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int find_seq_warp(const int32_t* __restrict__ cu, int n_seq, int row) {
    // decode-first batches: cu[s] == s for the decode prefix -> one probe
    if (row < n_seq) {
        int a = __ldg(cu + row), b = __ldg(cu + row + 1);
        if (a == row && b == row + 1) return row;
    }
    int lo = 0, hi = n_seq;  // largest s in [lo, hi) with cu[s] <= row
    const int lane = lane_id();
    while (hi - lo > 1) {
        const int step = (hi - lo + 31) >> 5;
        const int idx = lo + lane * step;
        const bool pred = (idx < hi) && (__ldg(cu + idx) <= row);
        const int k = __popc(__ballot_sync(0xffffffffu, pred));
        const int nlo = lo + (k - 1) * step;
        hi = min(hi, nlo + step);
        lo = nlo;
    }
    return lo;
}

template <int D>
__global__ void __launch_bounds__(256) pa_kv_append_kernel(const int4* __restrict__ k_new, const int4* __restrict__ v_new,
                                                           int4* __restrict__ k_pool, int4* __restrict__ v_pool,
                                                           const int32_t* __restrict__ cu, const int32_t* __restrict__ ctx,
                                                           const int32_t* __restrict__ bt, int max_blocks_per_seq,
                                                           int Hkv, int n_seq, int n_tok) {
    constexpr int CPH = D / 8;  // 16-byte chunks per head row
    // the attention launch that follows on the stream may bring its CTAs up (barrier init, descriptor prefetch)
    // while the rows are copied; it reads the pool only after its grid-dependency wait
    pdl_launch_dependents();
    const int row = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (row >= n_tok) return;
    const int lane = lane_id();
    const int s = find_seq_warp(cu, n_seq, row);
    const int t = __ldg(ctx + s) + (row - __ldg(cu + s));
    const int64_t blk = __ldg(bt + (int64_t)s * max_blocks_per_seq + t / kBlock);
    const int within = t % kBlock;
    const int total = Hkv * CPH;
    for (int c = lane; c < total; c += 32) {
        const int g = c / CPH, cc = c % CPH;
        const int64_t src = ((int64_t)row * Hkv + g) * CPH + cc;
        const int64_t dst = ((blk * Hkv + g) * kBlock + within) * CPH + cc;
        const int4 kv = __ldg(k_new + src), vv = __ldg(v_new + src);
        k_pool[dst] = kv;
        v_pool[dst] = vv;
    }
}

template <int D>
__global__ void __launch_bounds__(256) pa_kv_gather_kernel(const int4* __restrict__ k_pool, const int4* __restrict__ v_pool,
                                                           const int32_t* __restrict__ table_row, int Hkv, int kv_len,
                                                           int4* __restrict__ k_out, int4* __restrict__ v_out) {
    constexpr int CPH = D / 8;
    const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (t >= kv_len) return;
    const int lane = lane_id();
    const int64_t blk = __ldg(table_row + t / kBlock);
    const int within = t % kBlock;
    const int total = Hkv * CPH;
    for (int c = lane; c < total; c += 32) {
        const int g = c / CPH, cc = c % CPH;
        const int64_t src = ((blk * Hkv + g) * kBlock + within) * CPH + cc;
        const int64_t dst = ((int64_t)t * Hkv + g) * CPH + cc;
        k_out[dst] = __ldg(k_pool + src);
        v_out[dst] = __ldg(v_pool + src);
    }
}

cudaError_t launch_kv_append(const LaunchShape& sh, const void* k_new, const void* v_new, void* k_pool, void* v_pool,
                             const int32_t* cu, const int32_t* ctx, const int32_t* bt, int32_t n_seq, int32_t n_tok,
                             cudaStream_t stream) {
    // launched normally: measured on B200, launching kv_append itself with programmatic stream serialization (its
    // CTAs queued under the previous attention launch) made the step 4 us SLOWER
    const int warps = 8;
    dim3 grid((n_tok + warps - 1) / warps), block(warps * 32);
    if (sh.D == 128)
        pa_kv_append_kernel<128><<<grid, block, 0, stream>>>((const int4*)k_new, (const int4*)v_new, (int4*)k_pool,
                                                             (int4*)v_pool, cu, ctx, bt, sh.max_blocks_per_seq, sh.Hkv,
                                                             n_seq, n_tok);
    else
        pa_kv_append_kernel<256><<<grid, block, 0, stream>>>((const int4*)k_new, (const int4*)v_new, (int4*)k_pool,
                                                             (int4*)v_pool, cu, ctx, bt, sh.max_blocks_per_seq, sh.Hkv,
                                                             n_seq, n_tok);
    return cudaGetLastError();
}

cudaError_t launch_kv_gather(const LaunchShape& sh, const void* k_pool, const void* v_pool, const int32_t* table_row,
                             int32_t kv_len, void* k_out, void* v_out, cudaStream_t stream) {
    const int warps = 8;
    dim3 grid((kv_len + warps - 1) / warps), block(warps * 32);
    if (sh.D == 128)
        pa_kv_gather_kernel<128><<<grid, block, 0, stream>>>((const int4*)k_pool, (const int4*)v_pool, table_row, sh.Hkv,
                                                             kv_len, (int4*)k_out, (int4*)v_out);
    else
        pa_kv_gather_kernel<256><<<grid, block, 0, stream>>>((const int4*)k_pool, (const int4*)v_pool, table_row, sh.Hkv,
                                                             kv_len, (int4*)k_out, (int4*)v_out);
    return cudaGetLastError();
}


// ------------------------------------------------------------------------------------------------
// a7 mixed single launch: one persistent CTA per SM, 12 warps.  CTAs [0, prefill_ctas) start in the
// prefill role (tcgen05/TMEM), the rest in the decode role (8 TMA + mma.sync workers); when a CTA's
// own queue runs dry it switches to the other role, so neither the tensor pipe nor HBM idles while
// work remains.  The last CTA to leave resets the queues for the next launch.
// Shared memory (from a 1024-byte aligned base): [0, 224 KB) tile region shared by the two roles,
// then the prefill control block (512 B), then the decode workers' scratch (8 x 192 B).
// ------------------------------------------------------------------------------------------------
constexpr int kTileRegion = 224 * 1024;
constexpr int kCtrlBytes = 512;
constexpr int kAttnSmemBytes = 1024 + kTileRegion + kCtrlBytes + kDecodeWarps * 192;
static_assert(kAttnSmemBytes <= 232448, "attention kernel shared memory");
static_assert(kDecodeWarps * DecodeCfg<128>::kStreamBytes <= kTileRegion, "decode streams fit the tile region");
static_assert(kDecodeWarps * DecodeCfg<256>::kStreamBytes <= kTileRegion, "decode streams fit the tile region");

template <int D, bool kPinTmem>
__global__ void __launch_bounds__(kAttnThreads, 1)
pa_attention_kernel(const AttnParams p, const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmQd,
                    const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                    const __grid_constant__ TailMaps tails) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* tiles = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    PrefillCtrl* ctrl = reinterpret_cast<PrefillCtrl*>(tiles + kTileRegion);
    uint8_t* dec_aux = tiles + kTileRegion + kCtrlBytes;
    const PlanView& pl = p.plan;
    if (threadIdx.x == 0) { PA_TL(15, 399, 0); PA_TL_CTA(0); }
    // set-up spread over threads (it is on the critical path of microsecond-scale launches): thread 0 the prefill
    // barriers, threads 32.. one decode stream each, thread 64 the descriptor prefetches
    if (threadIdx.x == 0 && pl.n_units > 0) prefill_init_barriers(ctrl, PrefillCfg<D, kPinTmem>::NQ);
    if (threadIdx.x >= 32 && threadIdx.x < 32 + kDecodeWarps && pl.n_bundles > 0)
        decode_init_barriers<D>(dec_aux, (int)threadIdx.x - 32);
    if (threadIdx.x == 64) {
        tma_prefetch_desc(&tmK);
        tma_prefetch_desc(&tmV);
        if (pl.n_units > 0) tma_prefetch_desc(&tmQ);
        if (pl.n_bundles > 0) {
            tma_prefetch_desc(&tmQd);
            tma_prefetch_desc(&tails.k[0]);
            tma_prefetch_desc(&tails.v[0]);
        }
    }
    if (threadIdx.x < 64) {
        fence_mbar_init();
        fence_proxy_async();
    }
    __syncthreads();
    // everything above touches only this CTA's shared memory and the kernel parameters; the pools, the plan and the
    // queues are read below, after the preceding kernel of the stream (normally kv_append) has completed
    pdl_grid_dependency_wait();
    if (threadIdx.x == 0) PA_TL(15, 399, 1);
    const bool starts_prefill = (int)blockIdx.x < p.prefill_ctas;
    const int dec_rank = (int)blockIdx.x - p.prefill_ctas;       // rank among the initial decode CTAs
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
        const bool do_prefill = (pass == 0) == starts_prefill;
        if (do_prefill) {
            // late joiners only if units beyond the statically assigned ones exist
            if (pl.n_units > 0 && (starts_prefill || pl.n_units > p.prefill_ctas))
                prefill_role<D, kPinTmem>(p, &tmQ, &tmK, &tmV, tiles, ctrl, starts_prefill ? (int)blockIdx.x : -1);
        } else {
            if (pl.n_bundles > 0 && (!starts_prefill || pl.n_bundles * pl.n_levels > p.decode_workers))
                decode_role<D>(p, &tmQd, &tmK, &tmV, &tails, tiles, dec_aux, starts_prefill ? -1 : dec_rank);
        }
        __syncthreads();
        if (threadIdx.x == 0) { PA_TL(15, 397 + pass, 0); PA_TL_CTA(1 + pass); }
    }
    // The last CTA to leave resets the queues for the next launch and recomputes, with the plain row loop, the prefill
    // rows whose one-pass softmax overflowed (normally none).  Pattern: writers fence before the counting atomic,
    // the last arriver fences after it.
    int* last_flag = reinterpret_cast<int*>(&ctrl->unit[0]);
    if (threadIdx.x == 0) {
        __threadfence();
        *last_flag = atomicAdd(&pl.queue[1], 1) == (int)gridDim.x - 1;
    }
    __syncthreads();
    if (*last_flag) {
        __threadfence();
        const int n_redo = *reinterpret_cast<volatile int*>(&pl.queue[3]);
        for (int i = threadIdx.x >> 5; i < n_redo; i += kAttnThreads / 32) {
            const int2 e = __ldcg(pl.redo + i);
            const PreTile t = pl.tiles[e.x];
            const int j = t.q_begin + (e.y >> 8);
            simple_row<D>(p, t.seq, t.ctx, j, (int64_t)t.row0 + j, e.y & 0xff, lane_id());
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            pl.queue[0] = 0;
            pl.queue[1] = 0;
            pl.queue[2] = 0;
            pl.queue[3] = 0;
            pl.queue[4] += n_redo;      // cumulative since pa_plan: rows recomputed by the plain loop (introspection)
            __threadfence();
        }
    }
}

int attention_smem_bytes() { return kAttnSmemBytes; }

template <int D, bool T>
static cudaError_t set_attr() {
    return cudaFuncSetAttribute(pa_attention_kernel<D, T>, cudaFuncAttributeMaxDynamicSharedMemorySize, kAttnSmemBytes);
}

cudaError_t configure_kernels() {
    cudaError_t e = set_attr<128, true>();
    if (e == cudaSuccess) e = set_attr<128, false>();
    if (e == cudaSuccess) e = set_attr<256, true>();
    if (e == cudaSuccess) e = set_attr<256, false>();
    return e;
}

cudaError_t launch_attention(const AttnLaunch& a, cudaStream_t stream, int* launches_out) {
    AttnParams p;
    p.q = reinterpret_cast<const __nv_bfloat16*>(a.q);
    p.out = reinterpret_cast<__nv_bfloat16*>(a.out);
    p.k_pool = reinterpret_cast<const __nv_bfloat16*>(a.k_pool);
    p.v_pool = reinterpret_cast<const __nv_bfloat16*>(a.v_pool);
    p.cu_seqlens_q = a.cu_seqlens_q;
    p.context_lens = a.context_lens;
    p.block_tables = a.block_tables;
    p.max_blocks_per_seq = a.sh.max_blocks_per_seq;
    p.Hq = a.sh.Hq;
    p.Hkv = a.sh.Hkv;
    p.G = a.sh.Hq / a.sh.Hkv;
    p.scale_log2 = a.softmax_scale * 1.4426950408889634f;
    p.plan = a.plan;
    p.decode_workers = a.decode_ctas * kDecodeWarps;
    p.prefill_ctas = a.prefill_ctas;
    int launches = 0;
    cudaError_t e = cudaSuccess;
    const int grid_ctas = a.decode_ctas + a.prefill_ctas;
    if (grid_ctas > 0) {
        dim3 grid(grid_ctas), block(kAttnThreads);
        const CUtensorMap& tq = a.tmQ ? *a.tmQ : *a.tmK;    // unused when there are no prefill units
        const CUtensorMap& tqd = a.tmQd ? *a.tmQd : *a.tmK;  // unused when there are no decode bundles
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = grid;
        cfg.blockDim = block;
        cfg.dynamicSmemBytes = kAttnSmemBytes;
        cfg.stream = stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // see pdl_grid_dependency_wait in the kernel
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        if (a.sh.D == 128) {
            if (a.p_in_tmem) e = cudaLaunchKernelEx(&cfg, pa_attention_kernel<128, true>, p, tq, tqd, *a.tmK, *a.tmV, *a.tails);
            else e = cudaLaunchKernelEx(&cfg, pa_attention_kernel<128, false>, p, tq, tqd, *a.tmK, *a.tmV, *a.tails);
        } else {
            if (a.p_in_tmem) e = cudaLaunchKernelEx(&cfg, pa_attention_kernel<256, true>, p, tq, tqd, *a.tmK, *a.tmV, *a.tails);
            else e = cudaLaunchKernelEx(&cfg, pa_attention_kernel<256, false>, p, tq, tqd, *a.tmK, *a.tmV, *a.tails);
        }
        if (e != cudaSuccess) return e;
        ++launches;
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    if (a.n_simple_tiles > 0) {
        dim3 grid(a.n_simple_tiles, a.sh.Hq), block(128);
        if (a.sh.D == 128)
            pa_simple_kernel<128><<<grid, block, 0, stream>>>(p);
        else
            pa_simple_kernel<256><<<grid, block, 0, stream>>>(p);
        ++launches;
        e = cudaGetLastError();
    }
    if (launches_out) *launches_out = launches;
    return e;
}

}  // namespace pa
