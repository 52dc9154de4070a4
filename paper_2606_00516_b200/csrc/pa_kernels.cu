// Kernels of libpa_b200.so (sm_100a) and their launch wrappers.
#include "pa_launch.h"
#include "pa_common.cuh"
#include "pa_decode.cuh"
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
// a5/a6 decode launch: persistent, one CTA per SM, kDecodeWarps independent workers per CTA.
// ------------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(kDecodeWarps * 32, 1)
pa_decode_kernel(const AttnParams p, const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* base = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    const int warp = threadIdx.x >> 5;
    uint8_t* ring = base + warp * DecodeCfg<D>::kRingBytes;
    uint8_t* aux = base + kDecodeWarps * DecodeCfg<D>::kRingBytes + warp * DecodeCfg<D>::kAuxBytes;
    if (threadIdx.x == 0) {
        tma_prefetch_desc(&tmK);
        tma_prefetch_desc(&tmV);
    }
    // interleave so that the first gridDim.x bundles land on distinct SMs
    const int worker_id = warp * gridDim.x + blockIdx.x;
    decode_worker<D>(p, &tmK, &tmV, ring, aux, worker_id);
}

int decode_smem_bytes(int D) { return D == 128 ? DecodeCfg<128>::kSmemBytes : DecodeCfg<256>::kSmemBytes; }

cudaError_t configure_kernels() {
    cudaError_t e;
    e = cudaFuncSetAttribute(pa_decode_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, DecodeCfg<128>::kSmemBytes);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(pa_decode_kernel<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, DecodeCfg<256>::kSmemBytes);
    return e;
}

cudaError_t launch_attention(const AttnLaunch& a, cudaStream_t stream, int* launches_out) {
    AttnParams p;
    p.q = reinterpret_cast<const __nv_bfloat16*>(a.q);
    p.out = reinterpret_cast<__nv_bfloat16*>(a.out);
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
    p.decode_cta_begin = 0;
    int launches = 0;
    cudaError_t e = cudaSuccess;
    if (a.decode_ctas > 0 && a.plan.n_bundles > 0) {
        dim3 grid(a.decode_ctas), block(kDecodeWarps * 32);
        if (a.sh.D == 128)
            pa_decode_kernel<128><<<grid, block, DecodeCfg<128>::kSmemBytes, stream>>>(p, *a.tmK, *a.tmV);
        else
            pa_decode_kernel<256><<<grid, block, DecodeCfg<256>::kSmemBytes, stream>>>(p, *a.tmK, *a.tmV);
        ++launches;
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    if (a.n_simple_tiles > 0) {
        dim3 grid(a.n_simple_tiles, a.sh.Hq), block(128);
        if (a.sh.D == 128)
            pa_simple_kernel<128><<<grid, block, 0, stream>>>(p, (const __nv_bfloat16*)a.k_pool, (const __nv_bfloat16*)a.v_pool);
        else
            pa_simple_kernel<256><<<grid, block, 0, stream>>>(p, (const __nv_bfloat16*)a.k_pool, (const __nv_bfloat16*)a.v_pool);
        ++launches;
        e = cudaGetLastError();
    }
    if (launches_out) *launches_out = launches;
    return e;
}

}  // namespace pa
