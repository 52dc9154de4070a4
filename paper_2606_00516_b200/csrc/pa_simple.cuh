// Plain one-warp-per-(query row, q head) paged attention: an online-softmax loop over the keys with an exact
// rescale at every step, correct for every row type (decode, prefill chunk over prior context) and for any finite
// scores.  Used (i) by the debug kernel behind PA_FLAG_DEBUG_SIMPLE (the v0 of the prefill path)
// and (ii) inside pa_attention_kernel to recompute the rare prefill rows whose one-pass tensor-core softmax
// overflowed (include/pa.h, pa_batch_attention "Range").  The production paths are pa_decode.cuh / pa_prefill.cuh.
#pragma once
#include "pa_common.cuh"
#include "pa_internal.h"
#include "pa_decode.cuh"

namespace pa {

// one warp: query j of sequence `seq` (packed row `row`, ctx cached tokens), q head h
template <int D>
__device__ __forceinline__ void simple_row(const AttnParams& p, int seq, int ctx, int j, int64_t row, int h, int lane) {
    constexpr int EPL = D / 32;  // elements per lane
    const int kvh = h / p.G;
    const int32_t* bt = p.block_tables + (int64_t)seq * p.max_blocks_per_seq;
    const int n_keys = ctx + j + 1;
    float qv[EPL], acc[EPL];
    const __nv_bfloat16* qp = p.q + (row * p.Hq + h) * D + lane * EPL;
#pragma unroll
    for (int e = 0; e < EPL; ++e) { qv[e] = __bfloat162float(qp[e]); acc[e] = 0.f; }
    float m = -INFINITY, l = 0.f;
    for (int t = 0; t < n_keys; ++t) {
        const int64_t blk = __ldg(bt + t / kBlock);
        const int64_t off = ((blk * p.Hkv + kvh) * kBlock + (t % kBlock)) * D + lane * EPL;
        float dot = 0.f;
#pragma unroll
        for (int e = 0; e < EPL; ++e) dot += qv[e] * __bfloat162float(p.k_pool[off + e]);
#pragma unroll
        for (int s = 16; s >= 1; s >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, s);
        const float z = dot * p.scale_log2;
        const float mn = fmaxf(m, z);
        const float c = exp2f(m - mn), w = exp2f(z - mn);
        l = l * c + w;
#pragma unroll
        for (int e = 0; e < EPL; ++e) acc[e] = acc[e] * c + w * __bfloat162float(p.v_pool[off + e]);
        m = mn;
    }
    __nv_bfloat16* op = p.out + (row * p.Hq + h) * D + lane * EPL;
    const float inv = 1.f / l;
#pragma unroll
    for (int e = 0; e < EPL; ++e) op[e] = __float2bfloat16_rn(acc[e] * inv);
}

template <int D>
__global__ void __launch_bounds__(128) pa_simple_kernel(AttnParams p) {
    const PreTile tile = p.plan.tiles[blockIdx.x];
    const int warp = threadIdx.x >> 5, lane = lane_id();
    for (int jj = warp; jj < tile.q_rows; jj += 4)
        simple_row<D>(p, tile.seq, tile.ctx, tile.q_begin + jj, (int64_t)tile.row0 + tile.q_begin + jj, blockIdx.y, lane);
}

}  // namespace pa
