// Host-callable launch wrappers (defined in pa_kernels.cu) used by the C-ABI layer (pa_api.cu).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cstdint>

#include "pa_internal.h"

namespace pa {

struct LaunchShape {
    int32_t Hq, Hkv, D;
    int32_t max_blocks_per_seq;
};

cudaError_t launch_kv_append(const LaunchShape& sh, const void* k_new, const void* v_new, void* k_pool, void* v_pool,
                             const int32_t* cu_seqlens_q, const int32_t* context_lens, const int32_t* block_tables,
                             int32_t n_seq, int32_t n_tok, cudaStream_t stream);

cudaError_t launch_kv_gather(const LaunchShape& sh, const void* k_pool, const void* v_pool, const int32_t* table_row,
                             int32_t kv_len, void* k_out, void* v_out, cudaStream_t stream);

// Pool tensor maps of the decode role: the pool viewed as the 5-D tensor [block][kv head][D/64][16 rows][64 cols]
// (row stride 2·D bytes, 64-column plane stride 128 bytes), box = 64 columns x rows x 2 planes, so ONE tensor load
// brings the 128-column K (or V) unit of a block-head into the ring slot as [plane][row][128 B] (128B swizzle).
// Index 0: 16-row, two-plane box (a full block); 1..4: 8, 4, 2, 1 rows of ONE plane — the filled rows of a partly
// filled last block are fetched as the binary decomposition of their count (per plane), so decode never reads slots
// that hold no token.
struct TailMaps {
    CUtensorMap k[5], v[5];
};

struct AttnLaunch {
    LaunchShape sh;
    const void* q;
    void* out;
    const void* k_pool;
    const void* v_pool;
    const int32_t* cu_seqlens_q;
    const int32_t* context_lens;
    const int32_t* block_tables;
    float softmax_scale;
    PlanView plan;
    int32_t decode_ctas;     // CTAs that start in the decode role (0 = none)
    int32_t prefill_ctas;    // CTAs that start in the prefill role (0 = none)
    int32_t p_in_tmem;       // prefill variant: P staged in TMEM (1) or shared memory (0)
    int32_t n_simple_tiles;  // tiles routed to the plain kernel (debug)
    const CUtensorMap* tmQ;  // host copy of the query tensor map (null without prefill units)
    const CUtensorMap* tmQd; // query tensor map of the decode role: [n_tok*Hq, D], box = G rows x 64 columns (null without decode bundles)
    const CUtensorMap* tmK;  // host copies of the pool tensor maps
    const CUtensorMap* tmV;
    const TailMaps* tails;
};

// Set opt-in shared memory sizes once per process/device.
cudaError_t configure_kernels();
cudaError_t launch_attention(const AttnLaunch& a, cudaStream_t stream, int* launches_out);
int attention_smem_bytes();

}  // namespace pa
