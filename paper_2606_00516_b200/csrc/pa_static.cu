// pa_decode_attention_static (include/pa.h): decode attention for callers that cannot allocate device memory.
//
// A variant of the split-KV decode step (a5/a6 of SURVEY §8(a): "Decode attention streams the full KV-cache context
// per token") whose scratch — the per-split partials (m, l, unnormalised O) and the arrival counters of
// the in-launch merge — lives in a file-scope __device__ array of kScratchBytes instead of a caller workspace.  No
// context, no plan upload, no pinned staging: the call enqueues one memset of the counters and one kernel and nothing
// else.  It is a plain kernel (one warp per (sequence, q head, KV split), fp32 online softmax); the tuned path is
// pa_batch_attention.  Self-contained: shares only the pool-layout constant with the rest of the library.
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "../../include/pa.h"
#include "pa_internal.h"

namespace {

constexpr int64_t kScratchBytes = PA_STATIC_SCRATCH_BYTES;
constexpr int kMaxDevices = 64;
constexpr int kMaxSplits = 32;

// Held by every GPU that loads the library, until the process exits.  Shared by all calls on a device.
static __device__ __align__(256) unsigned char g_static_scratch[kScratchBytes];

std::mutex g_setup_mutex;
unsigned char* g_scratch_dev[kMaxDevices];     // device address of g_static_scratch, per device ordinal (null = not looked up yet)
thread_local char g_err[256] = "";

int32_t fail(int32_t code, const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

int64_t align_up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }

struct StaticParams {
    const __nv_bfloat16* q;
    const __nv_bfloat16* k_pool;
    const __nv_bfloat16* v_pool;
    __nv_bfloat16* out;
    const int32_t* context_lens;
    const int32_t* block_tables;
    int32_t* counters;      // [n_seq * Hq] arrivals per output row (zeroed by the call's memset)
    float2* part_ml;        // [n_seq * Hq][n_splits] (m in the log2 domain, l)
    float* part_o;          // [n_seq * Hq][n_splits][D] unnormalised partial outputs
    int32_t n_seq, Hq, Hkv, G, max_blocks_per_seq, n_splits;
    float scale_log2;
};

// one warp: q head h of decode sequence s over the keys of split `sp`; the last-arriving warp of (s, h) merges
template <int D>
__global__ void __launch_bounds__(256) pa_decode_static_kernel(StaticParams p) {
    constexpr int EPL = D / 32;     // elements per lane
    const int lane = threadIdx.x & 31;
    const int g = threadIdx.x >> 5;                 // q head within the KV group
    const int sp = blockIdx.x, kvh = blockIdx.y, s = blockIdx.z;
    const int h = kvh * p.G + g;
    const int kv_len = p.context_lens[s] + 1;       // the new token attends to itself
    const int nblk = (kv_len + pa::kBlock - 1) / pa::kBlock;
    const int per = (nblk + p.n_splits - 1) / p.n_splits;
    const int t0 = min(sp * per, nblk) * pa::kBlock;
    const int t1 = min(min((sp + 1) * per, nblk) * pa::kBlock, kv_len);
    const int32_t* bt = p.block_tables + (int64_t)s * p.max_blocks_per_seq;
    const int64_t row = (int64_t)s * p.Hq + h;

    float qv[EPL], acc[EPL];
    const __nv_bfloat16* qp = p.q + row * D + lane * EPL;
#pragma unroll
    for (int e = 0; e < EPL; ++e) { qv[e] = __bfloat162float(qp[e]); acc[e] = 0.f; }
    float m = -INFINITY, l = 0.f;
    for (int t = t0; t < t1; ++t) {
        const int64_t blk = __ldg(bt + t / pa::kBlock);
        const int64_t off = ((blk * p.Hkv + kvh) * pa::kBlock + (t % pa::kBlock)) * D + lane * EPL;
        float dot = 0.f;
#pragma unroll
        for (int e = 0; e < EPL; ++e) dot += qv[e] * __bfloat162float(p.k_pool[off + e]);
#pragma unroll
        for (int x = 16; x >= 1; x >>= 1) dot += __shfl_xor_sync(0xffffffffu, dot, x);
        const float z = dot * p.scale_log2;
        const float mn = fmaxf(m, z);
        const float c = exp2f(m - mn), w = exp2f(z - mn);
        l = l * c + w;
#pragma unroll
        for (int e = 0; e < EPL; ++e) acc[e] = acc[e] * c + w * __bfloat162float(p.v_pool[off + e]);
        m = mn;
    }
    // partial of this split (an empty split leaves m = -inf, l = 0, acc = 0: weight 0 in the merge)
    const int64_t slot = row * p.n_splits + sp;
    float* po = p.part_o + slot * D + lane * EPL;
#pragma unroll
    for (int e = 0; e < EPL; ++e) po[e] = acc[e];
    if (lane == 0) p.part_ml[slot] = make_float2(m, l);
    __threadfence();
    __syncwarp();
    int arrived = 0;
    if (lane == 0) arrived = atomicAdd(p.counters + row, 1);
    arrived = __shfl_sync(0xffffffffu, arrived, 0);
    if (arrived != p.n_splits - 1) return;
    __threadfence();
    // merge: split 0 always holds key 0, so the maximum is finite
    float M = -INFINITY;
    for (int i = 0; i < p.n_splits; ++i) M = fmaxf(M, __ldcg(&p.part_ml[row * p.n_splits + i].x));
    float L = 0.f;
#pragma unroll
    for (int e = 0; e < EPL; ++e) acc[e] = 0.f;
    for (int i = 0; i < p.n_splits; ++i) {
        const float2 ml = __ldcg(&p.part_ml[row * p.n_splits + i]);
        const float w = exp2f(ml.x - M);
        L += w * ml.y;
        const float* pi = p.part_o + (row * p.n_splits + i) * D + lane * EPL;
#pragma unroll
        for (int e = 0; e < EPL; ++e) acc[e] += w * __ldcg(pi + e);
    }
    const float inv = 1.f / L;
    __nv_bfloat16* op = p.out + row * D + lane * EPL;
#pragma unroll
    for (int e = 0; e < EPL; ++e) op[e] = __float2bfloat16_rn(acc[e] * inv);
}

}  // namespace

extern "C" {

int64_t pa_static_scratch_bytes(void) { return kScratchBytes; }

const char* pa_static_last_error(void) { return g_err; }

int32_t pa_decode_attention_static(const void* q, const void* k_pool, const void* v_pool, const int32_t* d_context_lens,
                                   const int32_t* d_block_tables, int32_t n_seq, int32_t num_q_heads,
                                   int32_t num_kv_heads, int32_t head_dim, int32_t max_blocks_per_seq,
                                   int32_t max_kv_len, float softmax_scale, void* out, int32_t device, void* stream) {
    g_err[0] = 0;
    if (n_seq < 0) return fail(PA_ERR_INVALID, "pa_decode_attention_static: negative n_seq");
    if (num_q_heads <= 0 || num_kv_heads <= 0 || max_blocks_per_seq <= 0 || max_kv_len <= 0 ||
        max_kv_len > (int64_t)max_blocks_per_seq * pa::kBlock)
        return fail(PA_ERR_INVALID, "pa_decode_attention_static: non-positive size, or max_kv_len > max_blocks_per_seq * 16");
    if ((head_dim != 128 && head_dim != 256) || num_q_heads % num_kv_heads != 0 || num_q_heads / num_kv_heads > pa::kMaxGroup)
        return fail(PA_ERR_UNSUPPORTED, "pa_decode_attention_static: head_dim not in {128, 256}, or Hq/Hkv not an integer <= 8");
    if (device < 0 || device >= kMaxDevices) return fail(PA_ERR_INVALID, "pa_decode_attention_static: device ordinal out of range");
    if (!(softmax_scale > 0.f) || !std::isfinite(softmax_scale))
        return fail(PA_ERR_INVALID, "pa_decode_attention_static: softmax_scale must be positive and finite");
    if (n_seq == 0) return PA_OK;
    if (n_seq > 65535) return fail(PA_ERR_INVALID, "pa_decode_attention_static: n_seq > 65535");
    if (!q || !k_pool || !v_pool || !d_context_lens || !d_block_tables || !out)
        return fail(PA_ERR_INVALID, "pa_decode_attention_static: null pointer");
    // ---- scratch layout: counters | part_ml | part_o, for the largest split count that fits the static array
    const int64_t rows = (int64_t)n_seq * num_q_heads;
    const int64_t cnt_bytes = align_up(rows * 4, 256);
    auto need = [&](int64_t splits) {
        return cnt_bytes + align_up(rows * splits * (int64_t)sizeof(float2), 256) + rows * splits * head_dim * 4;
    };
    if (need(1) > kScratchBytes)
        return fail(PA_ERR_WORKSPACE,
                    "pa_decode_attention_static: n_seq * num_q_heads = %lld rows need %lld bytes of scratch even unsplit; "
                    "the static scratch holds %lld (use pa_batch_attention with a caller workspace)",
                    (long long)rows, (long long)need(1), (long long)kScratchBytes);
    // enough (sequence, KV head, split) CTAs for a few waves over the SMs, splits of at least 256 keys
    const int64_t groups = (int64_t)n_seq * num_kv_heads;
    int64_t splits = std::min<int64_t>({kMaxSplits, (1184 + groups - 1) / groups, ((int64_t)max_kv_len + 255) / 256});
    splits = std::max<int64_t>(splits, 1);
    while (splits > 1 && need(splits) > kScratchBytes) --splits;

    int cur = -1;
    cudaError_t e = cudaGetDevice(&cur);
    if (e != cudaSuccess) return fail(PA_ERR_CUDA, "pa_decode_attention_static: cudaGetDevice: %s", cudaGetErrorString(e));
    if (cur != device)
        return fail(PA_ERR_INVALID, "pa_decode_attention_static: current CUDA device %d is not `device` %d", cur, device);

    // ---- once per device, with that device current: the device address of the scratch array (in host code the
    // array's name is only a stand-in for the symbol, not an address a kernel can use)
    unsigned char* scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_setup_mutex);
        if (!g_scratch_dev[device]) {
            void* ptr = nullptr;
            e = cudaGetSymbolAddress(&ptr, g_static_scratch);
            if (e != cudaSuccess || !ptr) {
                cudaGetLastError();
                return fail(PA_ERR_CUDA, "pa_decode_attention_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            }
            g_scratch_dev[device] = static_cast<unsigned char*>(ptr);
        }
        scratch = g_scratch_dev[device];
    }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    StaticParams p;
    p.q = static_cast<const __nv_bfloat16*>(q);
    p.k_pool = static_cast<const __nv_bfloat16*>(k_pool);
    p.v_pool = static_cast<const __nv_bfloat16*>(v_pool);
    p.out = static_cast<__nv_bfloat16*>(out);
    p.context_lens = d_context_lens;
    p.block_tables = d_block_tables;
    p.counters = reinterpret_cast<int32_t*>(scratch);
    p.part_ml = reinterpret_cast<float2*>(scratch + cnt_bytes);
    p.part_o = reinterpret_cast<float*>(scratch + cnt_bytes + align_up(rows * splits * (int64_t)sizeof(float2), 256));
    p.n_seq = n_seq; p.Hq = num_q_heads; p.Hkv = num_kv_heads; p.G = num_q_heads / num_kv_heads;
    p.max_blocks_per_seq = max_blocks_per_seq; p.n_splits = (int32_t)splits;
    p.scale_log2 = softmax_scale * 1.4426950408889634f;
    // the array keeps the previous call's contents: the arrival counters must start at zero (the partials are
    // written before they are read, so they need no clearing)
    e = cudaMemsetAsync(p.counters, 0, (size_t)(rows * 4), st);
    if (e != cudaSuccess) return fail(PA_ERR_CUDA, "pa_decode_attention_static: cudaMemsetAsync: %s", cudaGetErrorString(e));
    const dim3 grid((unsigned)splits, (unsigned)num_kv_heads, (unsigned)n_seq), block(32 * p.G);
    if (head_dim == 128) pa_decode_static_kernel<128><<<grid, block, 0, st>>>(p);
    else pa_decode_static_kernel<256><<<grid, block, 0, st>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(PA_ERR_CUDA, "pa_decode_attention_static: launch: %s", cudaGetErrorString(e));
    return PA_OK;
}

}  // extern "C"
