// C-ABI layer of libpa_b200.so (include/pa.h): context, validation, planner (a1/a7), launches, timer (a8).
// Host code only; kernels live in pa_kernels.cu.
#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/pa.h"
#include "pa_launch.h"

using namespace pa;

struct pa_ctx {
    pa_config cfg{};
    int G = 1;
    int num_sms = 0;
    std::string err;
    // workspace layout (bytes from the workspace base)
    int64_t off_counters = 0, off_plan = 0, off_redo = 0, off_part_ml = 0, off_part_o = 0, ws_bytes = 0;
    int64_t plan_region_bytes = 0;
    int32_t max_bundles = 0, max_tiles = 0, max_split = 0, max_workers = 0;
    // pinned staging for the plan upload: a ring, so that pa_plan only waits when kStages plans are in flight
    static constexpr int kStages = 3;
    uint8_t* h_stage[kStages] = {nullptr, nullptr, nullptr};
    cudaEvent_t stage_ev[kStages] = {nullptr, nullptr, nullptr};
    bool stage_pending[kStages] = {false, false, false};
    int stage_next = 0;
    // current plan
    bool planned = false;
    PlanView view{};
    int32_t decode_ctas = 0, n_simple_tiles = 0, launches_per_call = 0, prefill_ctas = 0, p_in_tmem = 1;
    int32_t planned_n_tok = 0, n_items = 0, bundles_per_stream = 0, prefill_mode = 0, n_levels = 1;
    int64_t plan_host_ns = 0, plan_ns_validate = 0, plan_ns_lists = 0;   // whole call; validation; tiles + bundles (rest: enqueue of the upload)
    // tensor-map cache
    const void* tm_k_ptr = nullptr;
    const void* tm_v_ptr = nullptr;
    const void* tm_q_ptr = nullptr;
    int32_t tm_q_ntok = -1;
    const void* tm_qd_ptr = nullptr;
    int32_t tm_qd_ntok = -1;
    CUtensorMap tmK{}, tmV{}, tmQ{}, tmQd{};
    TailMaps tails{};   // decode views of the K and V pools (16/8/4/2/1-row boxes)
    // timer
    cudaEvent_t t0 = nullptr, t1 = nullptr;
    std::map<int, std::map<int, std::vector<double>>> samples;  // r per-mille -> n_tok -> seconds
};

namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn g_encode = nullptr;      // driver entry point, resolved once per process (std::call_once)
std::once_flag g_encode_once;

int32_t fail(pa_ctx* ctx, int32_t code, const std::string& msg) {
    if (ctx) ctx->err = msg;
    return code;
}
int32_t cuda_fail(pa_ctx* ctx, cudaError_t e, const char* where) {
    return fail(ctx, PA_ERR_CUDA, std::string(where) + ": " + cudaGetErrorString(e));
}
int64_t align_up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }

// every call that enqueues work requires cfg.device to be the calling thread's current device
int32_t check_device(pa_ctx* ctx, const char* where) {
    int cur = -1;
    cudaError_t e = cudaGetDevice(&cur);
    if (e != cudaSuccess) return cuda_fail(ctx, e, where);
    if (cur != ctx->cfg.device)
        return fail(ctx, PA_ERR_INVALID, std::string(where) + ": current CUDA device " + std::to_string(cur) +
                                             " is not the context's device " + std::to_string(ctx->cfg.device));
    return PA_OK;
}

bool resolve_encode() {
    std::call_once(g_encode_once, [] {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) == cudaSuccess && fn)
            g_encode = reinterpret_cast<EncodeTiledFn>(fn);
    });
    return g_encode != nullptr;
}

// pool[num_blocks][Hkv][16][D] bf16 -> 4-D tensor map, box = 64 columns x 16 tokens of one (block, head), 128B swizzle
// rows < 16: the same tensor with a shorter box, used to fetch only the filled rows of a sequence's last block
int32_t make_pool_map(pa_ctx* ctx, const void* pool, CUtensorMap* out, int rows = kBlock) {
    if (!resolve_encode()) return fail(ctx, PA_ERR_CUDA, "cuTensorMapEncodeTiled entry point not found");
    const pa_config& c = ctx->cfg;
    const cuuint64_t D = c.head_dim, Hkv = c.num_kv_heads;
    cuuint64_t dims[4] = {D, (cuuint64_t)kBlock, Hkv, (cuuint64_t)c.num_blocks};
    cuuint64_t strides[3] = {D * 2, (cuuint64_t)kBlock * D * 2, Hkv * kBlock * D * 2};
    cuuint32_t box[4] = {64, (cuuint32_t)rows, 1, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = g_encode(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 4, const_cast<void*>(pool), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(ctx, PA_ERR_CUDA, "cuTensorMapEncodeTiled failed (" + std::to_string((int)r) + ")");
    return PA_OK;
}

// decode view of the pool (pa_launch.h TailMaps): 5-D, box = 64 columns x `rows` tokens x `planes` column planes
int32_t make_pool_map5(pa_ctx* ctx, const void* pool, CUtensorMap* out, int rows, int planes) {
    const pa_config& c = ctx->cfg;
    const cuuint64_t D = c.head_dim, Hkv = c.num_kv_heads;
    cuuint64_t dims[5] = {64, (cuuint64_t)kBlock, D / 64, Hkv, (cuuint64_t)c.num_blocks};
    cuuint64_t strides[4] = {D * 2, 128, (cuuint64_t)kBlock * D * 2, Hkv * kBlock * D * 2};
    cuuint32_t box[5] = {64, (cuuint32_t)rows, (cuuint32_t)planes, 1, 1};
    cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    CUresult r = g_encode(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, const_cast<void*>(pool), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(ctx, PA_ERR_CUDA, "cuTensorMapEncodeTiled(pool, 5-D) failed (" + std::to_string((int)r) + ")");
    return PA_OK;
}

// q[n_tok][Hq][D] bf16 -> 3-D tensor map, box = 64 columns x 1 head x 128 token rows, 128B swizzle
// (rows past n_tok are zero-filled by the TMA unit)
int32_t make_q_map(pa_ctx* ctx, const void* q, int32_t n_tok, CUtensorMap* out) {
    const pa_config& c = ctx->cfg;
    const cuuint64_t D = c.head_dim, Hq = c.num_q_heads;
    cuuint64_t dims[3] = {D, Hq, (cuuint64_t)n_tok};
    cuuint64_t strides[2] = {D * 2, Hq * D * 2};
    cuuint32_t box[3] = {64, 1, (cuuint32_t)kQTile};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = g_encode(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(q), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(ctx, PA_ERR_CUDA, "cuTensorMapEncodeTiled(q) failed (" + std::to_string((int)r) + ")");
    return PA_OK;
}

// q[n_tok][Hq][D] bf16 viewed as [n_tok*Hq][D] -> 2-D tensor map, box = 64 columns x G head rows (the q heads of
// one KV head of one decode token are G consecutive rows), 128B swizzle
int32_t make_qdec_map(pa_ctx* ctx, const void* q, int32_t n_tok, CUtensorMap* out) {
    const pa_config& c = ctx->cfg;
    const cuuint64_t D = c.head_dim;
    cuuint64_t dims[2] = {D, (cuuint64_t)n_tok * c.num_q_heads};
    cuuint64_t strides[1] = {D * 2};
    cuuint32_t box[2] = {64, (cuuint32_t)ctx->G};
    cuuint32_t estr[2] = {1, 1};
    CUresult r = g_encode(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(q), dims, strides, box, estr,
                          CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(ctx, PA_ERR_CUDA, "cuTensorMapEncodeTiled(q decode) failed (" + std::to_string((int)r) + ")");
    return PA_OK;
}

double median(std::vector<double> v) {
    std::sort(v.begin(), v.end());
    size_t n = v.size();
    return n % 2 ? v[n / 2] : 0.5 * (v[n / 2 - 1] + v[n / 2]);
}

}  // namespace

extern "C" {

int32_t pa_create(pa_ctx** out, const pa_config* cfg) {
    if (!out || !cfg) return PA_ERR_INVALID;
    *out = nullptr;
    if (cfg->num_q_heads <= 0 || cfg->num_kv_heads <= 0 || cfg->num_blocks <= 0 || cfg->max_seqs <= 0 ||
        cfg->max_tokens <= 0 || cfg->max_blocks_per_seq <= 0 || cfg->device < 0 || cfg->tune_prefill_ctas < 0 ||
        cfg->tune_bundles_per_stream < 0 || cfg->tune_bundles_per_stream > 4 || cfg->tune_min_bundle_blocks < 0 ||
        cfg->tune_levels < 0 || cfg->tune_levels > 8)
        return PA_ERR_INVALID;
    if ((cfg->head_dim != 128 && cfg->head_dim != 256) || cfg->block_size != kBlock ||
        cfg->num_q_heads % cfg->num_kv_heads != 0 || cfg->num_q_heads / cfg->num_kv_heads > kMaxGroup)
        return PA_ERR_UNSUPPORTED;
    // the caller's current device is restored before returning (success or failure)
    int prev_device = -1;
    if (cudaGetDevice(&prev_device) != cudaSuccess) { cudaGetLastError(); return PA_ERR_CUDA; }
    pa_ctx* ctx = new pa_ctx();
    ctx->cfg = *cfg;
    ctx->G = cfg->num_q_heads / cfg->num_kv_heads;
    cudaError_t e = cudaSetDevice(cfg->device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, cfg->device);
    int cc_major = 0;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, cfg->device);
    // opt-in shared memory is a per-device function attribute: set it for this context's device every time
    if (e == cudaSuccess && cc_major == 10) e = configure_kernels();
    if (e != cudaSuccess || cc_major != 10) {
        cudaGetLastError();
        delete ctx;
        cudaSetDevice(prev_device);
        return PA_ERR_CUDA;  // no usable sm_100 device: there is no fallback path
    }
    // ---- workspace layout
    ctx->max_workers = ctx->num_sms * kDecodeWarps;
    // k <= 4 equal bundles per worker, plus the bundles that uncut short groups close early (at most one per group)
    const int32_t eq_bundles = ctx->max_workers * 5 + 8;
    ctx->max_bundles = eq_bundles + cfg->max_seqs * cfg->num_kv_heads;
    ctx->max_split = 2 * eq_bundles;          // only groups cut by a bundle boundary have partials
    ctx->max_tiles = cfg->max_tokens / kQTile + cfg->max_seqs + 1;
    int64_t off = 0;
    ctx->off_counters = off;
    off += align_up(16 * 4 + (int64_t)cfg->max_seqs * cfg->num_kv_heads * 4, 256);
    ctx->off_plan = off;
    ctx->plan_region_bytes = align_up((int64_t)ctx->max_bundles * sizeof(DecBundle), 256) +
                             align_up((int64_t)ctx->max_tiles * sizeof(PreTile), 256);
    off += ctx->plan_region_bytes;
    ctx->off_redo = off;
    off += align_up((int64_t)cfg->max_tokens * cfg->num_q_heads * sizeof(int2), 256);
    ctx->off_part_ml = off;
    off += align_up((int64_t)ctx->max_split * kMaxGroup * sizeof(float2), 256);
    ctx->off_part_o = off;
    off += align_up((int64_t)ctx->max_split * ctx->G * cfg->head_dim * 4, 256);
    ctx->ws_bytes = off;
    for (int i = 0; i < pa_ctx::kStages && e == cudaSuccess; ++i) {
        e = cudaMallocHost(reinterpret_cast<void**>(&ctx->h_stage[i]), (size_t)ctx->plan_region_bytes);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->stage_ev[i], cudaEventDisableTiming);
    }
    if (e == cudaSuccess) e = cudaEventCreate(&ctx->t0);
    if (e == cudaSuccess) e = cudaEventCreate(&ctx->t1);
    if (e != cudaSuccess) {
        cudaGetLastError();
        pa_destroy(ctx);
        cudaSetDevice(prev_device);
        return PA_ERR_CUDA;
    }
    cudaSetDevice(prev_device);
    *out = ctx;
    return PA_OK;
}

int32_t pa_destroy(pa_ctx* ctx) {
    if (!ctx) return PA_ERR_INVALID;
    for (int i = 0; i < pa_ctx::kStages; ++i) {
        if (ctx->stage_pending[i] && ctx->stage_ev[i]) cudaEventSynchronize(ctx->stage_ev[i]);
        if (ctx->h_stage[i]) cudaFreeHost(ctx->h_stage[i]);
        if (ctx->stage_ev[i]) cudaEventDestroy(ctx->stage_ev[i]);
    }
    if (ctx->t0) cudaEventDestroy(ctx->t0);
    if (ctx->t1) cudaEventDestroy(ctx->t1);
    delete ctx;
    return PA_OK;
}

int64_t pa_workspace_bytes(const pa_ctx* ctx) { return ctx ? ctx->ws_bytes : PA_ERR_INVALID; }

int64_t pa_kv_pool_bytes(const pa_ctx* ctx) {
    if (!ctx) return PA_ERR_INVALID;
    return ctx->cfg.num_blocks * ctx->cfg.num_kv_heads * (int64_t)kBlock * ctx->cfg.head_dim * 2;
}

const char* pa_last_error(const pa_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int32_t pa_kv_append(pa_ctx* ctx, const void* k_new, const void* v_new, void* k_pool, void* v_pool,
                     const int32_t* d_cu, const int32_t* d_ctx, const int32_t* d_bt, int32_t n_seq, int32_t n_tok,
                     void* stream) {
    if (!ctx) return PA_ERR_INVALID;
    if (n_seq < 0 || n_tok < 0) return fail(ctx, PA_ERR_INVALID, "pa_kv_append: negative size");
    if (n_seq == 0 || n_tok == 0) return PA_OK;
    if (!k_new || !v_new || !k_pool || !v_pool || !d_cu || !d_ctx || !d_bt)
        return fail(ctx, PA_ERR_INVALID, "pa_kv_append: null pointer");
    if (n_seq > ctx->cfg.max_seqs || n_tok > ctx->cfg.max_tokens)
        return fail(ctx, PA_ERR_INVALID, "pa_kv_append: n_seq/n_tok exceed the configured maxima");
    if (int32_t rc = check_device(ctx, "pa_kv_append")) return rc;
    LaunchShape sh{ctx->cfg.num_q_heads, ctx->cfg.num_kv_heads, ctx->cfg.head_dim, ctx->cfg.max_blocks_per_seq};
    cudaError_t e = launch_kv_append(sh, k_new, v_new, k_pool, v_pool, d_cu, d_ctx, d_bt, n_seq, n_tok,
                                     static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? PA_OK : cuda_fail(ctx, e, "pa_kv_append");
}

int32_t pa_kv_gather(pa_ctx* ctx, const void* k_pool, const void* v_pool, const int32_t* d_row, int32_t kv_len,
                     void* k_out, void* v_out, void* stream) {
    if (!ctx) return PA_ERR_INVALID;
    if (kv_len < 0) return fail(ctx, PA_ERR_INVALID, "pa_kv_gather: negative kv_len");
    if (kv_len == 0) return PA_OK;
    if (!k_pool || !v_pool || !d_row || !k_out || !v_out) return fail(ctx, PA_ERR_INVALID, "pa_kv_gather: null pointer");
    if (kv_len > (int64_t)ctx->cfg.max_blocks_per_seq * kBlock)
        return fail(ctx, PA_ERR_INVALID, "pa_kv_gather: kv_len exceeds max_blocks_per_seq * 16");
    if (int32_t rc = check_device(ctx, "pa_kv_gather")) return rc;
    LaunchShape sh{ctx->cfg.num_q_heads, ctx->cfg.num_kv_heads, ctx->cfg.head_dim, ctx->cfg.max_blocks_per_seq};
    cudaError_t e = launch_kv_gather(sh, k_pool, v_pool, d_row, kv_len, k_out, v_out, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? PA_OK : cuda_fail(ctx, e, "pa_kv_gather");
}

// ---------------------------------------------------------------------------------------------
// a1 plan.  Decode: the blocks of all (decode seq, KV head) groups form one stream (group order) that is cut into
// equal-cost bundles; a group cut by a bundle boundary is a split group whose partials the last-arriving worker
// merges.  The plan holds one 32-byte DecBundle per bundle (the streams derive their items from it and from
// context_lens), so it is O(bundles + sequences) host work and a few KB of upload, not O(groups).
// Prefill: 128-row query tiles in longest-first order.
// ---------------------------------------------------------------------------------------------
namespace {

// Cuts the decode block stream into bundles, writing DecBundle records in place.
struct BundleCutter {
    DecBundle* out;
    int32_t max_bundles, max_split;
    int64_t target;
    int32_t n_bundles = 0, n_split = 0, n_items = 0;
    int64_t cur = 0;          // blocks in the open bundle (out[n_bundles])
    bool open = false;
    bool overflow = false;

    void add(int32_t grp, int32_t b0, int32_t b1, int32_t nblk) {   // blocks [b0, b1) of group grp join the open bundle
        if (n_bundles >= max_bundles) { overflow = true; return; }
        DecBundle& d = out[n_bundles];
        if (!open) {
            d = DecBundle{grp, b0, grp, 0, -1, 1, -1, 1};
            open = true;
        }
        d.grp_end = grp;
        d.blk_end = b1 == nblk ? -1 : b1;
        cur += b1 - b0;
        ++n_items;
    }
    void add_whole_groups(int32_t grp0, int32_t groups, int32_t nblk) {   // `groups` consecutive groups of nblk blocks, uncut
        add(grp0, 0, nblk, nblk);
        if (overflow) return;
        out[n_bundles].grp_end = grp0 + groups - 1;
        n_items += groups - 1;
        cur += (int64_t)(groups - 1) * nblk;
    }
    // Groups that are never cut (short ones) make a bundle end a little before or after its target.  The difference is
    // carried into the next rounding decision, so that the boundaries stay near i * target and the number of bundles
    // near (total blocks) / target: without the carry 3.3 groups per stream always round to 3, and a tenth of the
    // streams get a second bundle while the others idle.
    // Long groups are cut exactly at `target`, so only the rounding decisions (round_target) see the carry.
    // Used with one static bundle per stream only: with queue-drawn bundles a few bundles more or less do not matter, and
    // the plain rule measured 1 % faster there (C4 r = 0.2, thirds: 2616 vs 2640 us).
    bool use_carry = false;
    int64_t carry = 0;
    int64_t round_target() const { return target + carry; }
    void close() {
        if (open) {
            ++n_bundles;
            open = false;
            if (use_carry) carry = std::max(-target / 2, std::min(target / 2, carry + target - cur));
        }
        cur = 0;
    }
    // the group `grp` was emitted as `parts` consecutive parts, the first one into bundle `first_bundle`
    void mark_split(int32_t grp, int32_t first_bundle, int32_t parts) {
        if (n_split + parts > max_split || parts > 0xffff) { overflow = true; return; }
        for (int32_t i = 0; i < parts; ++i) {
            DecBundle& d = out[first_bundle + i];
            if (d.grp_begin == grp) { d.first_part_base = n_split; d.first_part = (i << 16) | parts; }
            else { d.last_part_base = n_split; d.last_part = (i << 16) | parts; }
        }
        n_split += parts;
    }
};

}  // namespace

int32_t pa_plan(pa_ctx* ctx, const int32_t* h_cu, const int32_t* h_ctx, int32_t n_seq, int32_t num_decode_seqs,
                void* d_workspace, int64_t workspace_bytes, void* stream_) {
    if (!ctx) return PA_ERR_INVALID;
    const auto t_begin = std::chrono::steady_clock::now();
    ctx->planned = false;
    const pa_config& c = ctx->cfg;
    if (n_seq < 0 || num_decode_seqs < 0 || num_decode_seqs > n_seq)
        return fail(ctx, PA_ERR_INVALID, "pa_plan: bad n_seq / num_decode_seqs");
    if (n_seq > c.max_seqs) return fail(ctx, PA_ERR_INVALID, "pa_plan: n_seq > max_seqs");
    if (n_seq > 0 && (!h_cu || !h_ctx)) return fail(ctx, PA_ERR_INVALID, "pa_plan: null descriptor");
    if (!d_workspace || workspace_bytes < ctx->ws_bytes || (reinterpret_cast<uintptr_t>(d_workspace) & 255))
        return fail(ctx, PA_ERR_WORKSPACE, "pa_plan: workspace missing, misaligned or smaller than pa_workspace_bytes");
    if (n_seq > 0 && h_cu[0] != 0) return fail(ctx, PA_ERR_INVALID, "pa_plan: cu_seqlens_q[0] != 0");
    const int64_t max_kv = (int64_t)c.max_blocks_per_seq * kBlock;
    int64_t total_blocks_1 = 0;     // blocks of the decode sequences, per KV head
    for (int s = 0; s < n_seq; ++s) {
        const int64_t ql = (int64_t)h_cu[s + 1] - h_cu[s];
        if (ql < 0) return fail(ctx, PA_ERR_INVALID, "pa_plan: cu_seqlens_q not non-decreasing");
        if (h_ctx[s] < 0) return fail(ctx, PA_ERR_INVALID, "pa_plan: negative context length");
        if (s < num_decode_seqs) {
            if (ql != 1) return fail(ctx, PA_ERR_INVALID, "pa_plan: decode sequence with q_len != 1");
            total_blocks_1 += ((int64_t)h_ctx[s] + kBlock) / kBlock;     // ceil((ctx + 1) / 16)
        }
        if ((int64_t)h_ctx[s] + ql > max_kv) return fail(ctx, PA_ERR_INVALID, "pa_plan: kv_len exceeds max_blocks_per_seq * 16");
    }
    const int32_t n_tok = n_seq > 0 ? h_cu[n_seq] : 0;
    if (n_tok > c.max_tokens) return fail(ctx, PA_ERR_INVALID, "pa_plan: n_tok > max_tokens");
    if (int32_t rc = check_device(ctx, "pa_plan")) return rc;
    const auto t_valid = std::chrono::steady_clock::now();

    cudaStream_t stream = static_cast<cudaStream_t>(stream_);
    const int stage = ctx->stage_next;
    if (ctx->stage_pending[stage]) {    // only when kStages plans are already in flight
        cudaError_t e = cudaEventSynchronize(ctx->stage_ev[stage]);
        if (e != cudaSuccess) return cuda_fail(ctx, e, "pa_plan(stage sync)");
        ctx->stage_pending[stage] = false;
    }
    uint8_t* h_stage = ctx->h_stage[stage];
    const bool simple_all = (c.flags & PA_FLAG_DEBUG_SIMPLE) != 0;
    const int Hkv = c.num_kv_heads, D = c.head_dim, G = ctx->G;

    // ---- prefill tiles (built first: the decode bundling below depends on how many CTAs prefill takes);
    // staging layout: tiles | bundles
    PreTile* tiles = reinterpret_cast<PreTile*>(h_stage);
    int32_t n_tiles = 0;
    for (int s = simple_all ? 0 : num_decode_seqs; s < n_seq; ++s) {
        const int32_t ql = h_cu[s + 1] - h_cu[s];
        for (int32_t q0 = 0; q0 < ql; q0 += kQTile) {
            if (n_tiles >= ctx->max_tiles) return fail(ctx, PA_ERR_INVALID, "pa_plan: tile list overflow");
            tiles[n_tiles++] = PreTile{s, q0, std::min(kQTile, ql - q0), h_ctx[s], h_ctx[s] + ql, h_cu[s], {0, 0}};
        }
    }
    // longest first: the queue then hands out units in LPT order (causal tiles late in a chunk see more keys)
    std::stable_sort(tiles, tiles + n_tiles, [](const PreTile& a, const PreTile& b) {
        return a.ctx + a.q_begin + a.q_rows > b.ctx + b.q_begin + b.q_rows;
    });
    // prefill variant: 0 P in TMEM, 1 P in shared memory, 2 plain kernel
    const int prefill_mode = simple_all ? 2 : ((c.flags & PA_FLAG_PREFILL_P_SMEM) ? 1 : 0);
    const int NQ = D == 128 ? 2 : 1;
    const int32_t head_groups = (G + NQ - 1) / NQ;
    const int32_t n_units = prefill_mode == 2 ? 0 : n_tiles * Hkv * head_groups;
    const int n_dec = simple_all ? 0 : num_decode_seqs;
    const int64_t total_blocks = n_dec > 0 ? total_blocks_1 * Hkv : 0;
    // ---- CTA partition of the single launch (a7): share the SMs in proportion to the CTA-time of the two roles,
    // from rates measured with per-CTA timestamps on B200.  Prefill: ~7 us per unit (hand-out, Q/K fill, two-pass
    // first tile, epilogue) + ~0.95 us per (q-head tile, KV tile) pair.  Decode: ~2 us per item and stream plus its
    // bytes at ~16 GB/s per stream (8 streams per CTA) when latency-bound; when its HBM time on all SMs is the
    // larger figure decode is bandwidth-bound and ~96 CTAs saturate HBM, so prefill may take as many CTAs as it
    // needs to finish within the decode's HBM time.  CTAs switch role when their own queue runs dry, so the split
    // only has to be roughly right.
    const int sms = ctx->num_sms;
    int32_t pre_ctas = 0;
    if (n_units > 0 && total_blocks > 0) {
        const int KT = D == 128 ? 128 : 64;
        double t_pre = 0.0;   // CTA-microseconds
        for (int32_t i = 0; i < n_tiles; ++i) {
            const PreTile& t = tiles[i];
            const double n_kv = std::ceil((double)(t.ctx + t.q_begin + t.q_rows) / KT);
            t_pre += (double)Hkv * (head_groups * 7.0 + n_kv * G * 0.95);
        }
        const double dec_bytes = (double)total_blocks * kBlock * D * 2 * 2;
        const double n_groups = (double)n_dec * Hkv;
        const double t_hbm = dec_bytes / 6.5e12 * 1e6;                                        // us, all SMs
        const double t_lat = n_groups * 2.0 / kDecodeWarps + dec_bytes / 16e9 / kDecodeWarps * 1e6;   // CTA-us
        if (sms * t_hbm >= t_lat) {
            const double need = t_pre / t_hbm;                                               // CTAs to hide prefill under decode
            pre_ctas = (int32_t)std::lround(std::min<double>(need, sms - 96));
            pre_ctas = std::max(pre_ctas, (int32_t)std::lround(sms * t_pre / (t_pre + sms * t_hbm)));
        } else {
            // latency-bound launches (C2): the per-unit figures above are round-1 measurements and the prefill role
            // has become faster since; with 0.65 of them the two roles finish together (C2 r = 0.1 ... 0.9, attention
            // launch with factor 1 / 0.8 / 0.64: 38.9 / 35.8 / 33.8, -- / 37.8 / 34.9, 41.9 / 39.0 / 37.9, -- / 39.4 / 38.9,
            // 43.1 / 42.0 / 39.9, -- / 43.9 / 43.0, 46.1 / 46.0 / 44.5, -- / 47.9 / 48.1, 50.1 / 48.2 / 48.1 us)
            pre_ctas = (int32_t)std::lround(sms * 0.65 * t_pre / (0.65 * t_pre + t_lat));
        }
        if (c.tune_prefill_ctas > 0) pre_ctas = c.tune_prefill_ctas;
        pre_ctas = std::max(1, std::min({pre_ctas, sms - 1, n_units}));
    } else if (n_units > 0) {
        pre_ctas = std::min(sms, n_units);
    }
    // ---- decode bundles
    const int64_t off_b = align_up((int64_t)n_tiles * sizeof(PreTile), 256);
    BundleCutter bc{reinterpret_cast<DecBundle*>(h_stage + off_b), ctx->max_bundles, ctx->max_split, 1};
    int k = 0, levels = 1;
    if (total_blocks > 0) {
        // workers that start in the decode role; in a mixed launch the prefill CTAs join through the queue when
        // their units run out (if the rule below leaves bundles in the queue)
        const int64_t W = (int64_t)(sms - pre_ctas) * kDecodeWarps;
        // Bundles per worker (measured on B200): pure decode — one static bundle per stream is best up to a few GB of
        // KV (every extra cut adds parts to the in-launch merges: 4 sequences x 128k keys run at 0.95 of the HBM
        // roofline with 1 bundle per worker and 0.57 with 4); from ~16 GB on a launch lasts milliseconds and a second,
        // queue-drawn bundle per worker evens out unequal stream rates (C5: -5 %).
        const double kv_bytes = (double)total_blocks * kBlock * D * 2 * 2;
        // (C5 on one B200, same call, interleaved, median [min, max] over 24 launches: k = 1 6.47 [5.87, 6.81] ms,
        // k = 2 6.67 [5.81, 6.90], k = 3 5.86 [5.81, 5.91], k = 4 6.31 [6.22, 6.41]: three per stream from 16 GB on.)
        // The rule below is the best, or within 1 % of the best, of k = 1, 2, 3 on every configuration swept under
        // bench.py's timing protocol at the end of round 2 (DESIGN.md §6.5 has the table):
        //  - two equal queue-drawn halves per stream (k = 2) leave a tail of up to half a share when a fast stream
        //    takes a third one, and which stream does differs from run to run (same plan: 1600 or 1780 us); mixed
        //    launches (> 2 prefill CTAs) take thirds from 4.5 GB of KV on so that late-joining prefill CTAs find
        //    queue-drawn work (below that one static bundle per stream is as fast or faster: 3.3 GB 587 -> 518 us,
        //    4.4 GB 712 -> 666);
        //  - ragged batches of >= 3 groups per stream (C4-shaped, lognormal contexts) with a small prefill role take
        //    three bundles per stream from 5 GB on (k = 1 / 2 / 3: 10.6 GB 1977 / 1666 / 1584 us; 12.6 GB 2438 / 1994 /
        //    1868; 8.4 GB 1605 / 1417 / 1241; 5.2 GB 879 / 872 / 839), everything from 16 GB on;
        //  - batches of a few long, equal sequences (under one group per stream) run at the read ceiling with one static
        //    bundle per stream and lose 0-7 % with three, so they keep k = 1 up to 16 GB.
        const double groups_per_share = (double)n_dec * Hkv / (double)W;
        // (mixed, >= 4.5 GB: halves or thirds by groups per stream — five fresh processes each, k = 2 / 3: 4.5 groups per
        // stream 1133-1148 / 992-1007 us, 5.9: 1420-1433 / 1275-1278, 6.1: 1338-1340 / 1343-1346, 7.9: 1342-1357 / 1346-1358,
        // 8.8: 1974-1987 / 2120)
        // Halves are not used at all (outside the guided hand-out): the same k = 2 plan of the headline's r = 0.1 batch ran
        // at 1342-1357 us in five processes and at 1480 us in a sixth, thirds at 1346-1358 in all; with >= 8.5 groups per
        // stream one static bundle (with the carried rounding) is as fast as halves (1989-2000 vs 1974-1987 us).
        k = (pre_ctas > 2 && kv_bytes >= 4.5e9 && groups_per_share < 8.5) ? 3 : 1;
        if (kv_bytes >= 16e9 || (kv_bytes >= 5e9 && groups_per_share >= 3.0 && pre_ctas <= 4)) k = 3;
        // Guided hand-out (PlanView::n_levels): when a stream's share holds many groups (>= 16) and the launch is long
        // enough for unequal stream rates to matter (>= 1 GB of KV, ~150 us), the bundles (two per stream) are taken in
        // eight pieces of 50, 20, 12, 7, 5, 3, 2, 1 % of their groups, large pieces first.  With whole bundles every
        // stream ends up with exactly k of them and the launch ends with its slowest stream; measured on C4 (one B200,
        // same call, interleaved): r = 0.3 / 0.5 / 0.7 / 0.9 / 1.0  4.51 / 6.86 / 10.0 / 13.0 / 14.2 ms with whole
        // bundles, 4.09 / 6.45 / 8.78 / 11.1 / 12.1 ms with pieces.  Pieces are whole groups: no group is cut more
        // often and the planner does no extra work.  Shares of few, long groups (C3, C5) stay with whole bundles
        // (pieces of one or two groups are erratic: C3 113 -> 150 us).
        levels = (groups_per_share >= 16.0 && kv_bytes >= 1e9) ? 8 : 1;
        if (c.tune_levels > 0) levels = c.tune_levels;
        if (levels > 1) k = 2;
        if (c.tune_bundles_per_stream > 0) k = c.tune_bundles_per_stream;
        const int64_t min_blocks = c.tune_min_bundle_blocks > 0 ? c.tune_min_bundle_blocks : 2;
        bc.target = std::max(min_blocks, (total_blocks + W * k - 1) / (W * k));
        bc.use_carry = k == 1;
        // One static bundle per stream must not leave a bundle over: it would run as a second wave on one stream.  The
        // carried rounding keeps the count within one of the stream count; if it still comes out above, cut again with
        // a slightly larger target (rare; one more O(bundles) pass).
        for (int attempt = 0;; ++attempt) {
        for (int s = 0; s < n_dec && !bc.overflow; ++s) {
            const int32_t nblk = (h_ctx[s] + kBlock) / kBlock;          // ceil((ctx + 1) / 16)
            const int32_t grp0 = s * Hkv;
            // a short group (<= 256 keys, or a quarter bundle) is never cut: partials + merge would cost more than
            // the imbalance it leaves (a microsecond or two of streaming)
            if (bc.cur + (int64_t)nblk * Hkv < bc.round_target()) {        // the whole sequence joins the open bundle
                bc.add_whole_groups(grp0, Hkv, nblk);
                continue;
            }
            const bool is_short = nblk <= 16 || (int64_t)nblk * 4 <= bc.target;
            for (int g = 0; g < Hkv && !bc.overflow;) {
                // as many whole groups as fit the open bundle, in one step (the work is O(bundle boundaries))
                const int64_t room = bc.round_target() - bc.cur;
                const int32_t n_fit = room < nblk ? 0 : (int32_t)std::min<int64_t>(
                    room < (int64_t(1) << 31) ? (int64_t)((uint32_t)room / (uint32_t)nblk) : room / nblk, Hkv - g);
                if (n_fit > 0) {
                    bc.add_whole_groups(grp0 + g, n_fit, nblk);
                    g += n_fit;
                    if (bc.cur >= bc.round_target()) bc.close();
                    continue;
                }
                const int32_t grp = grp0 + g++;
                if (is_short) {
                    // goes whole into this bundle or the next, whichever ends nearer the (carried) target
                    if (bc.cur + nblk - bc.round_target() > bc.round_target() - bc.cur) bc.close();
                    bc.add(grp, 0, nblk, nblk);
                    if (bc.cur >= bc.round_target()) bc.close();
                    continue;
                }
                if (bc.cur >= bc.target) bc.close();        // (uncut groups may have filled the bundle past the exact target)
                int32_t pos = 0, parts = 0;
                const int32_t first_bundle = bc.n_bundles;
                while (pos < nblk && !bc.overflow) {
                    const int32_t take = (int32_t)std::min<int64_t>(nblk - pos, bc.target - bc.cur);
                    bc.add(grp, pos, pos + take, nblk);
                    pos += take;
                    ++parts;
                    if (bc.cur >= bc.target) bc.close();
                }
                if (parts > 1) bc.mark_split(grp, first_bundle, parts);
            }
        }
        bc.close();
        if (k != 1 || bc.overflow || bc.n_bundles <= W || attempt == 3) break;
        const int64_t wider = bc.target + std::max<int64_t>(1, bc.target / 32);
        bc = BundleCutter{bc.out, bc.max_bundles, bc.max_split, wider};
        bc.use_carry = true;
        }
        if (bc.overflow) return fail(ctx, PA_ERR_INVALID, "pa_plan: decode bundle / partial-slot list overflow");
    }
    const int32_t n_bundles = bc.n_bundles;
    const int64_t used = off_b + align_up((int64_t)n_bundles * sizeof(DecBundle), 256);

    const auto t_lists = std::chrono::steady_clock::now();
    // ---- upload
    uint8_t* ws = static_cast<uint8_t*>(d_workspace);
    cudaError_t e = cudaMemsetAsync(ws + ctx->off_counters, 0, (size_t)(ctx->off_plan - ctx->off_counters), stream);
    if (e == cudaSuccess && used > 0)
        e = cudaMemcpyAsync(ws + ctx->off_plan, h_stage, (size_t)used, cudaMemcpyHostToDevice, stream);
    if (e == cudaSuccess) e = cudaEventRecord(ctx->stage_ev[stage], stream);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "pa_plan(upload)");
    ctx->stage_pending[stage] = true;
    ctx->stage_next = (stage + 1) % pa_ctx::kStages;

    PlanView& v = ctx->view;
    v.queue = reinterpret_cast<int32_t*>(ws + ctx->off_counters);
    v.group_counters = v.queue + 16;
    v.tiles = reinterpret_cast<const PreTile*>(ws + ctx->off_plan);
    v.bundles = reinterpret_cast<const DecBundle*>(ws + ctx->off_plan + off_b);
    v.redo = reinterpret_cast<int2*>(ws + ctx->off_redo);
    v.part_ml = reinterpret_cast<float2*>(ws + ctx->off_part_ml);
    v.part_o = reinterpret_cast<float*>(ws + ctx->off_part_o);
    v.n_bundles = n_bundles;
    v.n_tiles = n_tiles;
    v.n_split = bc.n_split;
    v.n_units = n_units;
    v.head_groups = head_groups;
    {   // cumulative shares of the pieces in 1/256 (the last one is stored as 255 and read as 256)
        static const uint8_t kCum8[8] = {128, 179, 210, 228, 241, 249, 254, 255};
        uint64_t cum = 0;
        for (int l = 1; l <= levels; ++l) {
            const uint64_t cv = (l == levels) ? 255 : (levels == 8 ? kCum8[l - 1] : (uint64_t)(256 * l / levels));
            cum |= cv << (8 * (l - 1));
        }
        v.n_levels = levels;
        v.level_cum = cum;
    }
    int32_t dec_ctas = 0;
    if (n_bundles > 0) dec_ctas = std::min(sms - pre_ctas, n_bundles);
    ctx->decode_ctas = dec_ctas;
    ctx->prefill_ctas = pre_ctas;
    ctx->p_in_tmem = prefill_mode == 0;
    ctx->prefill_mode = prefill_mode;
    ctx->bundles_per_stream = k;
    ctx->n_levels = levels;
    ctx->n_items = bc.n_items;
    ctx->n_simple_tiles = prefill_mode == 2 ? n_tiles : 0;
    ctx->planned_n_tok = n_tok;
    ctx->launches_per_call = (dec_ctas + pre_ctas > 0) + (ctx->n_simple_tiles > 0);
    ctx->planned = true;
    ctx->plan_host_ns = std::chrono::duration_cast<std::chrono::nanoseconds>(std::chrono::steady_clock::now() - t_begin).count();
    ctx->plan_ns_validate = std::chrono::duration_cast<std::chrono::nanoseconds>(t_valid - t_begin).count();
    ctx->plan_ns_lists = std::chrono::duration_cast<std::chrono::nanoseconds>(t_lists - t_valid).count();
    return PA_OK;
}

int32_t pa_batch_attention(pa_ctx* ctx, const void* q, const void* k_pool, const void* v_pool, const int32_t* d_cu,
                           const int32_t* d_ctx, const int32_t* d_bt, float softmax_scale, void* out, void* stream) {
    if (!ctx) return PA_ERR_INVALID;
    if (!ctx->planned) return fail(ctx, PA_ERR_INVALID, "pa_batch_attention: no valid pa_plan");
    if (ctx->view.n_bundles == 0 && ctx->view.n_tiles == 0) return PA_OK;  // empty batch
    if (!q || !k_pool || !v_pool || !d_cu || !d_ctx || !d_bt || !out)
        return fail(ctx, PA_ERR_INVALID, "pa_batch_attention: null pointer");
    if (!(softmax_scale > 0.f) || !std::isfinite(softmax_scale))
        return fail(ctx, PA_ERR_INVALID, "pa_batch_attention: softmax_scale must be positive and finite");
    if (int32_t rc = check_device(ctx, "pa_batch_attention")) return rc;
    if (ctx->tm_k_ptr != k_pool) {
        int32_t rc = make_pool_map(ctx, k_pool, &ctx->tmK);
        for (int i = 0; i < 5 && rc == PA_OK; ++i) rc = make_pool_map5(ctx, k_pool, &ctx->tails.k[i], 16 >> i, i == 0 ? 2 : 1);
        if (rc != PA_OK) return rc;
        ctx->tm_k_ptr = k_pool;
    }
    if (ctx->tm_v_ptr != v_pool) {
        int32_t rc = make_pool_map(ctx, v_pool, &ctx->tmV);
        for (int i = 0; i < 5 && rc == PA_OK; ++i) rc = make_pool_map5(ctx, v_pool, &ctx->tails.v[i], 16 >> i, i == 0 ? 2 : 1);
        if (rc != PA_OK) return rc;
        ctx->tm_v_ptr = v_pool;
    }
    if (ctx->view.n_units > 0 && (ctx->tm_q_ptr != q || ctx->tm_q_ntok != ctx->planned_n_tok)) {
        int32_t rc = make_q_map(ctx, q, ctx->planned_n_tok, &ctx->tmQ);
        if (rc != PA_OK) return rc;
        ctx->tm_q_ptr = q;
        ctx->tm_q_ntok = ctx->planned_n_tok;
    }
    if (ctx->view.n_bundles > 0 && (ctx->tm_qd_ptr != q || ctx->tm_qd_ntok != ctx->planned_n_tok)) {
        int32_t rc = make_qdec_map(ctx, q, ctx->planned_n_tok, &ctx->tmQd);
        if (rc != PA_OK) return rc;
        ctx->tm_qd_ptr = q;
        ctx->tm_qd_ntok = ctx->planned_n_tok;
    }
    AttnLaunch a;
    a.sh = LaunchShape{ctx->cfg.num_q_heads, ctx->cfg.num_kv_heads, ctx->cfg.head_dim, ctx->cfg.max_blocks_per_seq};
    a.q = q; a.out = out; a.k_pool = k_pool; a.v_pool = v_pool;
    a.cu_seqlens_q = d_cu; a.context_lens = d_ctx; a.block_tables = d_bt;
    a.softmax_scale = softmax_scale;
    a.plan = ctx->view;
    a.decode_ctas = ctx->decode_ctas;
    a.prefill_ctas = ctx->prefill_ctas;
    a.p_in_tmem = ctx->p_in_tmem;
    a.n_simple_tiles = ctx->n_simple_tiles;
    a.tmQ = ctx->view.n_units > 0 ? &ctx->tmQ : nullptr;
    a.tmQd = ctx->view.n_bundles > 0 ? &ctx->tmQd : nullptr;
    a.tmK = &ctx->tmK; a.tmV = &ctx->tmV;
    a.tails = &ctx->tails;
    int launches = 0;
    cudaError_t e = launch_attention(a, static_cast<cudaStream_t>(stream), &launches);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "pa_batch_attention");
    return PA_OK;
}

int64_t pa_plan_info(const pa_ctx* ctx, int32_t which) {
    if (!ctx || !ctx->planned) return PA_ERR_INVALID;
    switch (which) {
        case 0: return ctx->n_items;
        case 1: return ctx->view.n_bundles;
        case 2: return ctx->view.n_split;
        case 3: return ctx->view.n_tiles;
        case 4: return ctx->decode_ctas + ctx->prefill_ctas;
        case 5: return ctx->launches_per_call;
        case 6: return ctx->prefill_ctas;
        case 7: return ctx->bundles_per_stream;
        case 8: return ctx->prefill_mode;
        case 9: return ctx->plan_host_ns;
        case 10: return ctx->n_levels;
        case 11: return ctx->plan_ns_validate;
        case 12: return ctx->plan_ns_lists;
#ifdef PA_TIMELINE
        case 100: return ctx->off_redo;     // development instrumentation (pa_prefill.cuh PA_TL)
#endif
        default: return PA_ERR_INVALID;
    }
}

// ---------------------------------------------------------------------------------------------
// a8 step timer and OLS fit  T = alpha + beta * n_tok  (R^2 per PAPER.md:L439)
// ---------------------------------------------------------------------------------------------
int32_t pa_timer_begin(pa_ctx* ctx, void* stream) {
    if (!ctx) return PA_ERR_INVALID;
    cudaError_t e = cudaEventRecord(ctx->t0, static_cast<cudaStream_t>(stream));
    return e == cudaSuccess ? PA_OK : cuda_fail(ctx, e, "pa_timer_begin");
}

int32_t pa_timer_record(pa_ctx* ctx, double r, int32_t n_tok, double seconds) {
    if (!ctx) return PA_ERR_INVALID;
    if (!(r >= 0.0 && r <= 1.0) || n_tok < 0 || !(seconds >= 0.0)) return fail(ctx, PA_ERR_INVALID, "pa_timer_record: bad sample");
    ctx->samples[(int)std::floor(r * 1000.0 + 0.5)][n_tok].push_back(seconds);
    return PA_OK;
}

int32_t pa_timer_end(pa_ctx* ctx, void* stream, double r, int32_t n_tok, double* seconds_out) {
    if (!ctx) return PA_ERR_INVALID;
    cudaError_t e = cudaEventRecord(ctx->t1, static_cast<cudaStream_t>(stream));
    if (e == cudaSuccess) e = cudaEventSynchronize(ctx->t1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, ctx->t0, ctx->t1);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "pa_timer_end");
    const double sec = (double)ms * 1e-3;
    if (seconds_out) *seconds_out = sec;
    return pa_timer_record(ctx, r, n_tok, sec);
}

int32_t pa_timer_fit(pa_ctx* ctx, double r, double* alpha, double* beta, double* r2, int32_t* n_points) {
    if (!ctx || !alpha || !beta || !r2) return PA_ERR_INVALID;
    auto it = ctx->samples.find((int)std::floor(r * 1000.0 + 0.5));
    const int32_t n = it == ctx->samples.end() ? 0 : (int32_t)it->second.size();
    if (n_points) *n_points = n;
    if (n < 2) return fail(ctx, PA_ERR_TIMER, "pa_timer_fit: fewer than 2 distinct n_tok for this r");
    std::vector<double> x, y;
    for (auto& kv : it->second) {
        x.push_back((double)kv.first);
        y.push_back(median(kv.second));
    }
    double xb = 0, yb = 0;
    for (int i = 0; i < n; ++i) { xb += x[i]; yb += y[i]; }
    xb /= n; yb /= n;
    double sxx = 0, sxy = 0;
    for (int i = 0; i < n; ++i) { sxx += (x[i] - xb) * (x[i] - xb); sxy += (x[i] - xb) * (y[i] - yb); }
    const double b = sxy / sxx, a = yb - b * xb;
    double ss_res = 0, ss_tot = 0;
    for (int i = 0; i < n; ++i) {
        const double e = y[i] - (a + b * x[i]);
        ss_res += e * e;
        ss_tot += (y[i] - yb) * (y[i] - yb);
    }
    *alpha = a;
    *beta = b;
    *r2 = ss_tot == 0.0 ? (ss_res == 0.0 ? 1.0 : 0.0) : 1.0 - ss_res / ss_tot;
    return PA_OK;
}

// N1: quadratic fit of K(r) at fixed n_tok and kappa = 2 c2 / (c0 + c1 + c2)  (App. A.3, Eq. 9-11)
int32_t pa_timer_kappa(pa_ctx* ctx, int32_t n_tok, double* c, double* kappa, int32_t* n_points) {
    if (!ctx || !c || !kappa) return PA_ERR_INVALID;
    std::vector<double> x, y;
    for (auto& rk : ctx->samples) {
        auto it = rk.second.find(n_tok);
        if (it == rk.second.end() || it->second.empty()) continue;
        x.push_back(rk.first / 1000.0);
        y.push_back(median(it->second));
    }
    const int n = (int)x.size();
    if (n_points) *n_points = n;
    if (n < 3) return fail(ctx, PA_ERR_TIMER, "pa_timer_kappa: fewer than 3 distinct r at this n_tok");
    // normal equations of the 3-parameter least squares, solved by Gaussian elimination with partial pivoting
    double A[3][4] = {{0, 0, 0, 0}, {0, 0, 0, 0}, {0, 0, 0, 0}};
    for (int i = 0; i < n; ++i) {
        const double p[3] = {1.0, x[i], x[i] * x[i]};
        for (int a = 0; a < 3; ++a) {
            for (int b = 0; b < 3; ++b) A[a][b] += p[a] * p[b];
            A[a][3] += p[a] * y[i];
        }
    }
    for (int col = 0; col < 3; ++col) {
        int piv = col;
        for (int r = col + 1; r < 3; ++r)
            if (std::fabs(A[r][col]) > std::fabs(A[piv][col])) piv = r;
        if (std::fabs(A[piv][col]) < 1e-300) return fail(ctx, PA_ERR_TIMER, "pa_timer_kappa: singular system");
        for (int k = 0; k < 4; ++k) std::swap(A[col][k], A[piv][k]);
        for (int r = 0; r < 3; ++r) {
            if (r == col) continue;
            const double f = A[r][col] / A[col][col];
            for (int k = col; k < 4; ++k) A[r][k] -= f * A[col][k];
        }
    }
    for (int a = 0; a < 3; ++a) c[a] = A[a][3] / A[a][a];
    const double k1 = c[0] + c[1] + c[2];
    if (k1 == 0.0) return fail(ctx, PA_ERR_TIMER, "pa_timer_kappa: K(1) == 0");
    *kappa = 2.0 * c[2] / k1;
    return PA_OK;
}

// N3: Eq. 3 (base threshold under CFR) and Eq. 7 (crossover condition) — PAPER.md:L117-127, L184-191
int32_t pa_crossover_theta0(double x, double* theta0, double* zeta) {
    if (!theta0 || !zeta || !(x > 0.0) || !std::isfinite(x)) return PA_ERR_INVALID;
    // f(t) = t/(1-t) + ln(1-t) - x is increasing on (0,1) from -x to +inf: Newton from above is monotone
    // (f is convex), safeguarded by the bracket; f'(t) = t/(1-t)^2
    double lo = 0.0, hi = 1.0, t = x < 0.5 ? std::min(0.999, std::sqrt(2.0 * x) + x) : 1.0 - 1.0 / (x + 2.0);
    for (int it = 0; it < 200; ++it) {
        const double f = t / (1.0 - t) + std::log1p(-t) - x;
        if (f < 0.0) lo = t; else hi = t;
        double tn = t - f * (1.0 - t) * (1.0 - t) / t;
        if (!(tn > lo && tn < hi)) tn = 0.5 * (lo + hi);
        if (std::fabs(tn - t) <= 1e-16 * t) { t = tn; break; }
        t = tn;
    }
    *theta0 = t;
    *zeta = -std::log1p(-t);
    return PA_OK;
}

int32_t pa_crossover_eq7(const double* in, double* out) {
    if (!in || !out) return PA_ERR_INVALID;
    const double ap = in[0], bp = in[1], ad = in[2], bd = in[3], amb = in[4], bmb = in[5], muL = in[6], muO = in[7],
                 zeta = in[8], k0 = in[9], N = in[10];
    const double tok = muL + muO;
    if (!(tok > 0.0) || !(k0 > 0.0) || !(N > 0.0)) return PA_ERR_INVALID;
    const double beta_w = (bp * muL + bd * muO) / tok;
    const double fixed_eb = (ap + ad * zeta * muO) / k0, fixed_mb = amb * (1.0 + muO) / N;
    out[0] = bmb - beta_w;
    out[1] = (fixed_eb - fixed_mb) / tok;
    out[2] = beta_w;
    out[3] = 1.0 / (fixed_eb + beta_w * tok);
    out[4] = 1.0 / (fixed_mb + bmb * tok);
    return PA_OK;
}

int32_t pa_timer_reset(pa_ctx* ctx) {
    if (!ctx) return PA_ERR_INVALID;
    ctx->samples.clear();
    return PA_OK;
}

}  // extern "C"
