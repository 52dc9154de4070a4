/*
 * pa.h — C ABI of libpa_b200.so: paged-KV-cache attention over a mixed batch of prefill chunks and
 * decode tokens on one NVIDIA B200 (sm_100a).
 *
 * What the operations are (citations: PAPER.md = arxiv/paper_2606_00516 text, by line):
 *   - One serving step processes n_tok tokens, a fraction r = n_decode / n_tok of them decode tokens
 *     (§1).  Its attention is what the paper blames for the exclusive-vs-mixed
 *     crossover: "GEMM time is largely invariant to r, whereas Attention time grows with r"
 *     (§1; L494 App. A.2 (ii)).
 *   - Decode attention "streams the full KV-cache context per token"; ctx = tokens
 *     already in a request's KV cache.  Prefill is chunked: a chunk of new tokens
 *     attends to the prompt's earlier KV (§2; L437 App. A.1).
 *   - The KV cache is paged in blocks of b tokens and addressed through block tables
 *     (PagedAttention "unchanged", §4.1; blocks/b in PAPER.md:L1094-1100 Eq. 23).
 *   - Step time is modelled as T_iter = alpha + beta * n_tok per decode ratio r,
 *     fit quality by R^2 (App. A.1).
 * The paper fixes no attention algorithm; DESIGN.md §2 lists the readings (softmax base e, a new
 * token attends to itself, bottom-right causal alignment, GQA head map h -> h / (Hq/Hkv)).
 *
 * Conventions for every call
 *   - "dev" pointers are device (HBM) addresses on cfg.device; "host" pointers are ordinary host
 *     memory.  The library never allocates device memory and never takes ownership of a buffer:
 *     the caller (PyTorch in this repo) owns pools, workspace, inputs and outputs.
 *   - bf16 tensors are dense, C order, 16-byte aligned base.  int32 index arrays are dense.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  All device work
 *     is enqueued on it; no call synchronises the device except pa_timer_end (on its own events).
 *     pa_plan stages its lists in a small ring of pinned host buffers and only waits (on an event of
 *     its own) when the buffer it is about to reuse still has an upload in flight, i.e. when more
 *     than 3 plans are outstanding on the device.  pa_kv_append, pa_batch_attention and pa_kv_gather only
 *     enqueue kernels and may be captured into a CUDA graph; pa_plan (a host-to-device upload from
 *     library-owned staging) and the pa_timer_* calls must NOT be called during stream capture.
 *   - The CUDA device current on the calling thread must be cfg.device for every call that takes a
 *     stream (PA_ERR_INVALID otherwise).  pa_create restores the caller's current device before it
 *     returns.  A context is not thread-safe: one thread at a time per pa_ctx; different contexts
 *     (also on different devices) may be used concurrently.
 *   - No environment variable is read.  Every tuning knob is a field of pa_config.
 *   - Return value: PA_OK or a negative PA_ERR_*; pa_last_error(ctx) gives a message.  No
 *     exceptions, no aborts, no printing.  Out-of-range block ids inside block tables are
 *     undefined behaviour (not validated on the device).
 *
 * Paged pool layout (contract): per K and per V one pool
 *       pool[num_blocks][num_kv_heads][block_size = 16][head_dim]     bf16
 *   Logical position t of sequence s lives in slot
 *       (block_tables[s * max_blocks_per_seq + t / 16],  t % 16).
 *   Table entries at index >= ceil(kv_len / 16) are never used as block ids (the row itself, all
 *   max_blocks_per_seq entries of it, must be readable: an entry may be loaded ahead of the check that
 *   discards it); slots at positions >= kv_len are never read into a result and never written.
 *
 * Batch convention: sequences [0, num_decode_seqs) are decode sequences (exactly one new token
 *   each), sequences [num_decode_seqs, n_seq) are prefill chunks (q_len >= 0 new tokens over
 *   context_lens[s] >= 0 cached ones).  cu_seqlens_q[s] is the first token row of sequence s in
 *   the packed [n_tok, ...] tensors; context_lens[s] counts tokens cached BEFORE this step.
 *   Query j of sequence s attends to keys 0 .. context_lens[s] + j (itself included), so
 *   pa_kv_append must run before pa_batch_attention on the same stream.
 */
#ifndef PA_B200_H
#define PA_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PA_OK 0
#define PA_ERR_INVALID (-1)     /* null / negative / non-monotone cu_seqlens / decode q_len != 1 / size mismatch */
#define PA_ERR_UNSUPPORTED (-2) /* head_dim not in {128,256}, block_size != 16, Hq % Hkv != 0, Hq/Hkv > 8 */
#define PA_ERR_WORKSPACE (-3)   /* workspace missing or too small */
#define PA_ERR_CUDA (-4)        /* CUDA runtime/driver error; text in pa_last_error */
#define PA_ERR_TIMER (-5)       /* fewer than 2 distinct n_tok recorded for that r */

/* flags for pa_config.flags */
#define PA_FLAG_DEBUG_SIMPLE 1u   /* debug: route every row through the plain one-warp-per-(row,head) CUDA kernel */
#define PA_FLAG_PREFILL_P_SMEM 2u /* prefill variant that stages P in shared memory instead of TMEM (default: TMEM) */

typedef struct pa_ctx pa_ctx; /* opaque; owns host plan scratch, pinned staging, CUDA events, timer samples */

typedef struct {
    int32_t num_q_heads;        /* Hq */
    int32_t num_kv_heads;       /* Hkv, divides Hq, Hq/Hkv <= 8 */
    int32_t head_dim;           /* D in {128, 256} */
    int32_t block_size;         /* b, must be 16 */
    int64_t num_blocks;         /* blocks in each of the K and V pools */
    int32_t max_seqs;           /* upper bound on n_seq of any batch */
    int32_t max_tokens;         /* upper bound on n_tok of any batch */
    int32_t max_blocks_per_seq; /* row stride of block_tables (entries) */
    int32_t device;             /* CUDA device ordinal */
    uint32_t flags;             /* PA_FLAG_* */
    /* planner tuning; 0 = the planner's own choice.  Effective values: pa_plan_info 6, 7. */
    int32_t tune_prefill_ctas;        /* CTAs that start in the prefill role of a mixed launch (clamped to [1, SMs-1]) */
    int32_t tune_bundles_per_stream;  /* decode bundles per persistent stream, 1..4 */
    int32_t tune_min_bundle_blocks;   /* smallest decode bundle, in 16-token blocks (default 2) */
    int32_t tune_levels;              /* guided hand-out of decode bundles: pieces per bundle, 1..8 (1 = whole bundles);
                                         effective value: pa_plan_info 10 */
} pa_config;

/* Create / destroy a context for one shape.  `out` host.  PA_ERR_UNSUPPORTED for shapes outside the
 * supported set, PA_ERR_INVALID for non-positive sizes, PA_ERR_CUDA if the device is unusable. */
int32_t pa_create(pa_ctx** out, const pa_config* cfg);
int32_t pa_destroy(pa_ctx* ctx);

/* Bytes the caller must allocate (dev, 256-byte aligned) and pass to pa_plan as workspace; and the
 * bytes of ONE pool (K or V) = num_blocks * Hkv * 16 * D * 2.  Negative on error. */
int64_t pa_workspace_bytes(const pa_ctx* ctx);
int64_t pa_kv_pool_bytes(const pa_ctx* ctx);

/* a3 kv_append ("KV-cache management"): for every sequence s, new token
 * j in [0, q_len_s), KV head g:  pool[slot(s, context_lens[s] + j)][g][:] = new[cu_seqlens_q[s] + j][g][:]
 * (bit copy) for K and V.  Every other pool byte is left untouched.
 *   k_new, v_new    dev bf16 [n_tok, Hkv, D]            (read)
 *   k_pool, v_pool  dev bf16 pools                      (written at the target slots only)
 *   d_cu_seqlens_q  dev int32 [n_seq + 1], d_context_lens dev int32 [n_seq],
 *   d_block_tables  dev int32 [n_seq, max_blocks_per_seq]
 * n_tok must equal cu_seqlens_q[n_seq] (not checked on the device).  n_seq == 0 or n_tok == 0: PA_OK, no launch.
 * Two appends to the same slot in one call are undefined. */
int32_t pa_kv_append(pa_ctx* ctx, const void* k_new, const void* v_new, void* k_pool, void* v_pool,
                     const int32_t* d_cu_seqlens_q, const int32_t* d_context_lens, const int32_t* d_block_tables,
                     int32_t n_seq, int32_t n_tok, void* stream);

/* a1 plan: validate the batch descriptor and build the work lists of the next
 * pa_batch_attention calls (decode KV segments balanced over the persistent workers, prefill tiles,
 * the CTA partition of the mixed launch) from HOST copies of the lengths; uploads them into
 * d_workspace on `stream`.  One plan serves any number of pa_batch_attention calls (e.g. one per
 * layer) on the same stream until the next pa_plan.
 *   h_cu_seqlens_q host int32 [n_seq + 1] non-decreasing from 0; h_context_lens host int32 [n_seq] >= 0
 *   d_workspace dev, >= pa_workspace_bytes(ctx) bytes, must stay allocated while the plan is in use.
 * Errors: PA_ERR_INVALID (n_seq > max_seqs, n_tok > max_tokens, decode seq with q_len != 1,
 * kv_len > max_blocks_per_seq * 16, ...), PA_ERR_WORKSPACE. */
int32_t pa_plan(pa_ctx* ctx, const int32_t* h_cu_seqlens_q, const int32_t* h_context_lens, int32_t n_seq,
                int32_t num_decode_seqs, void* d_workspace, int64_t workspace_bytes, void* stream);

/* a4-a7 batch_attention: for every token row i = cu_seqlens_q[s] + j and q head h
 *     out[i][h][:] = softmax_t( softmax_scale * q[i][h] . K_s[t][h / (Hq/Hkv)] ) V_s[t][h / (Hq/Hkv)],
 *     t = 0 .. context_lens[s] + j,   K_s/V_s read from the pools through block_tables,
 * bf16 inputs, fp32 accumulation, bf16 output rounded once.  Uses the last pa_plan of ctx; the
 * device descriptor arrays must describe the same batch as the planned host copies.
 * Range: any finite bf16 inputs.  The tensor-core prefill path exponentiates a 128-key tile against the running
 * maximum of the EARLIER tiles of the row; a row in which one tile's scores exceed everything before them by more
 * than 2^127 (88 nats) overflows that pass, is detected (its row sum is not finite) and is recomputed in the same
 * launch by a plain two-pass loop, so the result is the general softmax for such rows too (just slower).
 *   q    dev bf16 [n_tok, Hq, D] (read);  out dev bf16 [n_tok, Hq, D] (every planned row written)
 *   k_pool, v_pool dev bf16 pools (read only).
 * Decode rows run the split-KV path (partials in the workspace, merged in the same launch by the
 * last-arriving worker); prefill tiles run the tensor-core path; both in ONE launch. */
int32_t pa_batch_attention(pa_ctx* ctx, const void* q, const void* k_pool, const void* v_pool,
                           const int32_t* d_cu_seqlens_q, const int32_t* d_context_lens,
                           const int32_t* d_block_tables, float softmax_scale, void* out, void* stream);

/* a2 test hook: gather one sequence's logical KV through its block-table row (bit copy).
 *   d_block_table_row dev int32 [>= ceil(kv_len/16)];  k_out, v_out dev bf16 [kv_len, Hkv, D]. */
int32_t pa_kv_gather(pa_ctx* ctx, const void* k_pool, const void* v_pool, const int32_t* d_block_table_row,
                     int32_t kv_len, void* k_out, void* v_out, void* stream);

/* a8 step timer (T_iter = alpha + beta * n_tok per r): CUDA events on `stream` around
 * whatever the caller enqueues between begin and end (kv_append + batch_attention of one layer, DESIGN R17).
 * pa_timer_end waits for its own end event, returns the elapsed seconds in *seconds_out (host) and
 * records the sample (r quantised to integer per-mille, n_tok, seconds).
 * pa_timer_fit: ordinary least squares over the per-n_tok MEDIANS recorded for that r (DESIGN R19):
 * alpha [s], beta [s/token], R^2, and the number of distinct n_tok; PA_ERR_TIMER with < 2 distinct n_tok. */
int32_t pa_timer_begin(pa_ctx* ctx, void* stream);
int32_t pa_timer_end(pa_ctx* ctx, void* stream, double r, int32_t n_tok, double* seconds_out);
int32_t pa_timer_record(pa_ctx* ctx, double r, int32_t n_tok, double seconds); /* add an externally timed sample */
int32_t pa_timer_fit(pa_ctx* ctx, double r, double* alpha, double* beta, double* r2, int32_t* n_points);
/* pa_timer_kappa (App. A.3, Eq. 9-11; L550-554 App. A.4): least-squares quadratic
 * K(r) = c0 + c1 r + c2 r^2 through the per-r MEDIAN step times recorded at this n_tok (one point per distinct r key,
 * r = key/1000), and the interference convexity index kappa = 2 c2 / (c0 + c1 + c2).  c[3] and kappa are host
 * outputs (seconds / dimensionless); *n_points = distinct r keys used.  PA_ERR_TIMER with < 3 distinct r, or if the
 * normal equations are singular or c0 + c1 + c2 == 0.  The gap of Eq. 10, K(r) - [(1-r)K(0) + rK(1)], is
 * -c2 r (1 - r).  Host arithmetic only (fp64); no device work. */
int32_t pa_timer_kappa(pa_ctx* ctx, int32_t n_tok, double* c, double* kappa, int32_t* n_points);
int32_t pa_timer_reset(pa_ctx* ctx);

/* N3 (Prop. 3.1 Eq. 3-4, L184-191 Prop. 3.4 Eq. 7): scalar host arithmetic (fp64)
 * on fitted coefficients; no device work, ctx may be NULL.
 * pa_crossover_theta0: the base CFR threshold theta0 in (0,1) solving theta0/(1-theta0) + ln(1-theta0) = x with
 *   x = p0*alpha_p/alpha_d > 0, and zeta = -ln(1-theta0).  PA_ERR_INVALID for x <= 0 or non-finite.
 * pa_crossover_eq7: in[11] = {alpha_p, beta_p, alpha_d, beta_d, alpha_MB, beta_MB^e, mu_L, mu_O, zeta, k0*, N};
 *   out[5] = {LHS = beta_MB^e - beta_EB^w,  RHS = [(alpha_p + alpha_d zeta mu_O)/k0* - alpha_MB(1+mu_O)/N]/(mu_L+mu_O),
 *             beta_EB^w = (beta_p mu_L + beta_d mu_O)/(mu_L+mu_O),  TP_EB(k0*, N) (Eq. 4),  TP_MB(N)}.
 *   Mixed batching wins iff LHS < RHS.  PA_ERR_INVALID unless mu_L + mu_O > 0, k0* > 0, N > 0. */
int32_t pa_crossover_theta0(double x, double* theta0, double* zeta);
int32_t pa_crossover_eq7(const double* in, double* out);

/* Introspection of the last plan (host ints; for bench.py's launch accounting and the tests).
 * which: 0 decode work items, 1 decode bundles, 2 split (partial-writing) items, 3 prefill tiles,
 *        4 CTAs in the attention launch, 5 kernel launches per pa_batch_attention call,
 *        6 CTAs given the prefill role in the mixed launch, 7 decode bundles per stream (effective),
 *        8 prefill variant (0 P in TMEM, 1 P in shared memory, 2 plain kernel),
 *        9 host nanoseconds the last pa_plan call took (validation + lists + enqueue of the upload),
 *        10 pieces a decode bundle is handed out in (guided hand-out; 1 = whole bundles),
 *        11 / 12 nanoseconds of (9) spent validating the descriptor / building the tile and bundle lists. */
int64_t pa_plan_info(const pa_ctx* ctx, int32_t which);

/* Library-owned message of the last error on ctx (valid until the next call on ctx); "" if none. */
const char* pa_last_error(const pa_ctx* ctx);

/* ---- Allocation-free decode attention (for callers that cannot call cudaMalloc: code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it).  Needs no pa_ctx, no workspace and no pa_plan.
 *
 * pa_decode_attention_static: the decode rows of pa_batch_attention (a5/a6; "Decode attention streams the full
 * KV-cache context per token") for a batch of n_seq decode sequences, one new token each: token row s
 * belongs to sequence s and attends to keys 0 .. context_lens[s] (its own KV already appended to the pools):
 *     out[s][h][:] = softmax_t( softmax_scale * q[s][h] . K_s[t][h / (Hq/Hkv)] ) V_s[t][h / (Hq/Hkv)]
 * bf16 in, fp32 accumulate, bf16 out; split-KV with the merge in the same launch, by a plain one-warp-per-
 * (sequence, q head, split) kernel (correct, not tuned: pa_batch_attention is the fast path).
 *   q, out           dev bf16 [n_seq, Hq, D];  k_pool, v_pool dev bf16 pools (layout above, read only)
 *   d_context_lens   dev int32 [n_seq];  d_block_tables dev int32 [n_seq, max_blocks_per_seq]
 *   max_kv_len       host upper bound on context_lens[s] + 1 (only chooses the split count; <= max_blocks_per_seq*16)
 *   device           CUDA ordinal; must be the calling thread's current device;  stream as for every other call
 * Scratch: the split partials and the merge's arrival counters live in a file-scope __device__ array of
 * PA_STATIC_SCRATCH_BYTES that every GPU that loads the library holds until the process exits.  The call calls no
 * cudaMalloc / cudaFree / allocating routine: it enqueues one cudaMemsetAsync (the counters, which must start at
 * zero; the array keeps the previous call's contents) and one kernel on `stream`.  The first call on a device also
 * looks up the array's device address (cudaGetSymbolAddress), so make one call per device outside stream capture.
 * Size limit: n_seq * Hq * (D*4 + 12) bytes (each of its three pieces rounded up to 256) must fit
 * PA_STATIC_SCRATCH_BYTES — about 1000 sequences of Hq = 32, D = 128; up to 32 KV splits are used when they fit.
 * Beyond it: PA_ERR_WORKSPACE, nothing enqueued.  ALL calls on a device share the array: calls that may overlap on the GPU (different streams, or
 * different host threads without ordering between their streams) race on it; calls on one stream are ordered and safe.
 * Errors: PA_ERR_INVALID / PA_ERR_UNSUPPORTED (same shape rules as pa_create) / PA_ERR_WORKSPACE / PA_ERR_CUDA;
 * pa_static_last_error() gives the calling thread's message ("" if its last call succeeded).  n_seq == 0: PA_OK. */
#define PA_STATIC_SCRATCH_BYTES (16 * 1024 * 1024)
int32_t pa_decode_attention_static(const void* q, const void* k_pool, const void* v_pool,
                                   const int32_t* d_context_lens, const int32_t* d_block_tables, int32_t n_seq,
                                   int32_t num_q_heads, int32_t num_kv_heads, int32_t head_dim,
                                   int32_t max_blocks_per_seq, int32_t max_kv_len, float softmax_scale, void* out,
                                   int32_t device, void* stream);
int64_t pa_static_scratch_bytes(void);        /* = PA_STATIC_SCRATCH_BYTES of the loaded library */
const char* pa_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PA_B200_H */
