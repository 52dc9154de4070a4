/*
 * ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path.
 *
 * Plain, slow, fp64 CPU statement of what the paged mixed-batch attention path computes,
 * written from the paper's problem statement and SURVEY.md §8(c) — NOT from the CUDA code,
 * with which it shares no source, header, table or helper.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md at build time; cited by line):
 *   - ctx = "the number of tokens already accumulated in each decode request's KV cache: at
 *     ctx = c, every decode token must stream c key-value pairs" (App. A.2)
 *     -> context_lens[s] counts tokens cached BEFORE this step.
 *   - decode attention "streams the full KV-cache context per token" (§1).
 *   - chunked prefill: a chunk of new tokens attends to the prompt's earlier KV
 *     (§2; L437 App. A.1).
 *   - PagedAttention is left unchanged (§4.1); KV blocks of size b
 *     (Eq. 23).
 *   - T_iter = alpha + beta * n_tok (§1), fit quality by R^2.
 * The paper states no attention algorithm; the readings R1-R8 of SURVEY.md §8(c) (listed in
 * DESIGN.md) fix: softmax base e over scale*q.k; a new token attends to itself (append, then
 * attend over ctx+j+1 keys); bottom-right causal alignment; q head h -> KV head h / (Hq/Hkv).
 *
 * Because tiling, online softmax, split-KV and merge are exact re-associations of the textbook
 * result, the oracle for attention IS the textbook definition (step 3 below), in fp64 on the
 * same bf16 inputs (bf16 -> fp64 widening is exact).
 *
 * Documented pool layout (a boundary contract, include/pa.h): per K and per V
 *     pool[block][kv_head][slot_in_block][d],  bf16, C order,
 * and slot(s, t) = (block_tables[s][t / b], t % b).
 *
 * Parity pins: every function here is pinned by tests/test_oracle_pins.py (P1-P15; oracle_theta0 and
 * oracle_eq7 by the hand-worked golden tests/golden/eq7_closed_forms.txt, the Eq. 3 residual and the
 * throughput identity of Proposition 3.4) — nothing is "parity unpinned".
 *
 * Threading (pthread) only distributes independent (token row, q head) items to host cores for
 * the timed cpu_baseline; each item is computed by the plain loop in attend_row_head().
 */
#include <math.h>
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct {
    int32_t num_q_heads, num_kv_heads, head_dim, block_size;
    int32_t max_blocks_per_seq; /* row stride of block_tables */
} oracle_shape;

/* exact bf16 -> fp64 (format widening: bf16 is the top 16 bits of an IEEE fp32) */
static double bf16_to_f64(uint16_t b) {
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

/* physical element offset of (seq s, logical position t, kv head g, dim 0) in a pool */
static int64_t slot_offset(const oracle_shape* sh, const int32_t* block_tables, int32_t s, int64_t t, int32_t g) {
    int64_t blk = block_tables[(int64_t)s * sh->max_blocks_per_seq + t / sh->block_size];
    int64_t within = t % sh->block_size;
    return ((blk * sh->num_kv_heads + g) * sh->block_size + within) * (int64_t)sh->head_dim;
}

/* Step 1: append.  For each seq s (batch order), each new token j, each KV head g:
 * pool[slot(s, ctx_s + j)][g][:] = new[cu_s + j][g][:]  (bit copy), same for V. */
int32_t oracle_kv_append(const oracle_shape* sh, const uint16_t* k_new, const uint16_t* v_new, uint16_t* k_pool,
                         uint16_t* v_pool, const int32_t* cu_seqlens_q, const int32_t* context_lens,
                         const int32_t* block_tables, int32_t n_seq) {
    for (int32_t s = 0; s < n_seq; ++s) {
        int32_t q_len = cu_seqlens_q[s + 1] - cu_seqlens_q[s];
        for (int32_t j = 0; j < q_len; ++j) {
            int64_t row = (int64_t)cu_seqlens_q[s] + j;
            for (int32_t g = 0; g < sh->num_kv_heads; ++g) {
                int64_t dst = slot_offset(sh, block_tables, s, (int64_t)context_lens[s] + j, g);
                int64_t src = (row * sh->num_kv_heads + g) * (int64_t)sh->head_dim;
                for (int32_t d = 0; d < sh->head_dim; ++d) {
                    k_pool[dst + d] = k_new[src + d];
                    v_pool[dst + d] = v_new[src + d];
                }
            }
        }
    }
    return 0;
}

/* Step 2: gather.  K_s[t][g][:] = pool[slot(s, t)][g][:] for t in [0, kv_len). */
int32_t oracle_kv_gather(const oracle_shape* sh, const uint16_t* k_pool, const uint16_t* v_pool,
                         const int32_t* block_tables, int32_t s, int32_t kv_len, uint16_t* k_out, uint16_t* v_out) {
    for (int64_t t = 0; t < kv_len; ++t)
        for (int32_t g = 0; g < sh->num_kv_heads; ++g) {
            int64_t src = slot_offset(sh, block_tables, s, t, g);
            int64_t dst = (t * sh->num_kv_heads + g) * (int64_t)sh->head_dim;
            for (int32_t d = 0; d < sh->head_dim; ++d) {
                k_out[dst + d] = k_pool[src + d];
                v_out[dst + d] = v_pool[src + d];
            }
        }
    return 0;
}

/* Step 3 for one (token row, q head), restricted to keys [key_lo, key_hi) of the
 * n_j = ctx_s + j + 1 visible keys (the full row is key_lo = 0, key_hi = n_j):
 *   z_t = scale * sum_d q[d] K_s[t][g][d];  m = max_t z_t;  w_t = exp(z_t - m);  l = sum_t w_t;
 *   o_un[:] = sum_t w_t V_s[t][g][:].
 * Returns m, l, and o_un (unnormalised).  w (optional, length key_hi-key_lo) receives w_t. */
static void attend_partial(const oracle_shape* sh, const uint16_t* q, const uint16_t* k_pool, const uint16_t* v_pool,
                           const int32_t* block_tables, int32_t s, int64_t row, int32_t h, int64_t key_lo,
                           int64_t key_hi, double scale, double* z_scratch, double* m_out, double* l_out,
                           double* o_un, double* w_out) {
    const int32_t D = sh->head_dim;
    const int32_t G = sh->num_q_heads / sh->num_kv_heads;
    const int32_t g = h / G; /* R4: contiguous GQA groups */
    const uint16_t* qv = q + (row * sh->num_q_heads + h) * (int64_t)D;
    double m = -INFINITY;
    for (int64_t t = key_lo; t < key_hi; ++t) {
        const uint16_t* kv = k_pool + slot_offset(sh, block_tables, s, t, g);
        double dot = 0.0;
        for (int32_t d = 0; d < D; ++d) dot += bf16_to_f64(qv[d]) * bf16_to_f64(kv[d]);
        double z = scale * dot;
        z_scratch[t - key_lo] = z;
        if (z > m) m = z;
    }
    double l = 0.0;
    for (int32_t d = 0; d < D; ++d) o_un[d] = 0.0;
    for (int64_t t = key_lo; t < key_hi; ++t) {
        double w = exp(z_scratch[t - key_lo] - m);
        if (w_out) w_out[t - key_lo] = w;
        l += w;
        const uint16_t* vv = v_pool + slot_offset(sh, block_tables, s, t, g);
        for (int32_t d = 0; d < D; ++d) o_un[d] += w * bf16_to_f64(vv[d]);
    }
    *m_out = m;
    *l_out = l;
}

/* sequence owning global token row `row` (cu_seqlens_q is non-decreasing; empty seqs skipped) */
static int32_t seq_of_row(const int32_t* cu_seqlens_q, int32_t n_seq, int64_t row) {
    int32_t s = 0;
    while (s < n_seq && !(cu_seqlens_q[s] <= row && row < cu_seqlens_q[s + 1])) ++s;
    return s;
}

typedef struct {
    const oracle_shape* sh;
    const uint16_t *q, *k_pool, *v_pool;
    const int32_t *cu_seqlens_q, *context_lens, *block_tables;
    int32_t n_seq;
    double scale;
    const int64_t* rows; /* token rows to compute */
    int64_t n_rows;
    double* out;         /* [n_rows][Hq][D] */
    double* lse;         /* optional [n_rows][Hq] */
    int64_t next;        /* work counter: item = row_index * Hq + h */
    pthread_mutex_t mu;
    int64_t max_keys;
} attn_job;

static void* attn_worker(void* arg) {
    attn_job* job = (attn_job*)arg;
    const oracle_shape* sh = job->sh;
    const int32_t Hq = sh->num_q_heads, D = sh->head_dim;
    double* z = (double*)malloc(sizeof(double) * (size_t)(job->max_keys > 0 ? job->max_keys : 1));
    double* o_un = (double*)malloc(sizeof(double) * (size_t)D);
    for (;;) {
        pthread_mutex_lock(&job->mu);
        int64_t item = job->next++;
        pthread_mutex_unlock(&job->mu);
        if (item >= job->n_rows * Hq) break;
        int64_t ri = item / Hq;
        int32_t h = (int32_t)(item % Hq);
        int64_t row = job->rows[ri];
        int32_t s = seq_of_row(job->cu_seqlens_q, job->n_seq, row);
        int64_t j = row - job->cu_seqlens_q[s];
        int64_t n_j = (int64_t)job->context_lens[s] + j + 1; /* R2/R3: keys 0 .. ctx+j inclusive */
        double m, l;
        attend_partial(sh, job->q, job->k_pool, job->v_pool, job->block_tables, s, row, h, 0, n_j, job->scale, z, &m,
                       &l, o_un, NULL);
        double* o = job->out + (ri * Hq + h) * (int64_t)D;
        for (int32_t d = 0; d < D; ++d) o[d] = o_un[d] / l;
        if (job->lse) job->lse[ri * Hq + h] = m + log(l);
    }
    free(z);
    free(o_un);
    return NULL;
}

/* Attention (step 3) for the listed token rows, all q heads.  out[i][h][:] for rows[i].
 * n_threads <= 1 runs inline.  Returns the number of threads used, or <0 on error. */
int32_t oracle_attention_rows(const oracle_shape* sh, const uint16_t* q, const uint16_t* k_pool, const uint16_t* v_pool,
                              const int32_t* cu_seqlens_q, const int32_t* context_lens, const int32_t* block_tables,
                              int32_t n_seq, double scale, const int64_t* rows, int64_t n_rows, double* out,
                              double* lse, int32_t n_threads) {
    attn_job job;
    job.sh = sh; job.q = q; job.k_pool = k_pool; job.v_pool = v_pool;
    job.cu_seqlens_q = cu_seqlens_q; job.context_lens = context_lens; job.block_tables = block_tables;
    job.n_seq = n_seq; job.scale = scale; job.rows = rows; job.n_rows = n_rows; job.out = out; job.lse = lse;
    job.next = 0;
    job.max_keys = 0;
    for (int32_t s = 0; s < n_seq; ++s) {
        int64_t kv = (int64_t)context_lens[s] + (cu_seqlens_q[s + 1] - cu_seqlens_q[s]);
        if (kv > job.max_keys) job.max_keys = kv;
    }
    for (int64_t i = 0; i < n_rows; ++i)
        if (rows[i] < 0 || rows[i] >= cu_seqlens_q[n_seq]) return -1;
    pthread_mutex_init(&job.mu, NULL);
    if (n_threads < 1) n_threads = 1;
    if (n_threads > 256) n_threads = 256;
    if (n_threads == 1) {
        attn_worker(&job);
    } else {
        pthread_t th[256];
        for (int32_t i = 0; i < n_threads; ++i) pthread_create(&th[i], NULL, attn_worker, &job);
        for (int32_t i = 0; i < n_threads; ++i) pthread_join(th[i], NULL);
    }
    pthread_mutex_destroy(&job.mu);
    return n_threads;
}

/* Weights p_t = w_t / l (length n_j) and lse of one (row, head): for the softmax pins. */
int32_t oracle_attention_weights(const oracle_shape* sh, const uint16_t* q, const uint16_t* k_pool,
                                 const uint16_t* v_pool, const int32_t* cu_seqlens_q, const int32_t* context_lens,
                                 const int32_t* block_tables, int32_t n_seq, double scale, int64_t row, int32_t h,
                                 double* p_out, int64_t p_capacity, double* lse_out) {
    int32_t s = seq_of_row(cu_seqlens_q, n_seq, row);
    if (s >= n_seq) return -1;
    int64_t n_j = (int64_t)context_lens[s] + (row - cu_seqlens_q[s]) + 1;
    if (p_capacity < n_j) return -1;
    double* z = (double*)malloc(sizeof(double) * (size_t)n_j);
    double* o_un = (double*)malloc(sizeof(double) * (size_t)sh->head_dim);
    double m, l;
    attend_partial(sh, q, k_pool, v_pool, block_tables, s, row, h, 0, n_j, scale, z, &m, &l, o_un, p_out);
    for (int64_t t = 0; t < n_j; ++t) p_out[t] /= l;
    if (lse_out) *lse_out = m + log(l);
    free(z);
    free(o_un);
    return (int32_t)n_j;
}

/* Split-KV partial: (m, l, unnormalised o[D]) of one (row, head) over keys
 * [key_lo, key_hi) of its visible keys. */
int32_t oracle_attention_partial(const oracle_shape* sh, const uint16_t* q, const uint16_t* k_pool,
                                 const uint16_t* v_pool, const int32_t* cu_seqlens_q, const int32_t* context_lens,
                                 const int32_t* block_tables, int32_t n_seq, double scale, int64_t row, int32_t h,
                                 int64_t key_lo, int64_t key_hi, double* m_out, double* l_out, double* o_un) {
    int32_t s = seq_of_row(cu_seqlens_q, n_seq, row);
    if (s >= n_seq) return -1;
    int64_t n_j = (int64_t)context_lens[s] + (row - cu_seqlens_q[s]) + 1;
    if (key_lo < 0 || key_hi > n_j || key_lo >= key_hi) return -1;
    double* z = (double*)malloc(sizeof(double) * (size_t)(key_hi - key_lo));
    attend_partial(sh, q, k_pool, v_pool, block_tables, s, row, h, key_lo, key_hi, scale, z, m_out, l_out, o_un, NULL);
    free(z);
    return 0;
}

/* Merge (flash-decoding combine):
 *   m = max_i m_i;  l = sum_i l_i e^{m_i - m};  o = (sum_i o_i e^{m_i - m}) / l. */
int32_t oracle_merge(int32_t n_parts, int32_t D, const double* m_i, const double* l_i, const double* o_i /*[n][D]*/,
                     double* o_out, double* lse_out) {
    double m = -INFINITY;
    for (int32_t i = 0; i < n_parts; ++i)
        if (m_i[i] > m) m = m_i[i];
    double l = 0.0;
    for (int32_t d = 0; d < D; ++d) o_out[d] = 0.0;
    for (int32_t i = 0; i < n_parts; ++i) {
        double f = exp(m_i[i] - m);
        l += l_i[i] * f;
        for (int32_t d = 0; d < D; ++d) o_out[d] += o_i[(int64_t)i * D + d] * f;
    }
    for (int32_t d = 0; d < D; ++d) o_out[d] /= l;
    if (lse_out) *lse_out = m + log(l);
    return 0;
}

/* Step 4: OLS line T = alpha + beta n (R^2 per PAPER.md:L439).
 *   beta = sum (n_i - nbar)(T_i - Tbar) / sum (n_i - nbar)^2;  alpha = Tbar - beta nbar;
 *   R^2 = 1 - SS_res / SS_tot  (R^2 := 1 when SS_tot = 0 and SS_res = 0).
 * Returns -5 when fewer than 2 distinct n (the line is undetermined). */
int32_t oracle_fit(const double* n, const double* T, int32_t count, double* alpha, double* beta, double* r2) {
    if (count < 2) return -5;
    double nbar = 0.0, Tbar = 0.0;
    for (int32_t i = 0; i < count; ++i) { nbar += n[i]; Tbar += T[i]; }
    nbar /= count; Tbar /= count;
    double sxx = 0.0, sxy = 0.0;
    for (int32_t i = 0; i < count; ++i) {
        sxx += (n[i] - nbar) * (n[i] - nbar);
        sxy += (n[i] - nbar) * (T[i] - Tbar);
    }
    if (sxx == 0.0) return -5;
    double b = sxy / sxx, a = Tbar - b * nbar;
    double ss_res = 0.0, ss_tot = 0.0;
    for (int32_t i = 0; i < count; ++i) {
        double e = T[i] - (a + b * n[i]);
        ss_res += e * e;
        ss_tot += (T[i] - Tbar) * (T[i] - Tbar);
    }
    *alpha = a;
    *beta = b;
    *r2 = (ss_tot == 0.0) ? (ss_res == 0.0 ? 1.0 : 0.0) : 1.0 - ss_res / ss_tot;
    return 0;
}

/* Quadratic least squares K(r) = c0 + c1 r + c2 r^2 and the interference convexity index
 * kappa = 2 c2 / (c0 + c1 + c2)  (App. A.3, Eq. 10-11).  Normal equations
 * solved by Cramer's rule on the 3x3 moment matrix.  Returns -5 with < 3 distinct r. */
int32_t oracle_quadratic_kappa(const double* r, const double* K, int32_t count, double* c /*[3]*/, double* kappa) {
    if (count < 3) return -5;
    double s[5] = {0, 0, 0, 0, 0}, t[3] = {0, 0, 0};
    for (int32_t i = 0; i < count; ++i) {
        double p = 1.0;
        for (int k = 0; k < 5; ++k) { s[k] += p; if (k < 3) t[k] += p * K[i]; p *= r[i]; }
    }
    double a[3][3] = {{s[0], s[1], s[2]}, {s[1], s[2], s[3]}, {s[2], s[3], s[4]}};
    double det = a[0][0] * (a[1][1] * a[2][2] - a[1][2] * a[2][1]) - a[0][1] * (a[1][0] * a[2][2] - a[1][2] * a[2][0]) +
                 a[0][2] * (a[1][0] * a[2][1] - a[1][1] * a[2][0]);
    if (fabs(det) < 1e-300) return -5;
    for (int col = 0; col < 3; ++col) {
        double b[3][3];
        for (int i = 0; i < 3; ++i)
            for (int j = 0; j < 3; ++j) b[i][j] = (j == col) ? t[i] : a[i][j];
        double dc = b[0][0] * (b[1][1] * b[2][2] - b[1][2] * b[2][1]) - b[0][1] * (b[1][0] * b[2][2] - b[1][2] * b[2][0]) +
                    b[0][2] * (b[1][0] * b[2][1] - b[1][1] * b[2][0]);
        c[col] = dc / det;
    }
    *kappa = 2.0 * c[2] / (c[0] + c[1] + c[2]);
    return 0;
}

/* Base threshold under CFR (§3.2.1, Proposition 3.1, Eq. 3): theta0 is the unique
 * solution in (0, 1) of
 *     theta0 / (1 - theta0) + ln(1 - theta0) = x,        x = p0 * alpha_p / alpha_d > 0,
 * and zeta = -ln(1 - theta0).  The left side is 0 at theta0 = 0, increasing (derivative
 * theta0 / (1 - theta0)^2 > 0) and unbounded as theta0 -> 1, so plain bisection on (0, 1) finds it.
 * Returns -1 for x <= 0 or non-finite x. */
int32_t oracle_theta0(double x, double* theta0, double* zeta) {
    if (!(x > 0.0) || !isfinite(x)) return -1;
    double lo = 0.0, hi = 1.0;
    for (int it = 0; it < 200; ++it) {
        double mid = 0.5 * (lo + hi);
        if (mid <= lo || mid >= hi) break;
        double f = mid / (1.0 - mid) + log(1.0 - mid) - x;
        if (f < 0.0) lo = mid; else hi = mid;
    }
    *theta0 = 0.5 * (lo + hi);
    *zeta = -log(1.0 - *theta0);
    return 0;
}

/* Crossover condition, Proposition 3.4 / Eq. 7 (§3.5):  TP_MB(N) > TP_EB(k0*, N)  iff
 *     beta_MB^e - beta_EB^w  <  1/(mu_L + mu_O) * [ (alpha_p + alpha_d zeta mu_O) / k0*  -  alpha_MB (1 + mu_O) / N ],
 * with beta_EB^w = (beta_p mu_L + beta_d mu_O) / (mu_L + mu_O)  (below the TP_EB formula).
 * Outputs: lhs (the marginal-cost gap), rhs (the amortised fixed-cost advantage of MB), beta_EB^w, and the two
 * throughputs the proposition compares, written out from their own formulas:
 *     TP_EB(k0*, N) = [ (alpha_p + alpha_d zeta mu_O) / k0*  +  beta_EB^w (mu_L + mu_O) ]^-1      (Eq. 4)
 *     TP_MB(N)      = [ alpha_MB (1 + mu_O) / N  +  beta_MB^e (mu_L + mu_O) ]^-1
 * Returns -1 unless mu_L + mu_O > 0, k0 > 0, N > 0. */
int32_t oracle_eq7(double alpha_p, double beta_p, double alpha_d, double beta_d, double alpha_mb, double beta_mb_e,
                   double mu_L, double mu_O, double zeta, double k0, double N,
                   double* lhs, double* rhs, double* beta_eb_w, double* tp_eb, double* tp_mb) {
    if (!(mu_L + mu_O > 0.0) || !(k0 > 0.0) || !(N > 0.0)) return -1;
    double bw = (beta_p * mu_L + beta_d * mu_O) / (mu_L + mu_O);
    *beta_eb_w = bw;
    *lhs = beta_mb_e - bw;
    *rhs = ((alpha_p + alpha_d * zeta * mu_O) / k0 - alpha_mb * (1.0 + mu_O) / N) / (mu_L + mu_O);
    *tp_eb = 1.0 / ((alpha_p + alpha_d * zeta * mu_O) / k0 + bw * (mu_L + mu_O));
    *tp_mb = 1.0 / (alpha_mb * (1.0 + mu_O) / N + beta_mb_e * (mu_L + mu_O));
    return 0;
}
