/*
 * cp_oracle.c -- CPU float64 ORACLE for paged decode attention on a shared KV pool.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, helper or table with the CUDA library under
 * paper_2606_24506_b200/ and neither includes the other.
 *
 * What it is: the plain DEFINITION of the result, written out.
 * The paper (CrossPool, arxiv 2606.24506) does not define an attention kernel: it
 * keeps "existing SGLang attention kernels ... over a paged KV-cache abstraction"
 * (§4) and contributes the problem statement -- a shared pool of
 * fixed-size KV pages behind "a uniform paged KV-cache interface" with "a logical KV
 * address space" (§3.1; L122), for KV-head-limited attention, MQA /
 * few-head GQA / MLA (§2.2), decode only, one new token per request
 * (PAPER.md:L160).  The arithmetic is the textbook softmax(q K^T * scale) V of the
 * works it cites ([34] MQA, [1] GQA, [12] MLA, [23] PagedAttention), with the shapes
 * of BASELINE.json.  Because the split-KV method on the GPU reaches exactly this result
 * up to rounding order, the oracle is the two-pass definition: no online softmax, no
 * blocking, no rounding of probabilities.
 *
 * Layout (reading R1): the arena is num_pages pages of page_bytes.  One
 * page holds page_tokens tokens of ONE kv head: K block [P][d_k] bf16 row-major, then
 * V block [P][d_v] bf16.  MLA: a single block [P][d_k]; V is the first d_v entries of
 * the same row.  A request's page list is page-major: page_ids[lp * Hkv + c] is the
 * physical page of logical page lp, kv head c.  Query head h uses kv head
 * c = h / (Hq / Hkv) (reading A2).
 *
 * Pins (tests/test_oracle_pins.py): single token, identical keys, two tokens, V
 * shift/scale, page permutation, split count, batch independence / poison, brute-force
 * dense numpy float64 on tiny shapes, GQA = replicated MQA, MLA = KV kind with V
 * aliasing K, golden vectors G1/G2 (exact rational dot products), gather round trip.
 * The paper prints no value on this path, so every pin is derived from the mathematics
 * ("parity unpinned" w.r.t. the paper).
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC cp_oracle.c -o libcp_oracle.so -lm
 * (-ffp-contract=off: every product and sum is a separately rounded float64 operation.)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define CPO_OK 0
#define CPO_ERR_ARG (-1)
#define CPO_ERR_MEM (-2)

enum { CPO_KIND_KV = 0, CPO_KIND_MLA = 1 };

/* exact bf16 -> binary32 -> binary64 */
static double bf16_to_double(uint16_t b)
{
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, sizeof f);
    return (double)f;
}

/* address (in uint16 units) of row `slot` of the K (is_v = 0) or V (is_v = 1) block of
 * physical page pid.  MLA has a single block; is_v selects the same row. */
static uint64_t row_offset_u16(uint32_t page_tokens, uint32_t page_bytes, int kind,
                               int d_k, int d_v, int32_t pid, uint32_t slot, int is_v)
{
    uint64_t base = (uint64_t)pid * (page_bytes / 2u);
    if (kind == CPO_KIND_MLA)
        return base + (uint64_t)slot * (uint64_t)d_k;
    if (!is_v)
        return base + (uint64_t)slot * (uint64_t)d_k;
    return base + (uint64_t)page_tokens * (uint64_t)d_k + (uint64_t)slot * (uint64_t)d_v;
}

int cpo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * Translation + gather (hot-path step a2): copy the 16-bit patterns of tokens
 * 0..context_len-1 into k_out [T][Hkv][d_k] and v_out [T][Hkv][d_v].
 * MLA: k_out is C [T][d_k]; v_out (may be NULL) receives C[:, :d_v].
 */
int cpo_gather(const uint16_t *arena, uint32_t page_tokens, uint32_t page_bytes, uint32_t num_pages,
               int kind, int n_kv_heads, int d_k, int d_v,
               const int32_t *page_ids, int n_page_ids, int context_len,
               uint16_t *k_out, uint16_t *v_out)
{
    if (!arena || !page_ids || !k_out || page_tokens == 0 || context_len < 1 || n_kv_heads < 1)
        return CPO_ERR_ARG;
    if (kind == CPO_KIND_MLA && n_kv_heads != 1)
        return CPO_ERR_ARG;
    int n_lp = (context_len + (int)page_tokens - 1) / (int)page_tokens;
    if (n_page_ids < n_lp * n_kv_heads)
        return CPO_ERR_ARG;
    for (int i = 0; i < n_lp * n_kv_heads; ++i)
        if (page_ids[i] < 0 || (uint32_t)page_ids[i] >= num_pages)
            return CPO_ERR_ARG;
    for (int t = 0; t < context_len; ++t) {
        int lp = t / (int)page_tokens;
        uint32_t slot = (uint32_t)(t % (int)page_tokens);
        for (int c = 0; c < n_kv_heads; ++c) {
            int32_t pid = page_ids[lp * n_kv_heads + c];
            uint64_t ko = row_offset_u16(page_tokens, page_bytes, kind, d_k, d_v, pid, slot, 0);
            memcpy(k_out + ((uint64_t)t * n_kv_heads + c) * d_k, arena + ko, (size_t)d_k * 2);
            if (v_out) {
                uint64_t vo = row_offset_u16(page_tokens, page_bytes, kind, d_k, d_v, pid, slot, 1);
                memcpy(v_out + ((uint64_t)t * n_kv_heads + c) * d_v, arena + vo, (size_t)d_v * 2);
            }
        }
    }
    return CPO_OK;
}

/*
 * KV append (the step right before attention in every decode iteration:
 * "physical KV pages [are mapped] on demand ... kept until their decode requests finish",
 * PAPER.md:L122): write the rows of ONE new token at position `pos` (= the context length before
 * the append) of a request: k_new [Hkv][d_k], v_new [Hkv][d_v] (MLA: k_new is the latent row
 * [d_k], v_new is ignored).  The page list must already cover logical page pos / P.  Only the
 * 16-bit patterns move; everything else in the arena stays untouched.
 */
int cpo_append(uint16_t *arena, uint32_t page_tokens, uint32_t page_bytes, uint32_t num_pages,
               int kind, int n_kv_heads, int d_k, int d_v,
               const int32_t *page_ids, int n_page_ids, int pos,
               const uint16_t *k_new, const uint16_t *v_new)
{
    if (!arena || !page_ids || !k_new || page_tokens == 0 || pos < 0 || n_kv_heads < 1)
        return CPO_ERR_ARG;
    if (kind == CPO_KIND_MLA && n_kv_heads != 1)
        return CPO_ERR_ARG;
    if (kind != CPO_KIND_MLA && !v_new)
        return CPO_ERR_ARG;
    int lp = pos / (int)page_tokens;
    uint32_t slot = (uint32_t)(pos % (int)page_tokens);
    if (n_page_ids < (lp + 1) * n_kv_heads)
        return CPO_ERR_ARG;
    for (int c = 0; c < n_kv_heads; ++c) {
        int32_t pid = page_ids[lp * n_kv_heads + c];
        if (pid < 0 || (uint32_t)pid >= num_pages)
            return CPO_ERR_ARG;
        uint64_t ko = row_offset_u16(page_tokens, page_bytes, kind, d_k, d_v, pid, slot, 0);
        memcpy(arena + ko, k_new + (uint64_t)c * d_k, (size_t)d_k * 2);
        if (kind != CPO_KIND_MLA) {
            uint64_t vo = row_offset_u16(page_tokens, page_bytes, kind, d_k, d_v, pid, slot, 1);
            memcpy(arena + vo, v_new + (uint64_t)c * d_v, (size_t)d_v * 2);
        }
    }
    return CPO_OK;
}

/* Attention of ONE query head over the token range [t0, t1) of one request, by the
 * definition: s_t = sigma * sum_i q_i k_{t,i} (i ascending); m = max_t s_t;
 * p_t = exp(s_t - m); l = sum_t p_t (t ascending); O_j = (sum_t p_t v_{t,j}) / l;
 * LSE = m + ln l.  `s` is scratch for t1 - t0 doubles. */
static void head_range(const uint16_t *arena, uint32_t page_tokens, uint32_t page_bytes, int kind,
                       int n_kv_heads, int d_k, int d_v, const int32_t *page_ids, int c,
                       const uint16_t *q_row, double sigma, int t0, int t1,
                       double *s, double *out, double *lse)
{
    int n = t1 - t0;
    double m = -INFINITY;
    for (int t = t0; t < t1; ++t) {
        int lp = t / (int)page_tokens;
        uint32_t slot = (uint32_t)(t % (int)page_tokens);
        int32_t pid = page_ids[lp * n_kv_heads + c];
        const uint16_t *k = arena + row_offset_u16(page_tokens, page_bytes, kind, d_k, d_v, pid, slot, 0);
        double acc = 0.0;
        for (int i = 0; i < d_k; ++i)
            acc += bf16_to_double(q_row[i]) * bf16_to_double(k[i]);
        double st = sigma * acc;
        s[t - t0] = st;
        if (st > m)
            m = st;
    }
    double l = 0.0;
    for (int j = 0; j < d_v; ++j)
        out[j] = 0.0;
    for (int t = t0; t < t1; ++t) {
        double p = exp(s[t - t0] - m);
        l += p;
        int lp = t / (int)page_tokens;
        uint32_t slot = (uint32_t)(t % (int)page_tokens);
        int32_t pid = page_ids[lp * n_kv_heads + c];
        const uint16_t *v = arena + row_offset_u16(page_tokens, page_bytes, kind, d_k, d_v, pid, slot, 1);
        for (int j = 0; j < d_v; ++j)
            out[j] += p * bf16_to_double(v[j]);
    }
    for (int j = 0; j < d_v; ++j)
        out[j] /= l;
    *lse = m + log(l);
    (void)n;
}

/*
 * Decode attention of one request (hot-path steps a2..a6 as ONE definition).
 *   q        bf16 [Hq][d_k];  heads_sel: which query heads to compute (NULL = all, then
 *   n_sel = Hq);  out double [n_sel][d_v];  lse double [n_sel] (natural log, scale inside).
 *   n_splits <= 1: the definition over all T tokens.
 *   n_splits  > 1: the logical pages are cut into n_splits contiguous ranges
 *                  [floor(s*n_lp/ns), floor((s+1)*n_lp/ns)), (lse_s, O_s) computed per
 *                  non-empty range by the same formulas, then combined
 *                  LSE = M + ln sum_s e^{lse_s - M},  O = sum_s e^{lse_s - LSE} O_s
 *                  (used only by the split-invariance pin P6).
 */
int cpo_attention(const uint16_t *arena, uint32_t page_tokens, uint32_t page_bytes, uint32_t num_pages,
                  int kind, int n_q_heads, int n_kv_heads, int d_k, int d_v, float softmax_scale,
                  const int32_t *page_ids, int n_page_ids, int context_len,
                  const uint16_t *q, const int32_t *heads_sel, int n_sel, int n_splits,
                  double *out, double *lse)
{
    if (!arena || !page_ids || !q || !out || !lse || page_tokens == 0)
        return CPO_ERR_ARG;
    if (context_len < 1 || n_q_heads < 1 || n_kv_heads < 1 || n_q_heads % n_kv_heads != 0)
        return CPO_ERR_ARG;
    if (kind == CPO_KIND_MLA && (n_kv_heads != 1 || d_v > d_k))
        return CPO_ERR_ARG;
    int n_lp = (context_len + (int)page_tokens - 1) / (int)page_tokens;
    if (n_page_ids < n_lp * n_kv_heads)
        return CPO_ERR_ARG;
    for (int i = 0; i < n_lp * n_kv_heads; ++i)
        if (page_ids[i] < 0 || (uint32_t)page_ids[i] >= num_pages)
            return CPO_ERR_ARG;
    if (!heads_sel)
        n_sel = n_q_heads;
    for (int k = 0; heads_sel && k < n_sel; ++k)
        if (heads_sel[k] < 0 || heads_sel[k] >= n_q_heads)
            return CPO_ERR_ARG;
    const int g = n_q_heads / n_kv_heads;
    const double sigma = (double)softmax_scale;
    int failed = 0;

#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < n_sel; ++k) {
        int h = heads_sel ? heads_sel[k] : k;
        int c = h / g;
        const uint16_t *q_row = q + (uint64_t)h * d_k;
        double *s = (double *)malloc(sizeof(double) * (size_t)context_len);
        if (!s) {
#pragma omp atomic write
            failed = 1;
            continue;
        }
        if (n_splits <= 1) {
            head_range(arena, page_tokens, page_bytes, kind, n_kv_heads, d_k, d_v, page_ids, c,
                       q_row, sigma, 0, context_len, s, out + (uint64_t)k * d_v, lse + k);
        } else {
            double *o_s = (double *)malloc(sizeof(double) * (size_t)n_splits * (size_t)d_v);
            double *lse_s = (double *)malloc(sizeof(double) * (size_t)n_splits);
            int *live = (int *)malloc(sizeof(int) * (size_t)n_splits);
            if (!o_s || !lse_s || !live) {
#pragma omp atomic write
                failed = 1;
                free(o_s); free(lse_s); free(live); free(s);
                continue;
            }
            double M = -INFINITY;
            for (int sp = 0; sp < n_splits; ++sp) {
                int p0 = (int)(((int64_t)sp * n_lp) / n_splits);
                int p1 = (int)(((int64_t)(sp + 1) * n_lp) / n_splits);
                int t0 = p0 * (int)page_tokens;
                int t1 = p1 * (int)page_tokens;
                if (t1 > context_len)
                    t1 = context_len;
                live[sp] = t1 > t0;
                if (!live[sp])
                    continue;
                head_range(arena, page_tokens, page_bytes, kind, n_kv_heads, d_k, d_v, page_ids, c,
                           q_row, sigma, t0, t1, s, o_s + (uint64_t)sp * d_v, lse_s + sp);
                if (lse_s[sp] > M)
                    M = lse_s[sp];
            }
            double z = 0.0;
            for (int sp = 0; sp < n_splits; ++sp)
                if (live[sp])
                    z += exp(lse_s[sp] - M);
            double L = M + log(z);
            double *o = out + (uint64_t)k * d_v;
            for (int j = 0; j < d_v; ++j)
                o[j] = 0.0;
            for (int sp = 0; sp < n_splits; ++sp) {
                if (!live[sp])
                    continue;
                double w = exp(lse_s[sp] - L);
                for (int j = 0; j < d_v; ++j)
                    o[j] += w * o_s[(uint64_t)sp * d_v + j];
            }
            lse[k] = L;
            free(o_s); free(lse_s); free(live);
        }
        free(s);
    }
    return failed ? CPO_ERR_MEM : CPO_OK;
}

/* ==========================================================================================
 * KV-cache planner (Eq. (1)-(2)).  TEST INFRASTRUCTURE, as
 * everything in this file.  Written out term by term in the paper's order and notation:
 *
 *   Q_i(u)     = (O_p,i + O_d,i * u / T_i) * 1{0 <= u < T_i}            active KV tokens at age u
 *   K_M(t)     = sum_i kappa(M) * Q_i(t - A_i)                          Eq. (1)
 *   K_pool(t)  = sum_M K_M(t)                                           Eq. (2)
 *
 * and the "P95/P99 trace-driven Monte Carlo quantile" (L112): K_pool evaluated at random
 * observation times t_n over the trace (the draws are an INPUT), then the empirical quantile;
 * "the planner rounds memory to pages and sets the shared KV-cache pool page budget".
 * Readings: u / T_i is computed before the product with O_d,i; each term
 * kappa * Q is rounded and added in trace order, models in index order; the empirical quantile
 * is the order statistic x_(k), k = ceil(q * N) (1-based, no interpolation -- the conservative
 * side); pages = ceil(K_q / page_bytes).
 * Pins (tests/test_oracle_pins.py P14-P18): a request worked by hand and its interval ends; the
 * exact time integral kappa * sum_i T_i (O_p,i + O_d,i / 2); linearity over models; the quantile
 * against a sort on small vectors and its special cases; Little's law on a long Poisson trace.
 * ========================================================================================== */

/* Eq. (1), first line. */
double cpo_active_tokens(double u, double o_p, double o_d, double t_res)
{
    if (!(u >= 0.0 && u < t_res)) return 0.0;
    return o_p + o_d * (u / t_res);
}

/* Eq. (1)-(2) at n_t observation times.  Model M owns trace entries [offs[M], offs[M+1]). */
int cpo_pool_demand(int n_models, const int64_t *offs, const double *kappa, const double *arrival,
                    const double *o_p, const double *o_d, const double *t_res, int64_t n_t,
                    const double *t_obs, double *k_pool)
{
    if (n_models < 0 || n_t < 0) return -1;
    for (int64_t n = 0; n < n_t; ++n) {
        double pool = 0.0;
        for (int m = 0; m < n_models; ++m) {
            double k_m = 0.0;
            for (int64_t i = offs[m]; i < offs[m + 1]; ++i)
                k_m += kappa[m] * cpo_active_tokens(t_obs[n] - arrival[i], o_p[i], o_d[i], t_res[i]);
            pool += k_m;
        }
        k_pool[n] = pool;
    }
    return 0;
}

static int cmp_double(const void *a, const void *b)
{
    const double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}

/* Empirical quantile: x_(k) with k = ceil(q * n), clamped to 1 .. n.  scratch: n doubles. */
int cpo_quantile(const double *x, int64_t n, double q, double *scratch, double *out)
{
    if (n < 1 || !(q > 0.0 && q <= 1.0)) return -1;
    for (int64_t i = 0; i < n; ++i) scratch[i] = x[i];
    qsort(scratch, (size_t)n, sizeof(double), cmp_double);
    int64_t k = (int64_t)ceil(q * (double)n);
    if (k < 1) k = 1;
    if (k > n) k = n;
    *out = scratch[k - 1];
    return 0;
}

/* "rounds memory to pages": pages that hold k_bytes. */
int64_t cpo_page_budget(double k_bytes, double page_bytes)
{
    return (int64_t)ceil(k_bytes / page_bytes);
}
