/*
 * sparrow_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, fp64 CPU statement of what Sparrow's sparse decode attention
 * computes, step by step in the order of SURVEY.md section 8(c) (O1..O8), which
 * restates the paper's decode step (Eq. 3: "landmark scores"
 * -> Top-k -> attention over the KV budget B = pagesize x num_pages
 * "pagesize-num_page"; dense while the context fits the budget)
 * with BASELINE.json north_star's default selector (per-channel key min/max page
 * summaries, upper-bound score, always-kept sink and local-window pages, top-k of
 * the remaining pages to fill B(L)).  Readings R1..R20 of DESIGN.md apply.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may call this.  It shares no code, header, table or helper with
 * the CUDA library under paper_2606_08446_b200/csrc; the structs below are the
 * oracle's own.
 *
 * Conventions
 *   - bf16 tensors arrive as raw uint16 bit patterns (exactly what the GPU reads)
 *     and are widened to double exactly; everything after that is double.
 *   - K and V pools: [n_phys_pages][Hkv][P][D] (P = page size 16, D = head dim 128,
 *     but P and D are plain parameters here).
 *   - q: [n][Hq][D]; query head h belongs to kv-head g = h / r, r = Hq / Hkv.
 *   - page_table: [n][max_pages] int32, logical page -> physical page.
 *   - L = cached length of a sequence INCLUDING the current token (R6).
 *   - No blocking, fusion or reordering: loops are written as the definitions read.
 *     The only parallelism is an OpenMP "for" over independent (sequence, kv-head)
 *     units in the *_step drivers, used when the oracle is timed as cpu_baseline.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): numpy brute force on tiny inputs,
 * closed-form budget values (tests/golden/), planted pages, q = 0 tie-break,
 * dense == sparse when B >= L, softmax rows sum to 1, chunked LSE merge == single
 * pass, Quest upper-bound invariant.  "parity unpinned": the paper's own tau=0.86
 * schedule tables (values exist only in figures) -- kind TABLE is pinned only for
 * its lookup rule, not for the paper's numbers.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ---------------------------------------------------------------- bf16 ---- */
static double bf16_to_f64(uint16_t b)
{
    uint32_t u = ((uint32_t)b) << 16;
    float f;
    memcpy(&f, &u, 4);
    return (double)f;
}

/* ------------------------------------------------------------ schedule ---- */
/* Oracle's own schedule description (R3).  kind: 0 DENSE, 1 FIXED, 2 CLAMP_FRAC,
 * 3 LINEAR_FRAC, 4 TABLE (budget in pages per length bin, 2K bins). */
typedef struct {
    int32_t kind;
    int32_t sink_tokens;   /* S */
    int32_t local_tokens;  /* W */
    int64_t fixed_tokens;  /* FIXED: B */
    int64_t floor_tokens;  /* CLAMP_FRAC / LINEAR_FRAC: lower clamp of B */
    int64_t f0_ppm;        /* keep fraction in parts per million (at L0 for LINEAR) */
    int64_t f1_ppm;        /* LINEAR: keep fraction at L1 */
    int64_t L0, L1;        /* LINEAR: fraction interpolated on clamp(L, L0, L1) */
    const int32_t *table_pages; /* TABLE: budget in pages for bin b = floor((L-1)/bin_tokens) */
    int32_t table_len;
    int32_t bin_tokens;
} oracle_schedule;

/* O2: B(L) in tokens, exact integer arithmetic (R3), clamped to [.., L]. */
int64_t oracle_budget_tokens(const oracle_schedule *s, int64_t L, int64_t page_size)
{
    int64_t B;
    if (s->kind == 0) {
        B = L;
    } else if (s->kind == 1) {
        B = s->fixed_tokens;
    } else if (s->kind == 2) {
        B = (L * s->f0_ppm) / 1000000;             /* floor(L * frac) */
        if (B < s->floor_tokens) B = s->floor_tokens;
    } else if (s->kind == 3) {
        int64_t Lc = L;
        if (Lc < s->L0) Lc = s->L0;
        if (Lc > s->L1) Lc = s->L1;
        /* frac(L) = f0 - (f0 - f1) * (Lc - L0) / (L1 - L0);  B = floor(L * frac) */
        int64_t num = s->f0_ppm * (s->L1 - s->L0) - (s->f0_ppm - s->f1_ppm) * (Lc - s->L0);
        int64_t den = 1000000 * (s->L1 - s->L0);
        B = (int64_t)(((__int128)L * (__int128)num) / (__int128)den);
        if (B < s->floor_tokens) B = s->floor_tokens;
    } else { /* TABLE: the paper's native form, a page count per length bin */
        int64_t b = (L - 1) / s->bin_tokens;
        if (b < 0) b = 0;
        if (b >= s->table_len) b = s->table_len - 1;
        B = (int64_t)s->table_pages[b] * page_size;  /* B = pagesize x num_pages */
    }
    if (B > L) B = L;
    return B;
}

static int64_t ceil_div(int64_t a, int64_t b) { return (a + b - 1) / b; }

/* O2 (second half): K_pages = min(ceil(B / P), n_pages)  (R4). */
int64_t oracle_k_pages(const oracle_schedule *s, int64_t L, int64_t page_size)
{
    int64_t n_pages = ceil_div(L, page_size);
    int64_t K = ceil_div(oracle_budget_tokens(s, L, page_size), page_size);
    return K < n_pages ? K : n_pages;
}

/* O3: forced pages F = sink pages  U  local-window pages  U  {last page}  (R7, R8, R9).
 * forced[p] in {0,1} for p < n_pages; returns |F|. */
int64_t oracle_forced_pages(int64_t L, int64_t S, int64_t W, int64_t page_size, uint8_t *forced)
{
    int64_t n_pages = ceil_div(L, page_size);
    int64_t cnt = 0;
    int64_t n_sink = ceil_div(S, page_size);               /* R8 */
    int64_t lo_tok = L - W; if (lo_tok < 0) lo_tok = 0;
    int64_t first_local = lo_tok / page_size;              /* R7: every page overlapping the last W tokens */
    for (int64_t p = 0; p < n_pages; ++p) {
        int f = 0;
        if (p < n_sink) f = 1;
        if (W > 0 && p >= first_local) f = 1;
        if (p == n_pages - 1) f = 1;                       /* last page always kept */
        forced[p] = (uint8_t)f;
        cnt += f;
    }
    return cnt;
}

/* ----------------------------------------------------------- summaries ---- */
/* O1: per (page, kv-head, channel) min and max of K over the page's valid tokens.
 * k_cache [n_phys][Hkv][P][D] bf16 bits; for update u: page_ids[u], n_valid[u] (NULL = P).
 * out [n_update][Hkv][2][D] double, [..][0][d] = min, [..][1][d] = max. */
void oracle_summarize(const uint16_t *k_cache, const int32_t *page_ids, const int32_t *n_valid,
                      int64_t n_update, int64_t Hkv, int64_t P, int64_t D, double *out)
{
    for (int64_t u = 0; u < n_update; ++u) {
        int64_t valid = n_valid ? n_valid[u] : P;
        for (int64_t g = 0; g < Hkv; ++g) {
            const uint16_t *tile = k_cache + (((int64_t)page_ids[u] * Hkv + g) * P) * D;
            double *mn = out + ((u * Hkv + g) * 2 + 0) * D;
            double *mx = out + ((u * Hkv + g) * 2 + 1) * D;
            for (int64_t d = 0; d < D; ++d) {
                double lo = INFINITY, hi = -INFINITY;
                for (int64_t t = 0; t < valid; ++t) {
                    double x = bf16_to_f64(tile[t * D + d]);
                    if (x < lo) lo = x;
                    if (x > hi) hi = x;
                }
                mn[d] = lo;
                mx[d] = hi;
            }
        }
    }
}

/* ------------------------------------------------------------- scoring ---- */
/* O5 for one (sequence, kv-head g): s[p] for EVERY logical page p < n_pages
 * (forced ones included -- the caller ignores them):
 *   s[p] = sum_{h in g} sum_d max(q[h][d]*mn[p][d], q[h][d]*mx[p][d])      (unscaled, R12)
 * mn/mx taken over the valid tokens of the page (R9). */
void oracle_scores_unit(const uint16_t *q_seq /* [Hq][D] */, const uint16_t *k_cache,
                        const int32_t *pt_row, int64_t L, int64_t g,
                        int64_t Hq, int64_t Hkv, int64_t P, int64_t D, double *s)
{
    int64_t r = Hq / Hkv;
    int64_t n_pages = ceil_div(L, P);
    for (int64_t p = 0; p < n_pages; ++p) {
        int64_t valid = (p == n_pages - 1) ? (L - P * p) : P;
        const uint16_t *tile = k_cache + (((int64_t)pt_row[p] * Hkv + g) * P) * D;
        double acc = 0.0;
        for (int64_t h = g * r; h < (g + 1) * r; ++h) {
            for (int64_t d = 0; d < D; ++d) {
                double lo = INFINITY, hi = -INFINITY;
                for (int64_t t = 0; t < valid; ++t) {
                    double x = bf16_to_f64(tile[t * D + d]);
                    if (x < lo) lo = x;
                    if (x > hi) hi = x;
                }
                double qv = bf16_to_f64(q_seq[h * D + d]);
                double a = qv * lo, b = qv * hi;
                acc += (a > b) ? a : b;
            }
        }
        s[p] = acc;
    }
}

/* --------------------------------------------------------------- top-k ---- */
typedef struct { double s; int32_t p; } cand_t;
static int cand_cmp(const void *a, const void *b)
{
    const cand_t *x = (const cand_t *)a, *y = (const cand_t *)b;
    if (x->s > y->s) return -1;           /* score descending */
    if (x->s < y->s) return 1;
    return (x->p > y->p) - (x->p < y->p);  /* ties: lower page index first (R10) */
}

/* O4, O6, O7 for one (sequence, kv-head): given scores s[p], forced flags and K_pages,
 * write Sel (ascending logical pages) and return |Sel|; *tau = score of the k-th candidate
 * (NaN when k == 0 or the sequence is dense). */
int64_t oracle_select_unit(const double *s, const uint8_t *forced, int64_t n_pages, int64_t K_pages,
                           int32_t *sel, double *tau)
{
    *tau = NAN;
    if (K_pages >= n_pages) {                 /* R13: dense, select all pages, no scoring */
        for (int64_t p = 0; p < n_pages; ++p) sel[p] = (int32_t)p;
        return n_pages;
    }
    int64_t n_forced = 0, n_cand = 0;
    cand_t *c = (cand_t *)malloc(sizeof(cand_t) * (size_t)(n_pages > 0 ? n_pages : 1));
    uint8_t *in = (uint8_t *)calloc((size_t)(n_pages > 0 ? n_pages : 1), 1);
    for (int64_t p = 0; p < n_pages; ++p) {
        if (forced[p]) { in[p] = 1; ++n_forced; }
        else { c[n_cand].s = s[p]; c[n_cand].p = (int32_t)p; ++n_cand; }
    }
    int64_t k = K_pages - n_forced;           /* R2: the budget includes the forced pages */
    if (k < 0) k = 0;
    if (k > n_cand) k = n_cand;
    qsort(c, (size_t)n_cand, sizeof(cand_t), cand_cmp);
    for (int64_t i = 0; i < k; ++i) in[c[i].p] = 1;
    if (k > 0) *tau = c[k - 1].s;
    int64_t m = 0;
    for (int64_t p = 0; p < n_pages; ++p) if (in[p]) sel[m++] = (int32_t)p;   /* O7 ascending */
    free(c);
    free(in);
    return m;
}

/* ----------------------------------------------------------- attention ---- */
/* O8 for one (sequence, kv-head g) over the logical pages pages[0..n_sel):
 *   z_t = sm_scale * q[h].K_t   for tokens t of those pages with global index < L
 *   p = softmax(z);  out[h] = sum_t p_t V_t;  lse[h] = ln sum_t exp(z_t)
 * out_g [r][D], lse_g [r]; probs_g (optional, may be NULL): [r][n_sel*P], masked slots = 0.
 * A unit with no valid token gives out = 0, lse = -inf. */
void oracle_attention_unit(const uint16_t *q_seq, const uint16_t *k_cache, const uint16_t *v_cache,
                           const int32_t *pt_row, int64_t L, const int32_t *pages, int64_t n_sel,
                           int64_t g, int64_t Hq, int64_t Hkv, int64_t P, int64_t D, double sm_scale,
                           double *out_g, double *lse_g, double *probs_g)
{
    int64_t r = Hq / Hkv;
    int64_t n_tok = n_sel * P;
    double *z = (double *)malloc(sizeof(double) * (size_t)(n_tok > 0 ? n_tok : 1));
    for (int64_t j = 0; j < r; ++j) {
        int64_t h = g * r + j;
        double m = -INFINITY;
        for (int64_t i = 0; i < n_sel; ++i) {
            const uint16_t *kt = k_cache + (((int64_t)pt_row[pages[i]] * Hkv + g) * P) * D;
            for (int64_t t = 0; t < P; ++t) {
                int64_t pos = (int64_t)pages[i] * P + t;
                double dot = 0.0;
                if (pos < L) {
                    for (int64_t d = 0; d < D; ++d)
                        dot += bf16_to_f64(q_seq[h * D + d]) * bf16_to_f64(kt[t * D + d]);
                    z[i * P + t] = dot * sm_scale;
                    if (z[i * P + t] > m) m = z[i * P + t];
                } else {
                    z[i * P + t] = -INFINITY;      /* masked: beyond the cached length (R9) */
                }
            }
        }
        double denom = 0.0;
        for (int64_t i = 0; i < n_tok; ++i)
            if (z[i] != -INFINITY) denom += exp(z[i] - m);
        for (int64_t d = 0; d < D; ++d) out_g[j * D + d] = 0.0;
        for (int64_t i = 0; i < n_sel; ++i) {
            const uint16_t *vt = v_cache + (((int64_t)pt_row[pages[i]] * Hkv + g) * P) * D;
            for (int64_t t = 0; t < P; ++t) {
                double pr = (z[i * P + t] != -INFINITY) ? exp(z[i * P + t] - m) / denom : 0.0;
                if (probs_g) probs_g[j * n_tok + i * P + t] = pr;
                if (pr != 0.0)
                    for (int64_t d = 0; d < D; ++d)
                        out_g[j * D + d] += pr * bf16_to_f64(vt[t * D + d]);
            }
        }
        lse_g[j] = (denom > 0.0) ? m + log(denom) : -INFINITY;
    }
    free(z);
}

/* a6 (partial form) for one (sequence, kv-head g) and one chunk of pages: the un-normalised
 * running state of SURVEY 8(a) a6:  m = max_t z_t,  l = sum_t exp(z_t - m),
 * o = sum_t exp(z_t - m) V_t.  An empty chunk gives m = -inf, l = 0, o = 0. */
void oracle_attention_partial_unit(const uint16_t *q_seq, const uint16_t *k_cache, const uint16_t *v_cache,
                                   const int32_t *pt_row, int64_t L, const int32_t *pages, int64_t n_sel,
                                   int64_t g, int64_t Hq, int64_t Hkv, int64_t P, int64_t D, double sm_scale,
                                   double *m_g /*[r]*/, double *l_g /*[r]*/, double *o_g /*[r][D]*/)
{
    int64_t r = Hq / Hkv;
    for (int64_t j = 0; j < r; ++j) {
        int64_t h = g * r + j;
        double m = -INFINITY;
        for (int pass = 0; pass < 2; ++pass) {
            if (pass == 1) { l_g[j] = 0.0; for (int64_t d = 0; d < D; ++d) o_g[j * D + d] = 0.0; }
            for (int64_t i = 0; i < n_sel; ++i) {
                const uint16_t *kt = k_cache + (((int64_t)pt_row[pages[i]] * Hkv + g) * P) * D;
                const uint16_t *vt = v_cache + (((int64_t)pt_row[pages[i]] * Hkv + g) * P) * D;
                for (int64_t t = 0; t < P; ++t) {
                    if ((int64_t)pages[i] * P + t >= L) continue;
                    double dot = 0.0;
                    for (int64_t d = 0; d < D; ++d)
                        dot += bf16_to_f64(q_seq[h * D + d]) * bf16_to_f64(kt[t * D + d]);
                    double zt = dot * sm_scale;
                    if (pass == 0) { if (zt > m) m = zt; }
                    else {
                        double e = exp(zt - m);
                        l_g[j] += e;
                        for (int64_t d = 0; d < D; ++d) o_g[j * D + d] += e * bf16_to_f64(vt[t * D + d]);
                    }
                }
            }
        }
        m_g[j] = m;
    }
}

/* a7: log-sum-exp merge of n_part partial states of ONE query head:
 *   m = max_i m_i;  l = sum_i l_i e^{m_i - m};  o = sum_i o_i e^{m_i - m} / l;  lse = m + ln l.
 * Partials with l_i = 0 (m_i = -inf) are skipped (they contribute nothing and must not make NaN). */
void oracle_lse_merge(const double *m_i, const double *l_i, const double *o_i /*[n_part][D]*/,
                      int64_t n_part, int64_t D, double *out /*[D]*/, double *lse)
{
    double m = -INFINITY;
    for (int64_t i = 0; i < n_part; ++i) if (l_i[i] > 0.0 && m_i[i] > m) m = m_i[i];
    double l = 0.0;
    for (int64_t d = 0; d < D; ++d) out[d] = 0.0;
    for (int64_t i = 0; i < n_part; ++i) {
        if (!(l_i[i] > 0.0)) continue;
        double w = exp(m_i[i] - m);
        l += l_i[i] * w;
        for (int64_t d = 0; d < D; ++d) out[d] += o_i[i * D + d] * w;
    }
    if (l > 0.0) {
        for (int64_t d = 0; d < D; ++d) out[d] /= l;
        *lse = m + log(l);
    } else {
        *lse = -INFINITY;
    }
}

/* --------------------------------------------------------- step drivers ---- */
/* The whole sparse decode step (O1..O8) for a batch.  Outputs (all caller-allocated):
 *   budget_tokens[n], k_pages[n], sel_count[n]        int64
 *   forced  [n][max_pages]            uint8 (0/1 for p < n_pages)
 *   scores  [n][Hkv][max_pages]       double (all pages; NaN where the sequence is dense)
 *   tau     [n][Hkv]                  double
 *   sel     [n][Hkv][max_sel]         int32 ascending, first sel_count[i] valid, rest -1
 *   out     [n][Hq][D]                double;  lse [n][Hq] double
 * do_attention = 0 skips O8 (selection only).  Returns 0, or -1 if max_sel is too small. */
int oracle_sparse_step(const uint16_t *q, const uint16_t *k_cache, const uint16_t *v_cache,
                       const int32_t *page_table, const int32_t *seq_lens, const oracle_schedule *sched,
                       int64_t n, int64_t Hq, int64_t Hkv, int64_t P, int64_t D,
                       int64_t max_pages, int64_t max_sel, double sm_scale, int do_attention,
                       int64_t *budget_tokens, int64_t *k_pages, int64_t *sel_count,
                       uint8_t *forced, double *scores, double *tau, int32_t *sel,
                       double *out, double *lse)
{
    int64_t r = Hq / Hkv;
    int err = 0;
    for (int64_t i = 0; i < n; ++i) {
        int64_t L = seq_lens[i];
        budget_tokens[i] = oracle_budget_tokens(sched, L, P);
        k_pages[i] = oracle_k_pages(sched, L, P);
        memset(forced + i * max_pages, 0, (size_t)max_pages);
        int64_t nf = oracle_forced_pages(L, sched->sink_tokens, sched->local_tokens, P, forced + i * max_pages);
        int64_t n_pages = ceil_div(L, P);
        int64_t cnt = k_pages[i] >= n_pages ? n_pages : (k_pages[i] > nf ? k_pages[i] : nf);
        sel_count[i] = cnt;
        if (cnt > max_sel) err = -1;
    }
    if (err) return err;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t u = 0; u < n * Hkv; ++u) {
        int64_t i = u / Hkv, g = u % Hkv;
        int64_t L = seq_lens[i];
        int64_t n_pages = ceil_div(L, P);
        const int32_t *pt_row = page_table + i * max_pages;
        double *s = scores + (i * Hkv + g) * max_pages;
        int32_t *sel_u = sel + (i * Hkv + g) * max_sel;
        for (int64_t p = 0; p < max_pages; ++p) s[p] = NAN;
        for (int64_t p = 0; p < max_sel; ++p) sel_u[p] = -1;
        int32_t *tmp = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n_pages > 0 ? n_pages : 1));
        if (k_pages[i] < n_pages)
            oracle_scores_unit(q + i * Hq * D, k_cache, pt_row, L, g, Hq, Hkv, P, D, s);
        int64_t m = oracle_select_unit(s, forced + i * max_pages, n_pages, k_pages[i], tmp, &tau[i * Hkv + g]);
        for (int64_t p = 0; p < m; ++p) sel_u[p] = tmp[p];
        if (do_attention)
            oracle_attention_unit(q + i * Hq * D, k_cache, v_cache, pt_row, L, tmp, m, g, Hq, Hkv, P, D, sm_scale,
                                  out + (i * Hq + g * r) * D, lse + i * Hq + g * r, NULL);
        free(tmp);
    }
    return 0;
}

/* O8 over caller-supplied page lists (R11: the oracle's attention evaluated on the GPU's own
 * set when the two sets differ only inside the tie band).  sel [n][Hkv][max_sel], sel_count[n]. */
void oracle_attention_on_sets(const uint16_t *q, const uint16_t *k_cache, const uint16_t *v_cache,
                              const int32_t *page_table, const int32_t *seq_lens,
                              const int32_t *sel, const int64_t *sel_count,
                              int64_t n, int64_t Hq, int64_t Hkv, int64_t P, int64_t D,
                              int64_t max_pages, int64_t max_sel, double sm_scale,
                              double *out, double *lse)
{
    int64_t r = Hq / Hkv;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t u = 0; u < n * Hkv; ++u) {
        int64_t i = u / Hkv, g = u % Hkv;
        oracle_attention_unit(q + i * Hq * D, k_cache, v_cache, page_table + i * max_pages, seq_lens[i],
                              sel + (i * Hkv + g) * max_sel, sel_count[i], g, Hq, Hkv, P, D, sm_scale,
                              out + (i * Hq + g * r) * D, lse + i * Hq + g * r, NULL);
    }
}

/* Dense entry (a8): O8 with Sel = all pages of the sequence (Eq. 2). */
void oracle_dense_step(const uint16_t *q, const uint16_t *k_cache, const uint16_t *v_cache,
                       const int32_t *page_table, const int32_t *seq_lens,
                       int64_t n, int64_t Hq, int64_t Hkv, int64_t P, int64_t D,
                       int64_t max_pages, double sm_scale, double *out, double *lse)
{
    int64_t r = Hq / Hkv;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t u = 0; u < n * Hkv; ++u) {
        int64_t i = u / Hkv, g = u % Hkv;
        int64_t n_pages = ceil_div(seq_lens[i], P);
        int32_t *all = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n_pages > 0 ? n_pages : 1));
        for (int64_t p = 0; p < n_pages; ++p) all[p] = (int32_t)p;
        oracle_attention_unit(q + i * Hq * D, k_cache, v_cache, page_table + i * max_pages, seq_lens[i],
                              all, n_pages, g, Hq, Hkv, P, D, sm_scale,
                              out + (i * Hq + g * r) * D, lse + i * Hq + g * r, NULL);
        free(all);
    }
}

int oracle_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    n = omp_get_max_threads();
#endif
    return n;
}
