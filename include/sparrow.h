/*
 * sparrow.h -- C ABI of the B200-native sparse decode attention of Sparrow's sparse rollout
 * (arxiv/paper_2606_08446).  One shared library, libsparrow_b200.so, hand-written CUDA for sm_100a.
 *
 * What the calls compute (paper passages; readings R1..R20):
 *   per decode step and layer:  page "landmark" scores  ->  Top-k pages under the KV budget
 *   B = pagesize x num_pages  ->  attention over the B selected tokens            (Eq. 3)
 *   the budget grows with sequence length (dynamic sparsity schedule, 2K-token bins)
 *   attention is dense while the context still fits the budget
 *   page size 16
 * The paper leaves the selector's details open; BASELINE.json north_star fixes them: page summaries are
 * per-channel key min/max, the score is the upper bound of q.k against the summary summed over the GQA
 * group, sink and local-window pages are always kept, the top-k remaining pages fill B(L).
 *
 * Conventions (all entry points)
 *   - Every pointer is a DEVICE pointer owned by the caller unless the parameter is documented "host".
 *     The library never allocates, frees or synchronises on the device-pointer entry points; work is
 *     enqueued on `stream` (a cudaStream_t passed as void*, NULL = the legacy default stream) and the
 *     calls can be captured in a CUDA graph.  Device pointers must be 16-byte aligned.
 *   - bf16 tensors are raw 16-bit patterns.  Layouts (row-major, innermost last):
 *       k_cache, v_cache  [n_phys_pages][n_kv_heads][page_size][head_dim=128]      bf16  ("HND" pages; page_size 16,
 *                                                      32, 64 or 128 -- a larger page is streamed as 16-token tiles)
 *       summaries         [n_phys_pages][n_kv_heads][2][128]                       bf16  ([0]=min, [1]=max)
 *       q, out            [n_seq][n_q_heads][128]                                  bf16
 *       lse               [n_seq][n_q_heads]                                       fp32  (natural log)
 *       page_table        [n_seq][max_pages_per_seq]                               int32 logical -> physical
 *       seq_lens          [n_seq]                                                  int32 L = cached length
 *                                                      INCLUDING the current token (R6); L >= 1
 *       sel_pages         [n_seq][n_kv_heads][max_sel]                             int32 logical pages,
 *                                                      ascending, forced pages included
 *       sel_count         [n_seq]                                                  int32 (same for all kv heads)
 *     Query head h uses kv head h / r, r = n_q_heads / n_kv_heads (GQA; K/V are read once per group).
 *   - Return value: SPARROW_OK (0) or a negative sparrow_status; nothing throws, aborts or falls back to
 *     the CPU.  Supported: head_dim = 128, page_size in {16, 32, 64, 128}, 1 <= r <= 8, bf16; anything else returns
 *     SPARROW_ERR_UNSUPPORTED.
 */
#ifndef SPARROW_H_
#define SPARROW_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ABI version of this header = what sparrow_version() of a matching library returns.  It changes whenever a struct layout or
 * a signature does: 100 = the first layout; 300 = sparrow_shape_t with landmark + kv_stride_*, sparrow_step_host over one
 * host block (sparrow_step / sparrow_step_workspace_bytes removed), sparrow_select_static.  A caller built against another
 * header must not pass its structs to this library: compare SPARROW_ABI_VERSION with sparrow_version() at start-up. */
#define SPARROW_ABI_VERSION 300

typedef enum sparrow_status {
    SPARROW_OK = 0,
    SPARROW_ERR_INVALID_ARG = -1,        /* null / negative / misaligned argument */
    SPARROW_ERR_UNSUPPORTED = -2,        /* shape outside the supported set (see above) */
    SPARROW_ERR_WORKSPACE_TOO_SMALL = -3,
    SPARROW_ERR_CUDA = -4,               /* launch or runtime failure; text via sparrow_strerror */
    SPARROW_ERR_STATIC_SCRATCH_TOO_SMALL = -5   /* sparrow_select_static only: the shape needs more than SPARROW_SELECT_STATIC_BYTES */
} sparrow_status;

typedef struct sparrow_shape {
    int32_t n_seq;               /* sequences in the batch (n) */
    int32_t n_q_heads;           /* Hq */
    int32_t n_kv_heads;          /* Hkv */
    int32_t head_dim;            /* D, must be 128 */
    int32_t page_size;           /* P: 16 (the paper's choice) or 32 / 64 / 128 (Table 4) */
    int32_t max_pages_per_seq;   /* row stride of page_table */
    int64_t n_phys_pages;        /* pages in the K/V pools */
    int32_t landmark;            /* SPARROW_LANDMARK_MINMAX (0, north_star's default) or SPARROW_LANDMARK_MEAN (1) */
    int32_t flags;               /* 0 or SPARROW_FLAG_DETERMINISTIC (below); occupies what was padding: offsets and size unchanged */
    /* Strides of the K and V pools in ELEMENTS (both pools share them; the head dim is contiguous): row t of kv-head g of
     * physical page p starts at p * kv_stride_page + g * kv_stride_head + t * kv_stride_tok.  All three 0 (the default) =
     * the packed "HND" layout [n_phys_pages][n_kv_heads][page_size][128] this library is tuned for (a (page, kv-head) tile
     * is contiguous: one TMA box of 32 x 128 B).  "NHD" pools [n_phys_pages][page_size][n_kv_heads][128] (the default of
     * vLLM / FlashInfer) are kv_stride_page = page_size * n_kv_heads * 128, kv_stride_tok = n_kv_heads * 128,
     * kv_stride_head = 128.  Each stride must be a multiple of 8 elements (16 bytes), kv_stride_tok >= 128, and rows must
     * not overlap; strided pools are fetched with one 5-D TMA box per tile instead of a 2-D one.  The summaries keep their
     * own packed layout either way. */
    int64_t kv_stride_page, kv_stride_head, kv_stride_tok;
} sparrow_shape_t;

/* sparrow_shape_t.flags.
 * SPARROW_FLAG_DETERMINISTIC: the decode entry points (sparse, dense, and the decode inside sparrow_step_host) hand their
 *   page tiles to the CTA's warps in a fixed pattern (warp w takes tile pairs w, w + 8, ...) and merge the pieces of a unit
 *   that spans CTAs in one fixed order, so `out` and `lse` are BIT-IDENTICAL from call to call on the same inputs, shape and
 *   GPU model (the split of the tile stream over the SMs depends on the SM count).  Without it tiles go to whichever warp is
 *   free, which balances the warps slightly better; results then agree only to the arithmetic's own error (see
 *   sparrow_sparse_decode).  A rollout engine whose log-probabilities are compared with a trainer's (PAPER.md:76-79,
 *   :409-414: the rollout / policy mismatch the paper measures) should set it.  Selection, summaries and append are
 *   bit-reproducible either way.  Measured cost: DESIGN.md 6.3 / profiles/r3_deterministic.md. */
enum { SPARROW_FLAG_DETERMINISTIC = 1 };

/* Form of the page landmark (PAPER.md:147 leaves it open; reading R1):
 *   MINMAX  per-channel min and max of the page's keys, summaries [n_phys_pages][n_kv_heads][2][128] (512 B), score =
 *           sum_{h in group} sum_d max(q*min, q*max) -- an upper bound of q.k over the page (north_star's default)
 *   MEAN    the mean key, summaries [n_phys_pages][n_kv_heads][128] (256 B), score = sum_{h in group} q_h . mean -- the
 *           one-vector-per-page landmark that the paper's cost model charges.  mean over the valid
 *           tokens, accumulated in fp32, rounded once to bf16: the stored code is the exactly rounded mean or, where the
 *           exact mean lies within the fp32 accumulation error of a rounding boundary, the neighbouring code (R24).
 * Everything else (budget, forced pages, top-k, attention) is the same. */
enum { SPARROW_LANDMARK_MINMAX = 0, SPARROW_LANDMARK_MEAN = 1 };

/* Dynamic sparsity schedule B(L) in EXACT integer arithmetic (R3), so that host, device and any checker
 * agree bit for bit.  Fractions are parts per million in [0, 1000000] (L1 - L0 < 2^31); anything else is
 * SPARROW_ERR_INVALID_ARG.  After the kind-specific value B is clamped to
 * at least floor_tokens (kinds 2, 3) and at most L.  K_pages = min(ceil(B/16), ceil(L/16)) (R4); a
 * sequence with K_pages >= n_pages is dense. */
enum {
    SPARROW_SCHED_DENSE = 0,        /* B = L */
    SPARROW_SCHED_FIXED = 1,        /* B = fixed_tokens */
    SPARROW_SCHED_CLAMP_FRAC = 2,   /* B = max(floor(L*f0_ppm/1e6), floor_tokens) */
    SPARROW_SCHED_LINEAR_FRAC = 3,  /* keep fraction falls linearly from f0_ppm at L0 to f1_ppm at L1 (clamped outside) */
    SPARROW_SCHED_TABLE = 4         /* the paper's native form: pages per length bin, bin b = (L-1)/bin_tokens
                                       (2K bins); B = table_pages[b] * 16 */
};
#define SPARROW_MAX_TABLE_BINS 64

typedef struct sparrow_schedule {
    int32_t kind;
    int32_t sink_tokens;          /* S: pages [0, ceil(S/16)) are always kept (R8) */
    int32_t local_tokens;         /* W: every page overlapping the last W tokens is always kept (R7);
                                     the last page is kept even when W = 0 (R9) */
    int64_t fixed_tokens;
    int64_t floor_tokens;
    int64_t f0_ppm, f1_ppm;
    int64_t L0, L1;
    const int32_t *table_pages;   /* HOST pointer, table_len <= SPARROW_MAX_TABLE_BINS entries; copied by value */
    int32_t table_len;
    int32_t bin_tokens;
    int32_t page_size;            /* tokens per page that turns B(L) into pages: 16, 32, 64 or 128; 0 = 16.  The device
                                     entry points use shape->page_size and refuse a non-zero value that differs */
} sparrow_schedule_t;

/* ---- a1: page summaries (north_star (a); "landmark") -------------------------------
 * For u < n_update: page = page_ids ? page_ids[u] : u; valid = n_valid ? n_valid[u] : 16.
 * summaries[page][g][0][d] = min over t < valid of k_cache[page][g][t][d], [1] = max.  Results are exact
 * (a min/max of bf16 values).  Runs on page fill (a few pages per step) or in bulk after prefill. */
int sparrow_summarize(const void *k_cache, void *summaries, const int32_t *page_ids, const int32_t *n_valid,
                      int64_t n_update, const sparrow_shape_t *shape, void *stream);

/* ---- a2..a5: budget, forced pages, fused page scoring + per-(sequence, kv-head) top-k ------------
 * For every sequence: B(L) from `sched`; forced pages F (sink, local window, last page); candidates =
 * the other pages, scored  s[p] = sum_{h in group} sum_d max(q[h][d]*min[p][d], q[h][d]*max[p][d])  in
 * fp32; the k = max(0, K_pages - |F|) best candidates (ties: lower page index, R10) join F.  Output:
 * sel_pages ascending, sel_count[i] = n_pages if dense else max(K_pages, |F|).  `max_sel` must be
 * >= sparrow_max_sel_pages(sched, longest L) (precondition; the kernel clamps instead of overflowing).
 * scores_dbg: optional fp32 [n_seq][n_kv_heads][max_pages_per_seq]; candidate scores are written there
 * (other entries untouched).  workspace: sparrow_select_workspace_bytes(shape) bytes, ZERO-INITIALISED
 * once by the caller; the kernel restores the zeros it uses, so it can be reused call after call. */
int sparrow_select(const void *q, const void *summaries, const int32_t *page_table, const int32_t *seq_lens,
                   const sparrow_schedule_t *sched, int32_t *sel_pages, int32_t max_sel, int32_t *sel_count,
                   float *scores_dbg, void *workspace, size_t workspace_bytes,
                   const sparrow_shape_t *shape, void *stream);

/* ---- a2..a5 for callers that cannot allocate device memory: sparrow_select with the scratch built into the library ----
 * Same computation, same arguments and same results as sparrow_select, minus `workspace`: the selector's scratch (arrival
 * counters + fp32 page scores, sparrow_select_workspace_bytes(shape) bytes) lives in a fixed array inside the library
 * image instead of a buffer the caller allocates.  It is meant for code that is handed device pointers for its inputs
 * and outputs but has no allocator of its own to call: a plug-in or custom op inside a serving process whose memory pool
 * has already claimed the whole GPU (a cudaMalloc there fails, or takes memory the pool believes it owns), a step inside
 * a latency-critical decode loop where cudaMalloc / cudaFree would stall the device, or a caller reaching this C ABI from
 * a language runtime that has no CUDA allocation binding at all.  The call itself performs no cudaMalloc, no cudaFree and
 * no library call that allocates.
 *   Limit: sparrow_select_workspace_bytes(shape) <= SPARROW_SELECT_STATIC_BYTES (4 MiB: roughly
 *     n_seq * n_kv_heads * max_pages_per_seq <= 1 000 000, e.g. 64 sequences x 8 kv-heads x 2 000 pages); a larger shape
 *     returns SPARROW_ERR_STATIC_SCRATCH_TOO_SMALL before anything is launched -- use sparrow_select there.  The 4 MiB
 *     are resident on every GPU the process uses this library on, from the moment the library is loaded there until the
 *     process exits, whether or not this entry point is ever called.
 *   First call on a device: looks up the array's address on that device (one synchronous runtime query, remembered per
 *     device).  Make that first call during start-up, with the device current, before any stream capture begins.
 *   Sharing: there is ONE array per GPU and every call on that GPU uses it, whatever the stream or host thread.  Calls
 *     that may overlap on the GPU (two streams, two threads) race on it and give wrong selections; calls ordered one after
 *     the other on a stream (or otherwise serialised) are fine.  The array keeps the previous call's contents; the
 *     counters that must start at zero are cleared on `stream` at the head of each call. */
#define SPARROW_SELECT_STATIC_BYTES (4u << 20)
int sparrow_select_static(const void *q, const void *summaries, const int32_t *page_table, const int32_t *seq_lens,
                          const sparrow_schedule_t *sched, int32_t *sel_pages, int32_t max_sel, int32_t *sel_count,
                          float *scores_dbg, const sparrow_shape_t *shape, void *stream);
size_t sparrow_select_static_bytes(void);   /* SPARROW_SELECT_STATIC_BYTES of the loaded build (host only) */

/* ---- a6 + a7: split-K flash-decode over the selected pages, log-sum-exp merge ---------------------
 * out[i][h] = softmax_t(sm_scale * q[i][h].K_t) V_t over tokens t < L of the pages sel_pages[i][h/r][0..sel_count[i]),
 * gathered through page_table; fp32 accumulation, bf16 output; lse (optional, may be NULL) = ln sum exp.
 * workspace: sparrow_decode_workspace_bytes(shape, max_sel) bytes, ZERO-INITIALISED once by the caller (it
 * holds the split-K arrival counters; the kernel restores the zeros it uses, so it can be reused call
 * after call, but not by two calls in flight at the same time).  n_seq <= 4096.  The merge of the splits
 * is fused into the same launch (one kernel per call).  The K/V tiles are fetched by TMA: each call encodes
 * two tensor maps over the pools on the host (cuTensorMapEncodeTiled, a few microseconds) and passes them by value,
 * so the call stays asynchronous and graph-capturable.  Reproducibility: the page tiles are handed to the CTA's warps at
 * run time, so the running maximum under which a probability is rounded to bf16, and the fp32 summation order, can
 * differ between two calls on the same inputs -- the two outs agree to the arithmetic's own error (about 1e-3 absolute
 * for unit-variance V, the distance of either from an exact evaluation), lse to fp32 rounding; nothing else varies. */
int sparrow_sparse_decode(const void *q, const void *k_cache, const void *v_cache, const int32_t *page_table,
                          const int32_t *seq_lens, const int32_t *sel_pages, int32_t max_sel,
                          const int32_t *sel_count, void *out, float *lse, float sm_scale,
                          void *workspace, size_t workspace_bytes, const sparrow_shape_t *shape, void *stream);

/* ---- a8: dense decode = the same kernels with B(L) = L (all ceil(L/16) pages) ---
 * workspace: sparrow_decode_workspace_bytes(shape, 0) bytes, zero-initialised once like the sparse entry's. */
int sparrow_dense_decode(const void *q, const void *k_cache, const void *v_cache, const int32_t *page_table,
                         const int32_t *seq_lens, void *out, float *lse, float sm_scale,
                         void *workspace, size_t workspace_bytes, const sparrow_shape_t *shape, void *stream);

/* ---- rollout step, cache side: append one token per sequence, summarize on page fill ----
 * The rollout decodes token after token; the budget follows the growing length (:109-119).
 * For every sequence i with L = seq_lens[i] tokens cached: the rows k_new[i], v_new[i] ([n_seq][n_kv_heads][128]
 * bf16) are written at token position L (logical page L/16 through page_table, row L%16), seq_lens[i] becomes
 * L + 1, and if the token fills its page (L%16 == 15) that page's min/max summary is (re)computed in the same
 * launch -- a1 "on page fill".  A sequence whose page table has no room (L/16 >= max_pages_per_seq) is left
 * untouched.  The caller then runs sparrow_select / sparrow_sparse_decode with the new lengths;
 * a partially filled last page needs no summary because it is always kept (R9). */
int sparrow_append(const void *k_new, const void *v_new, void *k_cache, void *v_cache, void *summaries,
                   const int32_t *page_table, int32_t *seq_lens, const sparrow_shape_t *shape, void *stream);

/* ---- whole step through HOST buffers (the end-to-end measurement path) ----------------------------
 * The step's inputs live in ONE host block (pinned memory makes the copy asynchronous) laid out as
 *     q [n][Hq][128] bf16 at offset 0 | seq_lens [n] int32 | page_ids [n_update] int32 | n_valid [n_update] int32
 * at the 256-byte-aligned offsets sparrow_step_host_block_bytes() reports, so that a single host-to-device copy brings
 * them over (the caller writes its q and lengths straight into the block).  The call copies the used part of the
 * block, runs summarize (n_update <= n_seq pages that just filled; 0 = none; has_n_valid = 0 means full pages) ->
 * select -> sparse decode (or the dense path when sched->kind == DENSE) on `stream`, copies out back to
 * out_host [n][Hq][128] bf16 and WAITS for the stream.  The K/V pools, summaries and page_table are the resident
 * cache state and stay device pointers.  `scratch` is a device buffer of at least
 * sparrow_step_scratch_bytes(shape, max_sel) bytes, zero-initialised once by the caller. */
int sparrow_step_host(const void *in_block_host, int64_t n_update, int has_n_valid,
                      const void *k_cache, const void *v_cache, void *summaries, const int32_t *page_table,
                      const sparrow_schedule_t *sched, int32_t max_sel, float sm_scale,
                      void *out_host, void *scratch, size_t scratch_bytes,
                      const sparrow_shape_t *shape, void *stream);
/* The same step, left ENQUEUED: returns once the copies and kernels are on `stream`, without waiting for them.  A model
 * step is many layers; waiting after each costs a host round trip per layer (36 per step at config 4) during which the GPU
 * idles.  The caller waits once (cudaStreamSynchronize / an event) before it reads out_host, and must leave in_block_host
 * and out_host untouched until then; pinned memory is needed for the copies to be asynchronous at all.  Calls on the
 * same stream may share `scratch` (they run in stream order). */
int sparrow_step_host_async(const void *in_block_host, int64_t n_update, int has_n_valid,
                            const void *k_cache, const void *v_cache, void *summaries, const int32_t *page_table,
                            const sparrow_schedule_t *sched, int32_t max_sel, float sm_scale,
                            void *out_host, void *scratch, size_t scratch_bytes,
                            const sparrow_shape_t *shape, void *stream);
/* Size of the host block and (optional out-parameters) the offsets of its seq_lens / page_ids / n_valid parts. */
size_t sparrow_step_host_block_bytes(const sparrow_shape_t *shape, size_t *off_seq_lens, size_t *off_page_ids,
                                     size_t *off_n_valid);

/* ---- the paper's divergence statistic (SURVEY.md 8(f)-3; PAPER.md:76-79 Eq. 1, :95, :101, :119) -------------
 * Per token position i < n_pos the dense policy P and the sparse policy Q each give their top_n (<= 32) tokens and
 * natural-log probabilities: ids_p, logp_p, ids_q, logp_q are [n_pos][top_n].  alpha[i] = sum over the tokens present
 * in BOTH lists of min(p, q) -- Eq. 1's sum_x min(p(x), q(x)) restricted to what the engine returns (reading R23; a
 * token missing from one list adds nothing; ids must be >= 0 -- the kernel pads short lists with -1 -- and distinct within a
 * list).  Positions are grouped in bins
 * b = min(positions[i] / bin_tokens, n_bins - 1) (2K-token bins in the paper); bin_count[b] = tokens in the bin and
 * bin_quantile[b] = the nearest-rank `quantile` (0.05 in the paper) of alpha over the bin: the value of rank
 * max(1, ceil(quantile * count)) in ascending order, NaN for an empty bin.  fp32 throughout; exact selection.
 * workspace: sparrow_acceptance_workspace_bytes(n_bins) bytes, ZERO-INITIALISED once, restored by the call. */
int sparrow_acceptance(const int32_t *ids_p, const float *logp_p, const int32_t *ids_q, const float *logp_q,
                       const int32_t *positions, int64_t n_pos, int32_t top_n, int32_t bin_tokens, int32_t n_bins,
                       float quantile, float *alpha, float *bin_quantile, int32_t *bin_count,
                       void *workspace, size_t workspace_bytes, void *stream);
size_t sparrow_acceptance_workspace_bytes(int32_t n_bins);

/* ---- rollout cost model (SURVEY.md 8(f)-4; PAPER.md:129-145 Eq. 2-3, :474-498 App. F) -- host only ----------
 * Equivalent-FLOP cost of a rollout: batch_size x n_samples responses of L_out tokens after a prompt of L_in,
 * model of P parameters, K/V width D, GQA ratio r, hardware intensity I (flops per element moved; R18), KV budget K
 * tokens, page size, c landmark vectors per page (1 = the paper's model, 2 = this library's min/max summaries, R1).
 *   attention elements   H = (2 L_in + L_d) L_d + 2 K (L_out - L_d)+ ,  L_d = min(L_out, max(K - L_in, 0))   (App. F)
 *   dense   comp = 2 P B N L_out + r B N (2 L_in + L_out) L_out D      mem = 2 P L_out + B N (2 L_in L_out + L_out^2) D
 *   sparse  comp = 2 P B N L_out + r B N D H                           mem = 2 P L_out + B N D H
 *   scoring (steps past the dense phase only; landmark visits S = sum over those steps of (L_in + t) / pagesize):
 *           comp = r c B N D S                                         mem = c B N D S         (Eq. 3; reading R21:
 *           with c = 1 and L_in = 0 these are the paper's printed r N D L_out^2 / (2 pagesize) and N D L_out^2 / (2 pagesize))
 *   total = comp + I * mem.  Returns SPARROW_ERR_INVALID_ARG for non-positive sizes. */
typedef struct sparrow_cost_args {
    double params, batch_size, n_samples, L_in, L_out, D, r, intensity, budget_tokens, page_size, landmarks_per_page;
} sparrow_cost_args_t;
typedef struct sparrow_cost {
    double attn_elems_dense, attn_elems_sparse, landmark_visits;
    double dense_comp, dense_mem, dense_total;
    double sparse_comp, sparse_mem, scoring_comp, scoring_mem, sparse_total;
} sparrow_cost_t;
int sparrow_cost_model(const sparrow_cost_args_t *args, sparrow_cost_t *cost);

/* ---- host helpers (no device work; callable without a GPU) ---------------------------------------- */
size_t sparrow_select_workspace_bytes(const sparrow_shape_t *shape);
size_t sparrow_decode_workspace_bytes(const sparrow_shape_t *shape, int32_t max_sel /* 0 = dense */);
size_t sparrow_step_scratch_bytes(const sparrow_shape_t *shape, int32_t max_sel);
/* B(L) in tokens, K_pages, number of forced pages, and the bound on sel_count over all L <= max_len. */
int64_t sparrow_budget_tokens(const sparrow_schedule_t *sched, int64_t L);
int32_t sparrow_k_pages(const sparrow_schedule_t *sched, int64_t L);
int32_t sparrow_forced_count(const sparrow_schedule_t *sched, int64_t L);
int32_t sparrow_sel_count(const sparrow_schedule_t *sched, int64_t L);
int32_t sparrow_max_sel_pages(const sparrow_schedule_t *sched, int64_t max_len);
const char *sparrow_strerror(int status);   /* static string; for SPARROW_ERR_CUDA includes the last CUDA error text */
int sparrow_version(void);
/* Kernels launched by the most recent entry-point call on this thread (for gpu_launches accounting). */
int sparrow_last_launch_count(void);
/* Profiling plumbing, not one of the method's calls.  Tracing build only (compiled with -DSPARROW_TRACE: `python -m paper_2606_08446_b200.build --trace`): the select and
 * decode kernels drop %globaltimer stamps per CTA / warp into `buffer`, a DEVICE array of 65536 x 8 64-bit words the
 * caller zeroes (layout: csrc/common.cuh); NULL switches the stamps off.  Synchronous (a symbol copy).  The normal build
 * carries no stamps and returns SPARROW_ERR_UNSUPPORTED.  Used by paper_2606_08446_b200/trace.py for the timelines under
 * profiles/. */
int sparrow_trace_set(void *buffer);

#ifdef __cplusplus
}
#endif
#endif /* SPARROW_H_ */
