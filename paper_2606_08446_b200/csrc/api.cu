// api.cu -- the C ABI of libsparrow_b200 (include/sparrow.h): argument validation, launch geometry, workspaces.
// Every step of the path runs in the kernels of summarize.cuh / select.cuh / decode.cuh; there is no CPU fallback.
#include <stdio.h>
#include <string.h>

#include <mutex>

#include "common.cuh"
#include "decode.cuh"
#include "select.cuh"
#include "summarize.cuh"
#include "append.cuh"
#include "accept.cuh"

using namespace sparrow;

namespace {

thread_local int g_launches = 0;
thread_local char g_errbuf[256] = "";
constexpr int kNumSmsB200 = 148;

// Per-device launch state: the SM count (queried once per device) and the dynamic shared memory each kernel has been
// allowed so far (cudaFuncSetAttribute is per device).  Guarded by one mutex: entry points may be called from several
// host threads, each on its own device.
struct DevState {
    bool init = false;
    int sms = 0;
    size_t dyn_decode[2] = {0, 0}, dyn_select[2] = {0, 0}, dyn_hist = 0, dyn_alpha[2] = {0, 0};
};
constexpr int kMaxDevices = 64;
DevState g_dev[kMaxDevices];
std::mutex g_dev_mutex;

// Returns the calling thread's current device state (nullptr + *rc on failure).  The library is written for the
// B200's 148 SMs: persistent grids are sized from the queried count and capped at 148 (the workspace bounds).
DevState *dev_state(int *rc)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= kMaxDevices) {
        snprintf(g_errbuf, sizeof(g_errbuf), "cudaGetDevice failed or device ordinal >= %d", kMaxDevices);
        *rc = SPARROW_ERR_CUDA;
        return nullptr;
    }
    DevState *d = &g_dev[dev];
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    if (!d->init) {
        e = cudaDeviceGetAttribute(&d->sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || d->sms <= 0) {
            snprintf(g_errbuf, sizeof(g_errbuf), "cannot query the SM count: %s", cudaGetErrorString(e));
            *rc = SPARROW_ERR_CUDA;
            return nullptr;
        }
        d->init = true;
    }
    return d;
}
// Raises a kernel's dynamic shared memory limit on this device if `bytes` exceeds what it has been given so far.
template <typename K>
int ensure_dyn_smem(K kernel, size_t bytes, size_t *granted, const char *what)
{
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    if (bytes > 32 * 1024 && bytes > *granted) {        // static + dynamic above 48 KiB needs the opt-in; kernels here have < 16 KiB static
        cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) {
            snprintf(g_errbuf, sizeof(g_errbuf), "CUDA error in cudaFuncSetAttribute(%s): %s", what, cudaGetErrorString(e));
            return SPARROW_ERR_CUDA;
        }
        *granted = bytes;
    }
    return SPARROW_OK;
}

int cuda_fail(cudaError_t e, const char *where)
{
    snprintf(g_errbuf, sizeof(g_errbuf), "CUDA error in %s: %s", where, cudaGetErrorString(e));
    return SPARROW_ERR_CUDA;
}
#define SPARROW_CHECK_LAUNCH(where)                         \
    do {                                                    \
        cudaError_t e__ = cudaGetLastError();               \
        if (e__ != cudaSuccess) return cuda_fail(e__, where); \
        ++g_launches;                                       \
    } while (0)

// Launch of a kernel of the step chain with programmatic stream serialization (see chain_entry() in common.cuh).
template <typename... KArgs, typename... Args>
cudaError_t launch_chain(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args &&...args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
#ifndef SPARROW_NO_PDL
    cfg.attrs = attr;
    cfg.numAttrs = 1;
#endif
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

int check_shape(const sparrow_shape_t *s)
{
    if (!s) return SPARROW_ERR_INVALID_ARG;
    if (s->n_seq < 0 || s->n_q_heads <= 0 || s->n_kv_heads <= 0 || s->max_pages_per_seq <= 0 || s->n_phys_pages < 0)
        return SPARROW_ERR_INVALID_ARG;
    if (s->head_dim != kDim) return SPARROW_ERR_UNSUPPORTED;
    if (s->page_size != 16 && s->page_size != 32 && s->page_size != 64 && s->page_size != 128) return SPARROW_ERR_UNSUPPORTED;
    if (s->n_q_heads % s->n_kv_heads != 0) return SPARROW_ERR_UNSUPPORTED;
    const int r = s->n_q_heads / s->n_kv_heads;
    if (r < 1 || r > kMaxGroup) return SPARROW_ERR_UNSUPPORTED;
    if (s->n_kv_heads > 65535 || s->n_seq > 65535) return SPARROW_ERR_UNSUPPORTED;     // grid.y / grid.z
    if (s->landmark != SPARROW_LANDMARK_MINMAX && s->landmark != SPARROW_LANDMARK_MEAN) return SPARROW_ERR_INVALID_ARG;
    if (s->flags & ~SPARROW_FLAG_DETERMINISTIC) return SPARROW_ERR_INVALID_ARG;          // unknown bits (or a caller that left the old padding unset)
    if (s->kv_stride_page != 0 || s->kv_stride_head != 0 || s->kv_stride_tok != 0) {
        const int64_t sp = s->kv_stride_page, sh = s->kv_stride_head, stt = s->kv_stride_tok;
        if (sp <= 0 || sh <= 0 || stt < kDim || (sp & 7) || (sh & 7) || (stt & 7)) return SPARROW_ERR_INVALID_ARG;
        // rows must not overlap: one of the two nestings token-inside-head (HND-like) or head-inside-token (NHD-like)
        const bool hnd_like = sh >= stt * s->page_size && sp >= sh * s->n_kv_heads;
        const bool nhd_like = sh >= kDim && stt >= sh * s->n_kv_heads && sp >= stt * s->page_size;
        if (!hnd_like && !nhd_like) return SPARROW_ERR_INVALID_ARG;
    }
    return SPARROW_OK;
}

// the pools' strides in elements; packed = the default HND layout, whose (page, kv-head) tiles are contiguous
KvLayout kv_layout(const sparrow_shape_t *s, bool *packed)
{
    KvLayout kv;
    const int64_t P = s->page_size;
    if (s->kv_stride_page == 0 && s->kv_stride_head == 0 && s->kv_stride_tok == 0) {
        kv.tok = kDim; kv.head = P * kDim; kv.page = (int64_t)s->n_kv_heads * P * kDim;
    } else {
        kv.tok = s->kv_stride_tok; kv.head = s->kv_stride_head; kv.page = s->kv_stride_page;
    }
    if (packed) *packed = kv.tok == kDim && kv.head == P * kDim && kv.page == (int64_t)s->n_kv_heads * P * kDim;
    return kv;
}

// page_tokens: the shape's page size for the device entry points; 0 = take the schedule's own (host helpers), default 16
int to_dev_sched(const sparrow_schedule_t *in, SchedDev *out, int page_tokens = 0)
{
    if (!in) return SPARROW_ERR_INVALID_ARG;
    if (in->kind < SPARROW_SCHED_DENSE || in->kind > SPARROW_SCHED_TABLE) return SPARROW_ERR_INVALID_ARG;
    if (in->sink_tokens < 0 || in->local_tokens < 0) return SPARROW_ERR_INVALID_ARG;
    memset(out, 0, sizeof(*out));
    out->kind = in->kind;
    out->sink_tokens = in->sink_tokens;
    out->local_tokens = in->local_tokens;
    out->fixed_tokens = in->fixed_tokens;
    out->floor_tokens = in->floor_tokens;
    out->f0_ppm = in->f0_ppm;
    out->f1_ppm = in->f1_ppm;
    out->L0 = in->L0;
    out->L1 = in->L1;
    out->bin_tokens = in->bin_tokens;
    if (in->page_size != 0 && in->page_size != 16 && in->page_size != 32 && in->page_size != 64 && in->page_size != 128)
        return SPARROW_ERR_INVALID_ARG;
    if (page_tokens != 0 && in->page_size != 0 && in->page_size != page_tokens) return SPARROW_ERR_INVALID_ARG;
    out->page = page_tokens != 0 ? page_tokens : (in->page_size != 0 ? in->page_size : kPage);
    out->page_log2 = out->page == 16 ? 4 : (out->page == 32 ? 5 : (out->page == 64 ? 6 : 7));
    out->inv_den = 1.0;
    if (in->kind == SPARROW_SCHED_FIXED && in->fixed_tokens < 0) return SPARROW_ERR_INVALID_ARG;
    constexpr int64_t kPpmMax = 1000000;                 // keep fractions are in [0, 1]
    if (in->kind == SPARROW_SCHED_CLAMP_FRAC && (in->f0_ppm < 0 || in->f0_ppm > kPpmMax || in->floor_tokens < 0))
        return SPARROW_ERR_INVALID_ARG;
    if (in->kind == SPARROW_SCHED_LINEAR_FRAC &&
        (in->L0 < 0 || in->L1 <= in->L0 || in->L1 - in->L0 > 0x7fffffffLL || in->f0_ppm < 0 || in->f0_ppm > kPpmMax ||
         in->f1_ppm < 0 || in->f1_ppm > kPpmMax || in->floor_tokens < 0))
        return SPARROW_ERR_INVALID_ARG;
    if (in->kind == SPARROW_SCHED_LINEAR_FRAC) out->inv_den = 1.0 / (1.0e6 * (double)(in->L1 - in->L0));
    if (in->kind == SPARROW_SCHED_TABLE) {
        if (!in->table_pages || in->table_len <= 0 || in->table_len > SPARROW_MAX_TABLE_BINS || in->bin_tokens <= 0)
            return SPARROW_ERR_INVALID_ARG;
        out->table_len = in->table_len;
        for (int i = 0; i < in->table_len; ++i) {
            if (in->table_pages[i] < 0) return SPARROW_ERR_INVALID_ARG;
            out->table[i] = in->table_pages[i];
        }
    }
    return SPARROW_OK;
}

// Decode workspace: per-unit counters + the tail-piece counter + the CTAs-done counter (all zero between calls), then the
// fp32 partial slots of the pieces (indexed unit + piece id) and their (m, l) pairs.  Pieces: one static piece per CTA
// plus the self-scheduled tail pieces of kTailChunk tiles (decode.cuh).
struct DecodeGeom {
    size_t bytes_o, bytes_ml, bytes_ctr;
};
DecodeGeom decode_geom(const sparrow_shape_t *s, int32_t max_sel /* 0 = dense */)
{
    DecodeGeom gm;
    const size_t units = (size_t)s->n_seq * s->n_kv_heads;
    const int64_t max_cnt = (max_sel > 0 && max_sel < s->max_pages_per_seq) ? max_sel : s->max_pages_per_seq;
    const int64_t t_max = (int64_t)units * max_cnt * (s->page_size / kPage);                       // tiles of the stream at most
    const int64_t tail_max = t_max - t_max * SPARROW_DEC_STATIC_NUM / SPARROW_DEC_STATIC_DEN;
    const size_t pieces = (size_t)kDecGrid + (size_t)((tail_max + kTailChunk - 1) / kTailChunk) + 1;
    const size_t rows = (units + pieces) * (s->n_q_heads / s->n_kv_heads);
    gm.bytes_o = (rows * kDim * sizeof(float) + 255) & ~(size_t)255;
    gm.bytes_ml = (rows * 2 * sizeof(float) + 255) & ~(size_t)255;
    gm.bytes_ctr = ((units + 2) * sizeof(int32_t) + 255) & ~(size_t)255;
    return gm;
}

// TMA view of a K or V pool: a 2-D bf16 tensor [rows = pages x kv-heads x page tokens][128 dims], row pitch 256 B, read in
// boxes of 16 rows x 64 columns (128 B wide: SWIZZLE_128B).  The encoder is a driver entry point (no link against libcuda).
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
int make_pool_map(CUtensorMap *tm, const void *pool, const sparrow_shape_t *s)
{
    static EncodeTiledFn encode = nullptr;
    static std::mutex m;
    {
        std::lock_guard<std::mutex> lock(m);
        if (!encode) {
            void *fn = nullptr;
            cudaDriverEntryPointQueryResult qres;
            cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
            if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) {
                snprintf(g_errbuf, sizeof(g_errbuf), "cuTensorMapEncodeTiled is not available from this driver");
                return SPARROW_ERR_CUDA;
            }
            encode = reinterpret_cast<EncodeTiledFn>(fn);
        }
    }
    bool packed = true;
    const KvLayout kv = kv_layout(s, &packed);
    CUresult rc;
    if (packed) {
        const cuuint64_t rows = (cuuint64_t)s->n_phys_pages * s->n_kv_heads * s->page_size * 2;     // 128-byte rows: (token, half)
        const cuuint64_t gdim[2] = {64, rows};
        const cuuint64_t gstride[1] = {128};
        const cuuint32_t box[2] = {64, (cuuint32_t)(2 * kPage)};
        const cuuint32_t estr[2] = {1, 1};
        rc = encode(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void *>(pool), gdim, gstride, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    } else {
        // strided pools (sparrow_shape_t kv_stride_*): [page][kv-head][token][half][64] as a 5-D tensor with the caller's
        // strides; one box = (64 columns, 2 halves, 16 tokens) of one kv-head of one page -- it lands in shared memory in the
        // same (token, half) row order and 128-byte swizzle as the packed layout's 32 x 64 box
        const cuuint64_t gdim[5] = {64, 2, (cuuint64_t)s->page_size, (cuuint64_t)s->n_kv_heads, (cuuint64_t)s->n_phys_pages};
        const cuuint64_t gstride[4] = {128, (cuuint64_t)kv.tok * 2, (cuuint64_t)kv.head * 2, (cuuint64_t)kv.page * 2};
        const cuuint32_t box[5] = {64, 2, (cuuint32_t)kPage, 1, 1};
        const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
        rc = encode(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, const_cast<void *>(pool), gdim, gstride, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    }
    if (rc != CUDA_SUCCESS) {
        snprintf(g_errbuf, sizeof(g_errbuf), "cuTensorMapEncodeTiled failed (CUresult %d)", (int)rc);
        return SPARROW_ERR_CUDA;
    }
    return SPARROW_OK;
}

size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

template <bool kDense>
int launch_decode(const void *q, const void *k_cache, const void *v_cache, const int32_t *page_table,
                  const int32_t *seq_lens, const int32_t *sel_pages, int32_t max_sel, const int32_t *sel_count,
                  void *out, float *lse, float sm_scale, void *workspace, size_t workspace_bytes,
                  const sparrow_shape_t *s, cudaStream_t st)
{
    const DecodeGeom gm = decode_geom(s, kDense ? 0 : max_sel);
    if (workspace_bytes < gm.bytes_ctr + gm.bytes_o + gm.bytes_ml) return SPARROW_ERR_WORKSPACE_TOO_SMALL;
    if (s->n_seq > kDecMaxSeq) return SPARROW_ERR_UNSUPPORTED;
    {   // flat tile positions and TMA row coordinates are 32-bit: the packed map's row coordinate is tile * 32 (decode.cuh),
        // so tile indices must stay below 2^26 (a 256 GiB pool -- beyond one B200, but the guard says what it protects)
        const int64_t max_cnt = kDense ? s->max_pages_per_seq : (max_sel < s->max_pages_per_seq ? max_sel : s->max_pages_per_seq);
        const int64_t tpp = s->page_size / kPage;
        if ((int64_t)s->n_seq * max_cnt * s->n_kv_heads * tpp >= (1LL << 31) || s->n_phys_pages * s->n_kv_heads * tpp >= (1LL << 26))
            return SPARROW_ERR_UNSUPPORTED;
    }
    if (s->n_seq == 0 || s->n_phys_pages == 0) return SPARROW_OK;
    int32_t *counters = reinterpret_cast<int32_t *>(workspace);
    float *ws_o = reinterpret_cast<float *>(reinterpret_cast<uint8_t *>(workspace) + gm.bytes_ctr);
    float *ws_ml = reinterpret_cast<float *>(reinterpret_cast<uint8_t *>(workspace) + gm.bytes_ctr + gm.bytes_o);

    constexpr int kSmemFixed = kDecRingBytes + kDecAccBytes + kDecDescBytes + kDecMetaBytes;
    constexpr int kSmemMax = kSmemFixed + ((kDecMaxSeq + 1) * 4 + 15) / 16 * 16;
    int rc_dev = SPARROW_OK;
    DevState *ds = dev_state(&rc_dev);
    if (!ds) return rc_dev;
    rc_dev = ensure_dyn_smem(decode_kernel<kDense>, kSmemMax, &ds->dyn_decode[kDense], "decode_kernel");
    if (rc_dev) return rc_dev;
    CUtensorMap tm_k, tm_v;
    if ((rc_dev = make_pool_map(&tm_k, k_cache, s)) != SPARROW_OK) return rc_dev;
    if ((rc_dev = make_pool_map(&tm_v, v_cache, s)) != SPARROW_OK) return rc_dev;
    const int smem = kSmemFixed + ((s->n_seq + 1) * 4 + 15) / 16 * 16;
    DecodeArgs A;
    A.q = (const uint16_t *)q;
    A.page_table = page_table; A.seq_lens = seq_lens; A.sel_pages = sel_pages; A.sel_count = sel_count;
    A.max_sel = max_sel; A.ws_o = ws_o; A.ws_ml = ws_ml; A.counters = counters;
    A.out = (uint16_t *)out; A.lse = lse; A.scale_log2 = sm_scale * 1.4426950408889634f;
    A.n_seq = s->n_seq; A.n_q_heads = s->n_q_heads; A.n_kv_heads = s->n_kv_heads; A.max_pages = s->max_pages_per_seq;
    A.tpp_log2 = s->page_size == 16 ? 0 : (s->page_size == 32 ? 1 : (s->page_size == 64 ? 2 : 3));
    {
        bool packed = true;
        kv_layout(s, &packed);
        A.strided = packed ? 0 : 1;
    }
    A.deterministic = (s->flags & SPARROW_FLAG_DETERMINISTIC) ? 1 : 0;
    const int grid = ds->sms < kDecGrid ? ds->sms : kDecGrid;   // one CTA per SM (the partial slots are sized for 148)
    launch_chain(decode_kernel<kDense>, dim3(grid), dim3(kDecThreads), smem, st, A, tm_k, tm_v);
    SPARROW_CHECK_LAUNCH("decode_kernel");
    return SPARROW_OK;
}

int summarize_impl(const void *k_cache, void *summaries, const int32_t *page_ids, const int32_t *n_valid,
                   int64_t n_update, const sparrow_shape_t *s, cudaStream_t st)
{
    if (n_update == 0) return SPARROW_OK;
    const int64_t tiles = n_update * s->n_kv_heads;
    const int64_t blocks = (tiles + kSumWarps - 1) / kSumWarps;
    if (blocks > 0x7fffffffLL) return SPARROW_ERR_UNSUPPORTED;
    if (s->landmark == SPARROW_LANDMARK_MEAN)
        launch_chain(summarize_mean_kernel, dim3((unsigned)blocks), dim3(kSumWarps * 32), 0, st, (const uint16_t *)k_cache,
                     (uint16_t *)summaries, page_ids, n_valid, n_update, s->n_kv_heads, s->page_size, kv_layout(s, nullptr));
    else
        launch_chain(summarize_kernel, dim3((unsigned)blocks), dim3(kSumWarps * 32), 0, st, (const uint16_t *)k_cache,
                     (uint16_t *)summaries, page_ids, n_valid, n_update, s->n_kv_heads, s->page_size, kv_layout(s, nullptr));
    SPARROW_CHECK_LAUNCH("summarize_kernel");
    return SPARROW_OK;
}

// Select workspace: arrival counters (one per (sequence, kv-head) unit; all zero between calls), then the fp32 scores
// [units][max_pages].
size_t select_ctr_bytes(const sparrow_shape_t *s) { return align256((size_t)s->n_seq * s->n_kv_heads * sizeof(int32_t)); }

int select_impl(const void *q, const void *summaries, const int32_t *page_table, const int32_t *seq_lens,
                const SchedDev &sd, int32_t *sel_pages, int32_t max_sel, int32_t *sel_count, float *scores_dbg,
                void *workspace, size_t workspace_bytes, const sparrow_shape_t *s, cudaStream_t st)
{
    if (workspace_bytes < sparrow_select_workspace_bytes(s)) return SPARROW_ERR_WORKSPACE_TOO_SMALL;
    if (s->max_pages_per_seq > kSelMaxPages) return SPARROW_ERR_UNSUPPORTED;
    if (s->n_phys_pages * s->n_kv_heads >= (1LL << 27)) return SPARROW_ERR_UNSUPPORTED;   // 32-bit offsets in 16-byte units
    if (s->n_seq == 0) return SPARROW_OK;
    int rc = SPARROW_OK;
    DevState *ds = dev_state(&rc);
    if (!ds) return rc;
    int32_t *counters = reinterpret_cast<int32_t *>(workspace);
    float *scores_ws = reinterpret_cast<float *>(reinterpret_cast<uint8_t *>(workspace) + select_ctr_bytes(s));
    // Pages per CTA: as large as keeps >= 4 CTAs per resident slot (4 per SM) so the tail stays short, because the
    // per-CTA fixed costs (loads of L / table entries / query rows, arrival) are amortised over the pages a CTA streams.
    const int64_t units = (int64_t)s->n_seq * s->n_kv_heads;
    // The mean landmark streams half the bytes per page, so its per-CTA fixed costs weigh twice as much: there the largest
    // slice that still leaves two CTAs per SM wins (measured, round 3: cfg2 27.6 -> 24.2 us, cfg5 37.8 -> 34.5 us, cfg3
    // unchanged; most units are then ONE CTA, which also skips the cross-CTA arrival before the top-k).
    const bool mean_lm = s->landmark == SPARROW_LANDMARK_MEAN;
    const int64_t ctas_wanted = mean_lm ? 2 * (int64_t)ds->sms : 4 * (int64_t)kSelMinBlocks * ds->sms;
    int pages_per_cta = kSelCtaPagesMin;
    for (int p = 4 * kSelCtaPagesMin; p > kSelCtaPagesMin; p >>= 1) {
        if (units * ((s->max_pages_per_seq + p - 1) / p) >= ctas_wanted) { pages_per_cta = p; break; }
    }
#ifdef SPARROW_SEL_PPC_FIXED
    pages_per_cta = SPARROW_SEL_PPC_FIXED;
#endif
    const size_t dyn = (size_t)s->max_pages_per_seq * sizeof(uint32_t);
    const bool mean = s->landmark == SPARROW_LANDMARK_MEAN;
    rc = mean ? ensure_dyn_smem(select_kernel<true>, dyn, &ds->dyn_select[1], "select_kernel<mean>")
              : ensure_dyn_smem(select_kernel<false>, dyn, &ds->dyn_select[0], "select_kernel");
    if (rc) return rc;
    dim3 grid((s->max_pages_per_seq + pages_per_cta - 1) / pages_per_cta, s->n_kv_heads, s->n_seq);
    if (mean)
        launch_chain(select_kernel<true>, grid, dim3(kSelThreads), dyn, st, (const uint16_t *)q, (const uint16_t *)summaries,
                     page_table, seq_lens, sd, sel_pages, max_sel, sel_count, scores_ws, counters, scores_dbg, s->n_q_heads,
                     s->n_kv_heads, s->max_pages_per_seq, pages_per_cta);
    else
        launch_chain(select_kernel<false>, grid, dim3(kSelThreads), dyn, st, (const uint16_t *)q, (const uint16_t *)summaries,
                     page_table, seq_lens, sd, sel_pages, max_sel, sel_count, scores_ws, counters, scores_dbg, s->n_q_heads,
                     s->n_kv_heads, s->max_pages_per_seq, pages_per_cta);
    SPARROW_CHECK_LAUNCH("select_kernel");
    return SPARROW_OK;
}

}  // namespace

extern "C" {

int sparrow_version(void) { return SPARROW_ABI_VERSION; }

int sparrow_trace_set(void *buffer)
{
#ifdef SPARROW_TRACE
    cudaError_t e = cudaMemcpyToSymbol(sparrow::g_trace, &buffer, sizeof(buffer));
    return e == cudaSuccess ? SPARROW_OK : cuda_fail(e, "cudaMemcpyToSymbol(g_trace)");
#else
    (void)buffer;
    return SPARROW_ERR_UNSUPPORTED;      // this build carries no stamps: build with -DSPARROW_TRACE (build.py --trace)
#endif
}
int sparrow_last_launch_count(void) { return g_launches; }

const char *sparrow_strerror(int status)
{
    switch (status) {
    case SPARROW_OK: return "ok";
    case SPARROW_ERR_INVALID_ARG: return "invalid argument (null, negative or misaligned)";
    case SPARROW_ERR_UNSUPPORTED:
        return "unsupported shape (need head_dim 128, page_size 16|32|64|128, 1 <= Hq/Hkv <= 8, bf16; decode: n_seq <= 4096, "
               "pool below 2^26 16-token tiles; select: n_seq <= 65535, max_pages_per_seq <= 16384)";
    case SPARROW_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
    case SPARROW_ERR_CUDA: return g_errbuf[0] ? g_errbuf : "CUDA error";
    case SPARROW_ERR_STATIC_SCRATCH_TOO_SMALL:
        return "shape needs more selector scratch than the library's built-in array holds (sparrow_select_static is limited "
               "to SPARROW_SELECT_STATIC_BYTES = 4 MiB, i.e. n_seq * n_kv_heads * max_pages_per_seq up to about one million): "
               "use sparrow_select with a workspace of your own";
    default: return "unknown status";
    }
}

size_t sparrow_select_workspace_bytes(const sparrow_shape_t *s)
{
    if (check_shape(s) != SPARROW_OK) return 0;
    const size_t units = (size_t)s->n_seq * s->n_kv_heads;
    return select_ctr_bytes(s) + align256(units * s->max_pages_per_seq * sizeof(float));
}

size_t sparrow_decode_workspace_bytes(const sparrow_shape_t *s, int32_t max_sel)
{
    if (check_shape(s) != SPARROW_OK) return 0;
    const DecodeGeom gm = decode_geom(s, max_sel);
    return gm.bytes_ctr + gm.bytes_o + gm.bytes_ml;
}

int sparrow_cost_model(const sparrow_cost_args_t *a, sparrow_cost_t *c)
{
    if (!a || !c) return SPARROW_ERR_INVALID_ARG;
    if (!(a->params >= 0) || !(a->batch_size > 0) || !(a->n_samples > 0) || !(a->L_in >= 0) || !(a->L_out > 0) || !(a->D > 0) ||
        !(a->r >= 1) || !(a->intensity >= 0) || !(a->budget_tokens > 0) || !(a->page_size > 0) || !(a->landmarks_per_page >= 0))
        return SPARROW_ERR_INVALID_ARG;
    const double BN = a->batch_size * a->n_samples, Li = a->L_in, Lo = a->L_out, K = a->budget_tokens;
    double Ld = K - Li;
    Ld = Ld < 0 ? 0 : (Ld > Lo ? Lo : Ld);
    const double rest = Lo - Ld;                                        // steps decoded under the budget
    c->attn_elems_dense = (2 * Li + Lo) * Lo;
    c->attn_elems_sparse = (2 * Li + Ld) * Ld + 2 * K * rest;
    c->landmark_visits = ((Li * Lo + 0.5 * Lo * Lo) - (Li * Ld + 0.5 * Ld * Ld)) / a->page_size;
    const double param_comp = 2 * a->params * BN * Lo, param_mem = 2 * a->params * Lo;
    c->dense_comp = param_comp + a->r * BN * c->attn_elems_dense * a->D;
    c->dense_mem = param_mem + BN * c->attn_elems_dense * a->D;
    c->dense_total = c->dense_comp + a->intensity * c->dense_mem;
    c->sparse_comp = param_comp + a->r * BN * a->D * c->attn_elems_sparse;
    c->sparse_mem = param_mem + BN * a->D * c->attn_elems_sparse;
    c->scoring_comp = a->r * a->landmarks_per_page * BN * a->D * c->landmark_visits;   // r D multiply-adds per landmark vector
    c->scoring_mem = a->landmarks_per_page * BN * a->D * c->landmark_visits;
    c->sparse_total = c->sparse_comp + c->scoring_comp + a->intensity * (c->sparse_mem + c->scoring_mem);
    return SPARROW_OK;
}

int64_t sparrow_budget_tokens(const sparrow_schedule_t *sched, int64_t L)
{
    SchedDev sd;
    if (to_dev_sched(sched, &sd) != SPARROW_OK || L < 0) return -1;
    return budget_tokens(sd, L);
}
int32_t sparrow_k_pages(const sparrow_schedule_t *sched, int64_t L)
{
    SchedDev sd;
    if (to_dev_sched(sched, &sd) != SPARROW_OK || L < 1) return -1;
    return make_plan(sd, L).k_pages;
}
int32_t sparrow_forced_count(const sparrow_schedule_t *sched, int64_t L)
{
    SchedDev sd;
    if (to_dev_sched(sched, &sd) != SPARROW_OK || L < 1) return -1;
    return make_plan(sd, L).n_forced;
}
int32_t sparrow_sel_count(const sparrow_schedule_t *sched, int64_t L)
{
    SchedDev sd;
    if (to_dev_sched(sched, &sd) != SPARROW_OK || L < 1) return -1;
    return make_plan(sd, L).count;
}
int32_t sparrow_max_sel_pages(const sparrow_schedule_t *sched, int64_t max_len)
{
    SchedDev sd;
    if (to_dev_sched(sched, &sd) != SPARROW_OK || max_len < 1) return -1;
    int32_t best = 0;      // B(L) need not be monotone (R15): scan every length (host only, ~1e5 evaluations at most)
    for (int64_t L = 1; L <= max_len; ++L) {
        const int32_t c = make_plan(sd, L).count;
        if (c > best) best = c;
    }
    return best;
}

int sparrow_summarize(const void *k_cache, void *summaries, const int32_t *page_ids, const int32_t *n_valid,
                      int64_t n_update, const sparrow_shape_t *shape, void *stream)
{
    g_launches = 0;
    int rc = check_shape(shape);
    if (rc) return rc;
    if (n_update < 0 || (!page_ids && n_update > shape->n_phys_pages)) return SPARROW_ERR_INVALID_ARG;
    if (n_update == 0) return SPARROW_OK;
    if (!k_cache || !summaries || !aligned16(k_cache) || !aligned16(summaries)) return SPARROW_ERR_INVALID_ARG;
    return summarize_impl(k_cache, summaries, page_ids, n_valid, n_update, shape, (cudaStream_t)stream);
}

int sparrow_select(const void *q, const void *summaries, const int32_t *page_table, const int32_t *seq_lens,
                   const sparrow_schedule_t *sched, int32_t *sel_pages, int32_t max_sel, int32_t *sel_count,
                   float *scores_dbg, void *workspace, size_t workspace_bytes, const sparrow_shape_t *shape, void *stream)
{
    g_launches = 0;
    int rc = check_shape(shape);
    if (rc) return rc;
    SchedDev sd;
    rc = to_dev_sched(sched, &sd, shape->page_size);
    if (rc) return rc;
    if (!q || !summaries || !page_table || !seq_lens || !sel_pages || !sel_count || !workspace || max_sel <= 0)
        return SPARROW_ERR_INVALID_ARG;
    if (!aligned16(q) || !aligned16(summaries) || !aligned16(workspace)) return SPARROW_ERR_INVALID_ARG;
    return select_impl(q, summaries, page_table, seq_lens, sd, sel_pages, max_sel, sel_count, scores_dbg, workspace,
                       workspace_bytes, shape, (cudaStream_t)stream);
}

}  // extern "C"

// ---- sparrow_select_static: page selection for callers that have no way to hand the library a workspace ----------------
// The selector needs scratch beyond its inputs and outputs (one arrival counter per (sequence, kv-head) unit and the fp32
// page scores the unit's last CTA ranks).  sparrow_select takes that from the caller; this variant takes it from the
// array below, which is part of the library image: the driver places it in every GPU's memory when the library is loaded
// on that GPU and keeps it until the process exits.  Nothing here calls cudaMalloc / cudaFree or any routine that does.
//
// In HOST code the name g_select_static_scratch is only a handle for the symbol: it is not a device address, and a kernel
// given it would read and write the wrong memory.  The address a kernel can use comes from cudaGetSymbolAddress, asked
// once per device with that device current (each GPU has its own copy of the array at its own address).
namespace {
static __device__ __align__(256) unsigned char g_select_static_scratch[SPARROW_SELECT_STATIC_BYTES];

void *g_select_static_ptr[kMaxDevices];             // per device: the array's device address (nullptr = not asked yet)
std::mutex g_select_static_mutex;

// The array's address on the calling thread's current device; first call per device does the look-up (a synchronous
// runtime call, which is why the header asks for that first call to come before any stream capture).
void *select_static_scratch(int *rc)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= kMaxDevices) {
        snprintf(g_errbuf, sizeof(g_errbuf), "cudaGetDevice failed or device ordinal >= %d", kMaxDevices);
        *rc = SPARROW_ERR_CUDA;
        return nullptr;
    }
    std::lock_guard<std::mutex> lock(g_select_static_mutex);
    if (!g_select_static_ptr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_select_static_scratch);
        if (e != cudaSuccess || !p) {
            snprintf(g_errbuf, sizeof(g_errbuf), "cudaGetSymbolAddress(select static scratch) on device %d: %s", dev,
                     cudaGetErrorString(e));
            *rc = SPARROW_ERR_CUDA;
            return nullptr;
        }
        g_select_static_ptr[dev] = p;
    }
    return g_select_static_ptr[dev];
}
}  // namespace

extern "C" {

size_t sparrow_select_static_bytes(void) { return SPARROW_SELECT_STATIC_BYTES; }

int sparrow_select_static(const void *q, const void *summaries, const int32_t *page_table, const int32_t *seq_lens,
                          const sparrow_schedule_t *sched, int32_t *sel_pages, int32_t max_sel, int32_t *sel_count,
                          float *scores_dbg, const sparrow_shape_t *shape, void *stream)
{
    g_launches = 0;
    int rc = check_shape(shape);
    if (rc) return rc;
    SchedDev sd;
    rc = to_dev_sched(sched, &sd, shape->page_size);
    if (rc) return rc;
    if (!q || !summaries || !page_table || !seq_lens || !sel_pages || !sel_count || max_sel <= 0) return SPARROW_ERR_INVALID_ARG;
    if (!aligned16(q) || !aligned16(summaries)) return SPARROW_ERR_INVALID_ARG;
    const size_t need = sparrow_select_workspace_bytes(shape);
    if (need > SPARROW_SELECT_STATIC_BYTES) return SPARROW_ERR_STATIC_SCRATCH_TOO_SMALL;   // before any CUDA call
    if (shape->n_seq == 0) return SPARROW_OK;
    void *ws = select_static_scratch(&rc);
    if (!ws) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    // The array still holds whatever the previous call (possibly of another shape, possibly one that failed half-way)
    // left in it.  Only the arrival counters must start at zero -- every score the ranking reads is written by this call
    // first -- so they are cleared here, on the caller's stream, ahead of the kernel.
    cudaError_t e = cudaMemsetAsync(ws, 0, select_ctr_bytes(shape), st);
    if (e != cudaSuccess) return cuda_fail(e, "memset(select static scratch counters)");
    return select_impl(q, summaries, page_table, seq_lens, sd, sel_pages, max_sel, sel_count, scores_dbg, ws,
                       SPARROW_SELECT_STATIC_BYTES, shape, st);
}

int sparrow_sparse_decode(const void *q, const void *k_cache, const void *v_cache, const int32_t *page_table,
                          const int32_t *seq_lens, const int32_t *sel_pages, int32_t max_sel, const int32_t *sel_count,
                          void *out, float *lse, float sm_scale, void *workspace, size_t workspace_bytes,
                          const sparrow_shape_t *shape, void *stream)
{
    g_launches = 0;
    int rc = check_shape(shape);
    if (rc) return rc;
    if (!q || !k_cache || !v_cache || !page_table || !seq_lens || !sel_pages || !sel_count || !out || !workspace || max_sel <= 0)
        return SPARROW_ERR_INVALID_ARG;
    if (!aligned16(q) || !aligned16(k_cache) || !aligned16(v_cache) || !aligned16(out) || !aligned16(workspace))
        return SPARROW_ERR_INVALID_ARG;
    return launch_decode<false>(q, k_cache, v_cache, page_table, seq_lens, sel_pages, max_sel, sel_count, out, lse,
                                sm_scale, workspace, workspace_bytes, shape, (cudaStream_t)stream);
}

int sparrow_dense_decode(const void *q, const void *k_cache, const void *v_cache, const int32_t *page_table,
                         const int32_t *seq_lens, void *out, float *lse, float sm_scale, void *workspace,
                         size_t workspace_bytes, const sparrow_shape_t *shape, void *stream)
{
    g_launches = 0;
    int rc = check_shape(shape);
    if (rc) return rc;
    if (!q || !k_cache || !v_cache || !page_table || !seq_lens || !out || !workspace) return SPARROW_ERR_INVALID_ARG;
    if (!aligned16(q) || !aligned16(k_cache) || !aligned16(v_cache) || !aligned16(out) || !aligned16(workspace))
        return SPARROW_ERR_INVALID_ARG;
    return launch_decode<true>(q, k_cache, v_cache, page_table, seq_lens, nullptr, 0, nullptr, out, lse, sm_scale,
                               workspace, workspace_bytes, shape, (cudaStream_t)stream);
}

int sparrow_append(const void *k_new, const void *v_new, void *k_cache, void *v_cache, void *summaries,
                   const int32_t *page_table, int32_t *seq_lens, const sparrow_shape_t *shape, void *stream)
{
    g_launches = 0;
    int rc = check_shape(shape);
    if (rc) return rc;
    if (!k_new || !v_new || !k_cache || !v_cache || !summaries || !page_table || !seq_lens) return SPARROW_ERR_INVALID_ARG;
    if (!aligned16(k_new) || !aligned16(v_new) || !aligned16(k_cache) || !aligned16(v_cache) || !aligned16(summaries))
        return SPARROW_ERR_INVALID_ARG;
    if (shape->n_seq == 0) return SPARROW_OK;
    const int warps = shape->n_kv_heads < kAppendMaxWarps ? shape->n_kv_heads : kAppendMaxWarps;
    launch_chain(append_kernel, dim3(shape->n_seq), dim3(warps * 32), 0, (cudaStream_t)stream, (const uint16_t *)k_new,
                 (const uint16_t *)v_new, (uint16_t *)k_cache, (uint16_t *)v_cache, (uint16_t *)summaries, page_table, seq_lens,
                 shape->n_kv_heads, shape->max_pages_per_seq, shape->page_size, shape->landmark, kv_layout(shape, nullptr));
    SPARROW_CHECK_LAUNCH("append_kernel");
    return SPARROW_OK;
}

size_t sparrow_acceptance_workspace_bytes(int32_t n_bins)
{
    if (n_bins <= 0) return 0;
    return align256((size_t)n_bins * kAccDigits * sizeof(int32_t)) + align256((size_t)n_bins * 4 * sizeof(uint32_t));
}

int sparrow_acceptance(const int32_t *ids_p, const float *logp_p, const int32_t *ids_q, const float *logp_q,
                       const int32_t *positions, int64_t n_pos, int32_t top_n, int32_t bin_tokens, int32_t n_bins,
                       float quantile, float *alpha, float *bin_quantile, int32_t *bin_count, void *workspace,
                       size_t workspace_bytes, void *stream)
{
    g_launches = 0;
    if (n_pos < 0 || top_n < 1 || top_n > 32 || bin_tokens <= 0 || n_bins <= 0 || n_bins > 65535 || !(quantile > 0.f) || !(quantile <= 1.f))
        return SPARROW_ERR_INVALID_ARG;
    if (!bin_quantile || !bin_count || !workspace) return SPARROW_ERR_INVALID_ARG;
    if (n_pos > 0 && (!ids_p || !logp_p || !ids_q || !logp_q || !positions || !alpha)) return SPARROW_ERR_INVALID_ARG;
    if (workspace_bytes < sparrow_acceptance_workspace_bytes(n_bins)) return SPARROW_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t st = (cudaStream_t)stream;
    int32_t *hist = reinterpret_cast<int32_t *>(workspace);
    uint32_t *state = reinterpret_cast<uint32_t *>(reinterpret_cast<uint8_t *>(workspace) +
                                                   align256((size_t)n_bins * kAccDigits * sizeof(int32_t)));
    cudaError_t e = cudaMemsetAsync(state, 0, (size_t)n_bins * 4 * sizeof(uint32_t), st);
    if (e != cudaSuccess) return cuda_fail(e, "memset(acceptance state)");
    if (n_pos > 0) {
        const int64_t blocks = (n_pos + kAlphaThreads - 1) / kAlphaThreads;
        if (blocks > 0x7fffffffLL) return SPARROW_ERR_UNSUPPORTED;
        const size_t asmem = (size_t)4 * kAlphaThreads * (top_n | 1) * sizeof(int);
        const int vec16 = (top_n & 3) == 0 && aligned16(ids_p) && aligned16(ids_q) && aligned16(logp_p) && aligned16(logp_q);
        int rc_dev = SPARROW_OK;
        DevState *ds = dev_state(&rc_dev);
        if (!ds) return rc_dev;
        if (top_n <= 20) {
            if ((rc_dev = ensure_dyn_smem(accept_alpha_kernel<20>, asmem, &ds->dyn_alpha[0], "accept_alpha_kernel<20>"))) return rc_dev;
            accept_alpha_kernel<20><<<(unsigned)blocks, kAlphaThreads, asmem, st>>>(ids_p, logp_p, ids_q, logp_q, n_pos, top_n, vec16, alpha);
        } else {
            if ((rc_dev = ensure_dyn_smem(accept_alpha_kernel<kAlphaMaxTop>, asmem, &ds->dyn_alpha[1], "accept_alpha_kernel<32>"))) return rc_dev;
            accept_alpha_kernel<kAlphaMaxTop><<<(unsigned)blocks, kAlphaThreads, asmem, st>>>(ids_p, logp_p, ids_q, logp_q, n_pos, top_n, vec16, alpha);
        }
        SPARROW_CHECK_LAUNCH("accept_alpha_kernel");
    }
    // 3-pass radix select per bin over the fp32 bit patterns: bits 31..21, 20..10, 9..0
    const int shifts[3] = {21, 10, 0}, bits[3] = {11, 11, 10};
    // bins per histogram block: as many 8 KiB histograms as fit in 200 KiB of shared memory (one CTA per SM then)
    const int bins_per_group = n_bins < 25 ? n_bins : 25;
    const int groups = (n_bins + bins_per_group - 1) / bins_per_group;
    const size_t hsmem = (size_t)bins_per_group * kAccDigits * sizeof(int);
    {
        int rc_dev = SPARROW_OK;
        DevState *ds = dev_state(&rc_dev);
        if (!ds) return rc_dev;
        rc_dev = ensure_dyn_smem(accept_hist_kernel, hsmem, &ds->dyn_hist, "accept_hist_kernel");
        if (rc_dev) return rc_dev;
    }
    int64_t gx = (n_pos + kHistThreads * 8 - 1) / (kHistThreads * 8);
    const int64_t gmax = kNumSmsB200;                    // one 1024-thread CTA per SM
    gx = gx < 1 ? 1 : (gx > gmax ? gmax : gx);
    for (int pass = 0; pass < 3; ++pass) {
        accept_hist_kernel<<<dim3((unsigned)gx, (unsigned)groups), kHistThreads, hsmem, st>>>(
            alpha, positions, n_pos, bin_tokens, n_bins, bins_per_group, shifts[pass], bits[pass], state, hist);
        SPARROW_CHECK_LAUNCH("accept_hist_kernel");
        accept_scan_kernel<<<n_bins, kAccThreads, 0, st>>>(hist, state, shifts[pass], bits[pass], pass == 0, quantile, pass == 2,
                                                           bin_quantile, bin_count);
        SPARROW_CHECK_LAUNCH("accept_scan_kernel");
    }
    return SPARROW_OK;
}

// Device scratch of the host-buffer step, carved in this order (each 256-byte aligned):
//   q | seq_lens | page_ids | n_valid   (the image of the caller's pinned host block: ONE H2D copy brings it over)
//   | sel_pages | sel_count | out | select workspace | decode workspace
namespace {
struct StepCarve {
    size_t q, lens, ids, nval, in_end, sel, cnt, out, sel_ws, dec_ws, total;
    size_t sel_ws_bytes, dec_ws_bytes;
};
StepCarve step_carve(const sparrow_shape_t *s, int32_t max_sel)
{
    StepCarve c;
    size_t o = 0;
    const size_t n = (size_t)s->n_seq;
    c.q = o; o += align256(n * s->n_q_heads * kDim * 2);
    c.lens = o; o += align256(n * 4);
    c.ids = o; o += align256(n * 4);               // at most one page per sequence fills in a step
    c.nval = o; o += align256(n * 4);
    c.in_end = o;
    c.sel = o; o += align256(n * s->n_kv_heads * (size_t)(max_sel > 0 ? max_sel : 1) * 4);
    c.cnt = o; o += align256(n * 4);
    c.out = o; o += align256(n * s->n_q_heads * kDim * 2);
    c.sel_ws_bytes = align256(sparrow_select_workspace_bytes(s));
    c.sel_ws = o; o += c.sel_ws_bytes;
    c.dec_ws_bytes = sparrow_decode_workspace_bytes(s, 0);       // one decode workspace serves the sparse and the dense call
    c.dec_ws = o; o += c.dec_ws_bytes;
    c.total = o;
    return c;
}
}  // namespace

size_t sparrow_step_scratch_bytes(const sparrow_shape_t *s, int32_t max_sel)
{
    if (check_shape(s) != SPARROW_OK) return 0;
    return step_carve(s, max_sel).total;
}

size_t sparrow_step_host_block_bytes(const sparrow_shape_t *s, size_t *off_seq_lens, size_t *off_page_ids, size_t *off_n_valid)
{
    if (check_shape(s) != SPARROW_OK) return 0;
    const StepCarve c = step_carve(s, 1);
    if (off_seq_lens) *off_seq_lens = c.lens;
    if (off_page_ids) *off_page_ids = c.ids;
    if (off_n_valid) *off_n_valid = c.nval;
    return c.in_end;
}

namespace {
int step_host_impl(const void *in_block_host, int64_t n_update, int has_n_valid, const void *k_cache, const void *v_cache,
                   void *summaries, const int32_t *page_table, const sparrow_schedule_t *sched, int32_t max_sel,
                   float sm_scale, void *out_host, void *scratch, size_t scratch_bytes, const sparrow_shape_t *s,
                   void *stream, bool wait)
{
    g_launches = 0;
    int rc = check_shape(s);
    if (rc) return rc;
    SchedDev sd;
    rc = to_dev_sched(sched, &sd, s->page_size);
    if (rc) return rc;
    if (!in_block_host || !k_cache || !v_cache || !summaries || !page_table || !out_host || !scratch || max_sel <= 0)
        return SPARROW_ERR_INVALID_ARG;
    if (n_update < 0 || n_update > s->n_seq) return SPARROW_ERR_INVALID_ARG;
    if (!aligned16(k_cache) || !aligned16(v_cache) || !aligned16(summaries) || !aligned16(scratch)) return SPARROW_ERR_INVALID_ARG;
    const StepCarve c = step_carve(s, max_sel);
    if (scratch_bytes < c.total) return SPARROW_ERR_WORKSPACE_TOO_SMALL;
    cudaStream_t st = (cudaStream_t)stream;
    uint8_t *base = reinterpret_cast<uint8_t *>(scratch);
    const size_t qbytes = (size_t)s->n_seq * s->n_q_heads * kDim * 2;
    // one copy for the step's inputs: the block up to the end of what this step uses
    const size_t in_bytes = n_update == 0 ? c.lens + (size_t)s->n_seq * 4
                                          : (has_n_valid ? c.nval : c.ids) + (size_t)n_update * 4;
    cudaError_t e;
    if ((e = cudaMemcpyAsync(base, in_block_host, in_bytes, cudaMemcpyHostToDevice, st)) != cudaSuccess) return cuda_fail(e, "H2D step inputs");
    const int32_t *lens_d = reinterpret_cast<const int32_t *>(base + c.lens);
    if (n_update > 0) {
        rc = summarize_impl(k_cache, summaries, reinterpret_cast<const int32_t *>(base + c.ids),
                            has_n_valid ? reinterpret_cast<const int32_t *>(base + c.nval) : nullptr, n_update, s, st);
        if (rc) return rc;
    }
    if (sd.kind == SPARROW_SCHED_DENSE) {
        rc = launch_decode<true>(base + c.q, k_cache, v_cache, page_table, lens_d, nullptr, 0, nullptr, base + c.out, nullptr,
                                 sm_scale, base + c.dec_ws, c.dec_ws_bytes, s, st);
    } else {
        rc = select_impl(base + c.q, summaries, page_table, lens_d, sd, reinterpret_cast<int32_t *>(base + c.sel), max_sel,
                         reinterpret_cast<int32_t *>(base + c.cnt), nullptr, base + c.sel_ws, c.sel_ws_bytes, s, st);
        if (rc) return rc;
        rc = launch_decode<false>(base + c.q, k_cache, v_cache, page_table, lens_d, reinterpret_cast<int32_t *>(base + c.sel),
                                  max_sel, reinterpret_cast<int32_t *>(base + c.cnt), base + c.out, nullptr, sm_scale,
                                  base + c.dec_ws, c.dec_ws_bytes, s, st);
    }
    if (rc) return rc;
    if ((e = cudaMemcpyAsync(out_host, base + c.out, qbytes, cudaMemcpyDeviceToHost, st)) != cudaSuccess) return cuda_fail(e, "D2H out");
    if (wait && (e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e, "stream sync");
    return SPARROW_OK;
}
}  // namespace

int sparrow_step_host(const void *in_block_host, int64_t n_update, int has_n_valid, const void *k_cache, const void *v_cache,
                      void *summaries, const int32_t *page_table, const sparrow_schedule_t *sched, int32_t max_sel,
                      float sm_scale, void *out_host, void *scratch, size_t scratch_bytes, const sparrow_shape_t *s,
                      void *stream)
{
    return step_host_impl(in_block_host, n_update, has_n_valid, k_cache, v_cache, summaries, page_table, sched, max_sel, sm_scale,
                          out_host, scratch, scratch_bytes, s, stream, true);
}

int sparrow_step_host_async(const void *in_block_host, int64_t n_update, int has_n_valid, const void *k_cache, const void *v_cache,
                            void *summaries, const int32_t *page_table, const sparrow_schedule_t *sched, int32_t max_sel,
                            float sm_scale, void *out_host, void *scratch, size_t scratch_bytes, const sparrow_shape_t *s,
                            void *stream)
{
    return step_host_impl(in_block_host, n_update, has_n_valid, k_cache, v_cache, summaries, page_table, sched, max_sel, sm_scale,
                          out_host, scratch, scratch_bytes, s, stream, false);
}

}  // extern "C"
