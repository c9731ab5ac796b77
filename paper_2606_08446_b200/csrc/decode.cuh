// decode.cuh -- kernel (c): split-K flash-decode over a page list with the log-sum-exp merge fused in.
// SURVEY.md 8(a) a6-a8; PAPER.md:140 (attention over the KV budget B), :131-135 (dense), north_star (c).
//
// Work decomposition ("stream-K" over pages): the (page, kv-head) tiles of the whole batch form ONE flat stream,
// ordered (sequence, kv-head, list position); its length T = Hkv * sum_i cnt_i is known from sel_count (or from
// seq_lens for the dense entry).  A persistent grid of one CTA per SM cuts it into equal contiguous CTA RANGES,
// whatever the mix of lengths and budgets.  Inside a CTA the work is warp-specialised:
//
//   * ONE PRODUCER WARP walks the CTA's range.  It resolves flat tile -> (sequence, kv-head, list position) ->
//     logical page -> physical tile in windows of 32 tiles (lane = tile; three look-up stages so that no stage
//     consumes a load issued by the stage before it in the same breath), and one elected lane issues the copies:
//     the 4 KiB K tile and the 4 KiB V tile of a page are each two TMA boxes of 16 tokens x 64 dims
//     (cp.async.bulk.tensor.2d, SWIZZLE_128B, mbarrier complete_tx) into a CTA-wide ring of kDecStages stages.
//   * EIGHT CONSUMER WARPS take the ring's tiles round-robin (tile i of the range -> consumer i mod 8), each with its
//     own online-softmax state for the (sequence, kv-head) unit the CTA is in.  When the CTA's part of a unit ends
//     the consumers park their (o, m, l) in shared memory, meet at a named barrier and merge: consumer h merges query
//     head h of the group.  The result is final (written straight to `out`) when the unit lies inside the CTA's
//     range; otherwise it is the CTA's partial, parked in slot unit + CTA index of a small fp32 workspace, and the
//     CTA that arrives last on the unit's counter merges the CTAs' partials in stream order (a7; no second launch).
//
// Why this shape (round 2): with one private stream per warp (round 1) a warp's progress is a sum of
// ~50 saturated-HBM latencies, the per-warp finish times spread with sigma ~7 us on a 90 us launch and the kernel
// ends with the slowest of 1184 warps (traced: median 80 us, maximum 97 us at cfg2).  A CTA-wide ring averages the
// latencies over eight times as many tiles, keeps 128 KiB in flight per SM whatever a single warp is doing, and the
// static round-robin keeps the summation order -- and so the result -- bit-for-bit reproducible.
// The whole GQA group (r <= 8 query heads) is processed together, so each K/V byte is read from HBM once.
//
// Shared layout of a tile: [half = dim/64][token 0..15][64 dims = 8 chunks of 16 B], chunk index XOR (token & 7) --
// exactly what a 16 x 64 box lands as under SWIZZLE_128B, conflict-free for ldmatrix.
//
// Math: the products are a [heads x 128] x [128 x 16 tokens] and a [heads x 16] x [16 x 128] contraction per page;
// at r >= 4 the plain FP32 pipes cannot keep up with HBM ("ALU budget"), so both run on the tensor
// cores with the query heads as the (zero-padded) M = 16 rows of mma.sync.m16n8k16 bf16 -> fp32:
//   S[head][token] = sum_d Q[head][d] K[token][d]     A = Q fragments (registers), B = K via ldmatrix
//   O[head][d]    += sum_t P[head][t] V[t][d]         A = P (bf16, from the S accumulators), B = V via ldmatrix.trans
// Softmax statistics (running max m in the log2 domain, sum l) are fp32.
#pragma once
#include <cuda.h>

#include "common.cuh"

namespace sparrow {

constexpr int kDecConsumers = 8;                                // consumer warps; consumer h also merges query head h
constexpr int kDecThreads = (kDecConsumers + 1) * 32;           // + the producer warp
#ifndef SPARROW_DEC_STAGES
#define SPARROW_DEC_STAGES 16
#endif
constexpr int kDecStages = SPARROW_DEC_STAGES;                  // CTA-wide ring depth (tiles in flight per SM)
constexpr int kStageBytes = 2 * kTileBytes;                     // K tile + V tile = 8 KiB
constexpr int kDecRingBytes = kDecStages * kStageBytes;         // 128 KiB
constexpr int kMaxGroup = 8;                                    // r <= 8 (rows 0..7 of the m16 tile)
static_assert(kMaxGroup <= kDecConsumers, "consumer h merges query head h");
#ifndef SPARROW_DEC_MAXSEQ
#define SPARROW_DEC_MAXSEQ 8192
#endif
constexpr int kDecMaxSeq = SPARROW_DEC_MAXSEQ;                  // prefix table of the batch lives in shared memory
constexpr int kDecGrid = 148;                                   // persistent: one CTA per B200 SM (fewer SMs: fewer CTAs)
constexpr int kParkRow = kDim + 4;                              // one parked head: o[128] | m | l | pad (16-byte rows)
constexpr int kDecParkBytes = kDecConsumers * kMaxGroup * kParkRow * 4;
constexpr int kDecMetaBytes = kDecStages * 4 + 2 * kDecStages * 8 + 64;   // valid counts | full / empty barriers | flag

__device__ __forceinline__ void ldsm_x4(uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3, uint32_t addr)
{
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_t(uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3, uint32_t addr)
{
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
// D(16x8) += A(16x16) B(16x8) with rows 8..15 of A identically zero (query heads pad the M tile):
// only c0, c1 (rows 0..7) are live; a1 = a3 = 0 and the row-8..15 outputs are discarded.
__device__ __forceinline__ void mma_rows07(float &c0, float &c1, uint32_t a0, uint32_t a2, uint32_t b0, uint32_t b1)
{
    float d2, d3;
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%5}, {%7,%8}, {%0,%1,%9,%9};"
                 : "+f"(c0), "+f"(c1), "=f"(d2), "=f"(d3)
                 : "r"(a0), "r"(0u), "r"(a2), "r"(b0), "r"(b1), "f"(0.f));
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi)
{
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
    return *reinterpret_cast<uint32_t *>(&v);
}
__device__ __forceinline__ float fast_exp2(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Swizzled byte offset of 16-byte chunk c (0..15) of token row t inside a 4 KiB tile.
__device__ __forceinline__ uint32_t tile_off(int t, int c)
{
    return (uint32_t)((c >> 3) * 2048 + t * 128 + (((c & 7) ^ (t & 7)) << 4));
}

// One TMA box: 16 rows x 64 bf16 columns of the [rows][128] view of a K or V pool, starting at (col, row), into 2 KiB of
// shared memory (SWIZZLE_128B), completing 2048 bytes on `bar`.
__device__ __forceinline__ void tma_box(uint32_t dst, const CUtensorMap *tm, int col, int row, uint32_t bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tm)), "r"(col), "r"(row), "r"(bar) : "memory");
}
// named barrier of the consumer warps (the producer never joins it)
__device__ __forceinline__ void consumer_sync() { asm volatile("bar.sync 1, %0;" ::"n"(kDecConsumers * 32) : "memory"); }

// Everything the decode needs (kernel arguments, passed on unchanged).
struct DecodeArgs {
    const uint16_t *q;
    const int32_t *page_table, *seq_lens, *sel_pages, *sel_count;
    int max_sel;
    float *ws_o, *ws_ml;         // CTA partials: [units + grid][r][128] and [..][r][2] (m, l)
    int32_t *counters;           // [units] CTAs arrived per unit (zero between calls)
    uint16_t *out;
    float *lse;
    float scale_log2;
    int n_seq, n_q_heads, n_kv_heads, max_pages;
    int tpp_log2;                // log2 of the 16-token tiles per page (page size 16, 32, 64, 128 -> 0, 1, 2, 3)
};

// The CTA ranges: T tiles over G CTAs, the first `extra` CTAs one tile longer.
struct CtaRanges {
    int per, extra;
    __device__ __forceinline__ int begin(int b) const { return b * per + (b < extra ? b : extra); }
    __device__ __forceinline__ int owner(int t) const
    {
        const int cut = extra * (per + 1);
        return t < cut ? t / (per + 1) : extra + (t - cut) / per;       // t >= cut implies per >= 1
    }
};

template <bool kDense>
__global__ void __launch_bounds__(kDecThreads, 1)
decode_kernel(const DecodeArgs A, const __grid_constant__ CUtensorMap tm_k, const __grid_constant__ CUtensorMap tm_v)
{
    chain_entry();
    extern __shared__ __align__(1024) uint8_t smem[];
    float *s_park = reinterpret_cast<float *>(smem + kDecRingBytes);                          // [consumer][head][kParkRow]
    int32_t *s_valid = reinterpret_cast<int32_t *>(smem + kDecRingBytes + kDecParkBytes);     // [stage] valid tokens of the tile
    uint64_t *s_full = reinterpret_cast<uint64_t *>(s_valid + kDecStages);                    // [stage] tile has landed
    uint64_t *s_empty = s_full + kDecStages;                                                  // [stage] consumer is done with it
    int32_t *s_flag = reinterpret_cast<int32_t *>(s_empty + kDecStages);                      // arrival result of the current unit
    int32_t *s_prefix = reinterpret_cast<int32_t *>(smem + kDecRingBytes + kDecParkBytes + kDecMetaBytes);   // [n_seq + 1] tiles per kv-head before sequence i
    __shared__ int s_scan[kDecThreads / 32];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n_seq = A.n_seq, n_kv_heads = A.n_kv_heads, max_sel = A.max_sel, max_pages = A.max_pages;
    const int r = A.n_q_heads / n_kv_heads;
    constexpr uint32_t kFull = 0xffffffffu;
    const uint32_t ring_u32 = smem_u32(smem);
    const uint32_t full_u32 = smem_u32(s_full), empty_u32 = smem_u32(s_empty);

    // ---- prologue: barriers; list length of every sequence -> exclusive prefix in shared memory ----
    if (tid == 0) {
        for (int s = 0; s < kDecStages; ++s) {
            mbar_init(full_u32 + 8 * s, 1);              // the producer's arrive.expect_tx; the copies complete the bytes
            mbar_init(empty_u32 + 8 * s, 1);             // lane 0 of the tile's consumer
        }
        fence_mbar_init();
    }
    {
        const int per = (n_seq + kDecThreads - 1) / kDecThreads;
        const int s0 = min(tid * per, n_seq), s1 = min(s0 + per, n_seq);
        auto count_of = [&](int s) {
            int c;
            const int page_tokens = kPage << A.tpp_log2;
            if (kDense) c = (__ldg(A.seq_lens + s) + page_tokens - 1) / page_tokens;
            else { c = __ldg(A.sel_count + s); c = c < max_sel ? c : max_sel; }
            return c > 0 ? c << A.tpp_log2 : 0;                  // in 16-token tiles
        };
        int sum = 0;
        for (int s = s0; s < s1; ++s) sum += count_of(s);
        int inc = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(kFull, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) s_scan[warp] = inc;
        __syncthreads();
        int run = inc - sum;
        for (int w = 0; w < warp; ++w) run += s_scan[w];
        for (int s = s0; s < s1; ++s) {
            s_prefix[s] = run;
            run += count_of(s);
        }
        if (tid == kDecThreads - 1) s_prefix[n_seq] = run;
        __syncthreads();
    }
    const int T = s_prefix[n_seq] * n_kv_heads;                  // tiles of the whole batch
    CtaRanges cr;
    cr.per = T / (int)gridDim.x;
    cr.extra = T - cr.per * (int)gridDim.x;
    const int ra = cr.begin(blockIdx.x), rb = cr.begin(blockIdx.x + 1);         // this CTA's tiles [ra, rb)
    if (ra >= rb) return;
    // sequence that holds flat tile p: the last one whose first tile is <= p and that is not empty
    auto seq_of = [&](int p) {
        int lo = 0, hi = n_seq - 1;
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (s_prefix[mid] * n_kv_heads <= p) lo = mid; else hi = mid - 1;
        }
        while (s_prefix[lo + 1] * n_kv_heads <= p) ++lo;         // empty lists share a prefix
        return lo;
    };

    if (warp == kDecConsumers) {
        // =========================================================== PRODUCER ===========================================
        // Look-up of flat tile p -> (sequence, kv-head, list position) -> logical page -> physical tile, as three stages
        // so that no stage consumes a load issued by the stage before it in the same breath.  A WINDOW is up to 32
        // consecutive tiles of the CTA's range, lane = tile.
        struct Lookup {
            int tile;        // stage C: index of the 4 KiB K (and V) tile in the pools
            int valid;       // stage B: valid tokens of the tile (0..16)
            int seq, unit, logical, len, phys, sub;
        };
        auto stage_a = [&](Lookup &m, int p, bool on) {
            m.tile = 0; m.valid = 0; m.seq = -1; m.unit = 0; m.logical = 0; m.len = 0; m.phys = 0; m.sub = 0;
            if (on) {
                const int seq = seq_of(p), base = s_prefix[seq], c = s_prefix[seq + 1] - base;
                const int rem = p - base * n_kv_heads;
                const int g = rem / c, i = rem - g * c;
                m.seq = seq;
                m.unit = seq * n_kv_heads + g;
                const int pi = i >> A.tpp_log2;                  // list position of the tile's page
                m.sub = i - (pi << A.tpp_log2);
                m.logical = kDense ? pi : __ldg(A.sel_pages + ((int64_t)m.unit) * max_sel + pi);
                m.len = __ldg(A.seq_lens + seq);
            }
        };
        auto stage_b = [&](Lookup &m) {
            if (m.seq >= 0) {
                m.phys = __ldg(A.page_table + (int64_t)m.seq * max_pages + m.logical);
                int valid = m.len - ((m.logical << A.tpp_log2) + m.sub) * kPage;
                m.valid = valid < 0 ? 0 : (valid > kPage ? kPage : valid);
            }
        };
        auto stage_c = [&](Lookup &m) { m.tile = ((m.phys * n_kv_heads + (m.unit - m.seq * n_kv_heads)) << A.tpp_log2) + m.sub; };

        int rp = ra;                                             // next tile not yet in a window
        auto open_window = [&](Lookup &m, int &n) {
            n = min(32, rb - rp);
            stage_a(m, rp + lane, lane < n);
            rp += n;
        };
        Lookup cur, nxt;
        int cn, nn, nxt_stage;                                   // tiles of the two windows; look-up stages of `nxt` done (1 = A, 2 = B, 3 = C)
        open_window(cur, cn);
        if (rp < rb) { open_window(nxt, nn); nxt_stage = 1; } else { nn = 0; nxt_stage = 3; }
        stage_b(cur);
        stage_c(cur);
        auto advance_nxt = [&](int target) {                     // warp-uniform
            if (nxt_stage < 2 && target >= 2) { stage_b(nxt); nxt_stage = 2; }
            if (nxt_stage < 3 && target >= 3) { stage_c(nxt); nxt_stage = 3; }
        };
        int it = 0;                                              // tiles issued so far: tile `it` goes to stage it % kDecStages
#pragma unroll 1
        while (cn > 0) {
            // look-up stages B and C of the next window run a third and two thirds of the way through this one
            const int jc = cn >= 24 ? 16 : max(0, min((2 * cn) / 3, cn - 2));
            const int jb = cn >= 24 ? 8 : min(cn / 3, jc);
#pragma unroll 1
            for (int j = 0; j < cn; ++j, ++it) {
                if (j == jb) advance_nxt(2);
                if (j == jc) advance_nxt(3);
                const int stage = it % kDecStages, use = it / kDecStages;
                const int tile = __shfl_sync(kFull, cur.tile, j), valid = __shfl_sync(kFull, cur.valid, j);
                if (lane == 0) {
                    if (use > 0) mbar_wait(empty_u32 + 8 * stage, (use - 1) & 1);      // its previous tile has been consumed
                    s_valid[stage] = valid;
                    const uint32_t bar = full_u32 + 8 * stage, dst = ring_u32 + stage * kStageBytes;
                    mbar_arrive_expect_tx(bar, kStageBytes);     // (release: orders the store of `valid` before the consumer's wait)
                    const int row = tile * kPage;
                    tma_box(dst, &tm_k, 0, row, bar);
                    tma_box(dst + 2048, &tm_k, 64, row, bar);
                    tma_box(dst + kTileBytes, &tm_v, 0, row, bar);
                    tma_box(dst + kTileBytes + 2048, &tm_v, 64, row, bar);
                }
                __syncwarp();
            }
            advance_nxt(3);
            cur = nxt; cn = nn;
            if (cn > 0 && rp < rb) { open_window(nxt, nn); nxt_stage = 1; }
            else { nn = 0; nxt_stage = 3; }
        }
        return;
    }

    // =============================================================== CONSUMERS ===========================================
    const int hrow = lane >> 2, col = 2 * (lane & 3);               // this lane's query head and column pair
    const int mat = lane >> 3, rr = lane & 7;
    const float scale_log2 = A.scale_log2;
    constexpr float kLn2 = 0.6931471805599453f;
    int p = ra;
    int seq = seq_of(p);
#pragma unroll 1
    while (p < rb) {
        // ---- the CTA's part of one unit: tiles [p, e) of the stream; the unit is tiles [u0, u1) ----
        const int base = s_prefix[seq], c = s_prefix[seq + 1] - base;
        const int rem = p - base * n_kv_heads;
        const int g = rem / c;
        const int u0 = base * n_kv_heads + g * c, u1 = u0 + c;
        const int e = min(u1, rb);
        const int unit = seq * n_kv_heads + g;
        uint32_t qa[8][2];                                          // Q fragments of the unit
        {
            const uint16_t *qrow = A.q + ((int64_t)unit * r + hrow) * kDim + col;
#pragma unroll
            for (int kk = 0; kk < 8; ++kk) {
                qa[kk][0] = hrow < r ? __ldg(reinterpret_cast<const uint32_t *>(qrow + kk * 16)) : 0u;
                qa[kk][1] = hrow < r ? __ldg(reinterpret_cast<const uint32_t *>(qrow + kk * 16 + 8)) : 0u;
            }
        }
        float o[16][2];                 // O[head = lane/4][dims nt*8 + col + {0,1}]
#pragma unroll
        for (int nt = 0; nt < 16; ++nt) { o[nt][0] = 0.f; o[nt][1] = 0.f; }
        float m_run = -INFINITY, l_run = 0.f;

        // this consumer's tiles of the part: those whose index in the CTA's range is = warp (mod 8)
#pragma unroll 1
        for (int t = p + ((warp - (p - ra)) & (kDecConsumers - 1)); t < e; t += kDecConsumers) {
            const int it = t - ra, stage = it % kDecStages;
            mbar_wait(full_u32 + 8 * stage, (it / kDecStages) & 1);
            const int valid = s_valid[stage];
            const uint32_t kb = ring_u32 + stage * kStageBytes;
            const uint32_t vb = kb + kTileBytes;
            if (valid < kPage) {
                // Warp-uniform, at most one tile per unit (plus the sub-tiles past L of a larger page): token rows >= valid
                // hold whatever the pool held (an unwritten or recycled page).  Their scores are masked to -inf below, so
                // p = 0, but 0 x NaN/Inf in the P V product would still poison the output row: zero those V rows in the
                // stage (K needs nothing: a masked score is replaced, never multiplied).
                for (int idx = valid * 16 + lane; idx < kPage * 16; idx += 32)
                    asm volatile("st.shared.v4.u32 [%0], {%1,%1,%1,%1};" ::"r"(vb + tile_off(idx >> 4, idx & 15)), "r"(0u) : "memory");
                __syncwarp();
            }
            // ---- S = Q K^T: two n-tiles (tokens 0-7, 8-15), 8 k-steps ----
            float s0a = 0.f, s0b = 0.f, s1a = 0.f, s1b = 0.f;
#pragma unroll
            for (int kk = 0; kk < 8; ++kk) {
                uint32_t b0, b1, b2, b3;   // matrices: (tok 0-7, chunk 2kk) (tok 0-7, 2kk+1) (tok 8-15, 2kk) (tok 8-15, 2kk+1)
                ldsm_x4(b0, b1, b2, b3, kb + tile_off((mat >> 1) * 8 + rr, 2 * kk + (mat & 1)));
                mma_rows07(s0a, s0b, qa[kk][0], qa[kk][1], b0, b1);
                mma_rows07(s1a, s1b, qa[kk][0], qa[kk][1], b2, b3);
            }
            // ---- online softmax: this lane holds head lane/4, tokens col, col+1, col+8, col+9 of the page ----
            float x0 = col < valid ? s0a * scale_log2 : -INFINITY;
            float x1 = col + 1 < valid ? s0b * scale_log2 : -INFINITY;
            float x2 = col + 8 < valid ? s1a * scale_log2 : -INFINITY;
            float x3 = col + 9 < valid ? s1b * scale_log2 : -INFINITY;
            float mx = fmaxf(fmaxf(x0, x1), fmaxf(x2, x3));
            mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, 1));
            mx = fmaxf(mx, __shfl_xor_sync(kFull, mx, 2));
            const float m_new = fmaxf(m_run, mx);
            const float m_safe = m_new == -INFINITY ? 0.f : m_new;
            const float alpha = fast_exp2(m_run - m_safe);
            const float p0 = fast_exp2(x0 - m_safe), p1 = fast_exp2(x1 - m_safe);
            const float p2 = fast_exp2(x2 - m_safe), p3 = fast_exp2(x3 - m_safe);
            l_run = l_run * alpha + ((p0 + p1) + (p2 + p3));
            m_run = m_new;
            if (!__all_sync(kFull, alpha == 1.f)) {
#pragma unroll
                for (int nt = 0; nt < 16; ++nt) { o[nt][0] *= alpha; o[nt][1] *= alpha; }
            }
            const uint32_t pa0 = pack_bf16(p0, p1), pa2 = pack_bf16(p2, p3);
            // ---- O += P V: 16 n-tiles of 8 dims, one k-step (16 tokens) ----
#pragma unroll
            for (int jn = 0; jn < 8; ++jn) {
                uint32_t b0, b1, b2, b3;   // matrices: (tok 0-7, chunk 2jn) (tok 8-15, 2jn) (tok 0-7, 2jn+1) (tok 8-15, 2jn+1)
                ldsm_x4_t(b0, b1, b2, b3, vb + tile_off((mat & 1) * 8 + rr, 2 * jn + (mat >> 1)));
                mma_rows07(o[2 * jn][0], o[2 * jn][1], pa0, pa2, b0, b1);
                mma_rows07(o[2 * jn + 1][0], o[2 * jn + 1][1], pa0, pa2, b2, b3);
            }
            // ---- the stage is free: every lane has read it (the zeroing above was a generic-proxy WRITE: make it visible to
            // the async proxy before the copy engine may overwrite the stage) ----
            if (valid < kPage) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_u32 + 8 * stage);
        }

        // ---- park this consumer's state of the part; consumer h then merges query head h over the eight parked states ----
        {
            float l_tot = l_run;
            l_tot += __shfl_xor_sync(kFull, l_tot, 1);
            l_tot += __shfl_xor_sync(kFull, l_tot, 2);
            if (hrow < r) {
                float *row = s_park + (warp * kMaxGroup + hrow) * kParkRow;
#pragma unroll
                for (int nt = 0; nt < 16; ++nt) *reinterpret_cast<float2 *>(row + nt * 8 + col) = make_float2(o[nt][0], o[nt][1]);
                if ((lane & 3) == 0) *reinterpret_cast<float2 *>(row + kDim) = make_float2(m_run, l_tot);
            }
        }
        consumer_sync();
        const bool whole = u0 >= ra && u1 <= rb;                    // the unit lies inside this CTA's range: the result is final
        const int c_first = cr.owner(u0), c_last = cr.owner(u1 - 1);
        const int h = warp;                                         // the query head this consumer merges
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        float m_star = -INFINITY, l_star = 0.f;
        if (h < r) {
            float mw[kDecConsumers], lw[kDecConsumers];
#pragma unroll
            for (int w2 = 0; w2 < kDecConsumers; ++w2) {
                const float2 ml = *reinterpret_cast<const float2 *>(s_park + (w2 * kMaxGroup + h) * kParkRow + kDim);
                mw[w2] = ml.x; lw[w2] = ml.y;
                if (ml.y > 0.f) m_star = fmaxf(m_star, ml.x);
            }
#pragma unroll
            for (int w2 = 0; w2 < kDecConsumers; ++w2) {           // fixed order: the result does not depend on timing
                const float wgt = lw[w2] > 0.f ? fast_exp2(mw[w2] - m_star) : 0.f;      // empty state: weight 0, never NaN
                const float4 v = *reinterpret_cast<const float4 *>(s_park + (w2 * kMaxGroup + h) * kParkRow + lane * 4);
                l_star = fmaf(lw[w2], wgt, l_star);
                acc.x = fmaf(v.x, wgt, acc.x); acc.y = fmaf(v.y, wgt, acc.y);
                acc.z = fmaf(v.z, wgt, acc.z); acc.w = fmaf(v.w, wgt, acc.w);
            }
            if (whole) {
                const float inv = l_star > 0.f ? 1.f / l_star : 0.f;
                uint2 pk;
                pk.x = pack_bf16(acc.x * inv, acc.y * inv);
                pk.y = pack_bf16(acc.z * inv, acc.w * inv);
                *reinterpret_cast<uint2 *>(A.out + ((int64_t)unit * r + h) * kDim + lane * 4) = pk;
                if (A.lse && lane == 0)
                    A.lse[(int64_t)unit * r + h] = l_star > 0.f ? (m_star + log2f(l_star)) * kLn2 : -INFINITY;
            } else {
                const int64_t slot = (int64_t)unit + blockIdx.x;    // unique: unit + CTA index increases along the stream
                *reinterpret_cast<float4 *>(A.ws_o + (slot * r + h) * kDim + lane * 4) = acc;
                if (lane == 0) *reinterpret_cast<float2 *>(A.ws_ml + (slot * r + h) * 2) = make_float2(m_star, l_star);
            }
        }
        if (!whole) {
            // ---- arrival (a7): release / acquire through ONE atomic of one thread: the consumer barrier orders the eight
            // warps' partial stores before the acq_rel atomic (cumulative at gpu scope), and the barrier after it orders
            // that acquire before the other threads' reads of the other CTAs' slots (ld.global.cg below) ----
            consumer_sync();
            if (tid == 0) {
                int old;
                asm volatile("atom.acq_rel.gpu.global.add.s32 %0, [%1], 1;" : "=r"(old) : "l"(A.counters + unit) : "memory");
                const int last = old == c_last - c_first;
                if (last) A.counters[unit] = 0;                     // restore the zero for the next call
                *s_flag = last;
            }
            consumer_sync();
            if (*s_flag && h < r) {
                // the last CTA to arrive merges the CTAs' partials in stream order (deterministic)
                const int nseg = c_last - c_first + 1;
                const int64_t row0 = ((int64_t)unit + c_first) * r + h;                 // slot row of CTA c: row0 + (c - c_first) * r
                m_star = -INFINITY;
                for (int s0 = 0; s0 < nseg; s0 += 32) {
                    const int s = s0 + lane;
                    float2 ml = make_float2(-INFINITY, 0.f);
                    if (s < nseg) ml = __ldcg(reinterpret_cast<const float2 *>(A.ws_ml + (row0 + (int64_t)s * r) * 2));
                    float mm = ml.y > 0.f ? ml.x : -INFINITY;
#pragma unroll
                    for (int of = 16; of > 0; of >>= 1) mm = fmaxf(mm, __shfl_xor_sync(kFull, mm, of));
                    m_star = fmaxf(m_star, mm);
                }
                acc = make_float4(0.f, 0.f, 0.f, 0.f);
                l_star = 0.f;
                for (int s0 = 0; s0 < nseg; s0 += 4) {               // four partial rows requested together
                    float4 v[4];
                    float2 ml[4];
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        v[k] = make_float4(0.f, 0.f, 0.f, 0.f);
                        ml[k] = make_float2(-INFINITY, 0.f);
                        if (s0 + k < nseg) {
                            v[k] = __ldcg(reinterpret_cast<const float4 *>(A.ws_o + (row0 + (int64_t)(s0 + k) * r) * kDim + lane * 4));
                            ml[k] = __ldcg(reinterpret_cast<const float2 *>(A.ws_ml + (row0 + (int64_t)(s0 + k) * r) * 2));
                        }
                    }
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const float wgt = ml[k].y > 0.f ? fast_exp2(ml[k].x - m_star) : 0.f;
                        l_star = fmaf(ml[k].y, wgt, l_star);
                        acc.x = fmaf(v[k].x, wgt, acc.x); acc.y = fmaf(v[k].y, wgt, acc.y);
                        acc.z = fmaf(v[k].z, wgt, acc.z); acc.w = fmaf(v[k].w, wgt, acc.w);
                    }
                }
                const float inv = l_star > 0.f ? 1.f / l_star : 0.f;
                uint2 pk;
                pk.x = pack_bf16(acc.x * inv, acc.y * inv);
                pk.y = pack_bf16(acc.z * inv, acc.w * inv);
                *reinterpret_cast<uint2 *>(A.out + ((int64_t)unit * r + h) * kDim + lane * 4) = pk;
                if (A.lse && lane == 0)
                    A.lse[(int64_t)unit * r + h] = l_star > 0.f ? (m_star + log2f(l_star)) * kLn2 : -INFINITY;
            }
        }
        consumer_sync();                                            // the parked states (and the flag) are free again
        // ---- next unit ----
        p = e;
        if (e == u1 && g + 1 == n_kv_heads) {
            ++seq;
            while (seq < n_seq && s_prefix[seq + 1] == s_prefix[seq]) ++seq;            // sequences with an empty list
        }
    }
}

}  // namespace sparrow
