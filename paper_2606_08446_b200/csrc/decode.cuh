// decode.cuh -- kernel (c): split-K flash-decode over a page list with the log-sum-exp merge fused in.
// SURVEY.md 8(a) a6-a8; PAPER.md:140 (attention over the KV budget B), :131-135 (dense), north_star (c).
//
// Work decomposition ("stream-K" over pages, self-scheduled): the (page, kv-head) tiles of the whole batch form
// ONE flat stream, ordered (sequence, kv-head, list position); its length T = Hkv * sum_i cnt_i is known from
// sel_count (or from seq_lens for the dense entry).  A persistent grid of one CTA per SM streams it, each warp a
// contiguous RANGE of tiles.  Default: ONE round of equal static ranges (range index = warp index, no atomic).  A
// factoring self-scheduler is built in but opt-in (SPARROW_DEC_R0_EIGHTHS < 8: round 0 hands out that many eighths
// of the fair share, every later round half of what is left, a warp that runs out takes the next range index from
// one atomic counter): measured slower, because every extra range adds a partial and a merge on the critical path
// (DESIGN.md 6.3).  The ranges are a pure function of T, which every warp evaluates from a small table in shared
// memory.  A range that crosses a (sequence, kv-head) boundary closes one softmax state and opens the next; the K/V
// ring keeps running across range boundaries.
// The whole GQA group (r <= 8 query heads) is processed together, so each K/V byte is read from HBM once.
//
// Split-K merge (a7): a (sequence, kv-head) unit covered by one range is normalised and written straight to `out`;
// otherwise each covering range parks its un-normalised (o, m, l) in slot unit + range index of a small fp32
// workspace (unit + range index is strictly increasing along the stream, hence unique) and bumps the unit's
// counter; the warp that arrives last merges the slots in stream order (deterministic; lanes load the slots'
// (m, l) pairs in parallel, the o rows are independent loads) and writes `out` / `lse`.  No second launch.
//
// Data path per warp: the 4 KiB K tile and 4 KiB V tile of a page are copied global -> shared with 16-byte cp.async
// (512 contiguous bytes per warp instruction) into a per-warp ring of kDecStages stages.  Shared layout of a tile:
// [half = dim/64][token 0..15][64 dims = 8 chunks of 16 B], chunk index XOR (token & 7) -- the 128-byte swizzle,
// conflict-free for ldmatrix.
//
// Math: the products are a [heads x 128] x [128 x 16 tokens] and a [heads x 16] x [16 x 128] contraction per page;
// at r >= 4 the plain FP32 pipes cannot keep up with HBM ("ALU budget"), so both run on the tensor
// cores with the query heads as the (zero-padded) M = 16 rows of mma.sync.m16n8k16 bf16 -> fp32:
//   S[head][token] = sum_d Q[head][d] K[token][d]     A = Q fragments (registers), B = K via ldmatrix
//   O[head][d]    += sum_t P[head][t] V[t][d]         A = P (bf16, from the S accumulators), B = V via ldmatrix.trans
// Softmax statistics (running max m in the log2 domain, sum l) are fp32.
#pragma once
#include "common.cuh"

namespace sparrow {

#ifndef SPARROW_DEC_WARPS
#define SPARROW_DEC_WARPS 8
#endif
#ifndef SPARROW_DEC_STAGES
#define SPARROW_DEC_STAGES 2
#endif
#ifndef SPARROW_DEC_MAXSEQ
#define SPARROW_DEC_MAXSEQ 8192
#endif
constexpr int kDecWarps = SPARROW_DEC_WARPS;
constexpr int kDecThreads = kDecWarps * 32;
constexpr int kDecStages = SPARROW_DEC_STAGES;                                   // per-warp ring depth
constexpr int kStageBytes = 2 * kTileBytes;                     // K tile + V tile = 8 KiB
constexpr int kDecRingBytes = kDecWarps * kDecStages * kStageBytes;   // 128 KiB (2 stages measured as fast as 3; one CTA per SM by registers)
constexpr int kMaxGroup = 8;                                    // r <= 8 (rows 0..7 of the m16 tile)
constexpr int kDecMaxSeq = SPARROW_DEC_MAXSEQ;                                // prefix table of the batch lives in shared memory
constexpr int kDecGrid = 148;                                   // persistent: one CTA per B200 SM
constexpr int kDecW = kDecGrid * kDecWarps;                     // warps that stream = ranges per round
#ifndef SPARROW_DEC_MIN_RANGE
#define SPARROW_DEC_MIN_RANGE 4
#endif
#ifndef SPARROW_DEC_R0_EIGHTHS
#define SPARROW_DEC_R0_EIGHTHS 8
#endif
constexpr int kDecMinRange = SPARROW_DEC_MIN_RANGE;             // tiles per range at least
constexpr int kDecMaxRounds = 24;                               // rounds of the factoring schedule at most

// Factoring self-scheduling of a stream of T tiles over kDecW warps.  Round k holds up to kDecW ranges of
// size[k] tiles starting at tile off[k]; every round but the last holds exactly kDecW, so range index
// i = k * kDecW + j is range j of round k.  `max_rounds` (<= kDecMaxRounds) caps the table: the last allowed
// round takes all that is left, so total <= kDecW * max_rounds whatever T is (this bounds the partial slots).
struct DecSchedule {
    int n_rounds, total;
    int off[kDecMaxRounds + 1];
    int size[kDecMaxRounds];
};
__host__ __device__ inline void decode_schedule(int T, int max_rounds, DecSchedule &s)
{
    int off = 0, k = 0, total = 0;
    while (off < T) {
        const int rem = T - off;
        int sz = k == 0 ? (int)(((int64_t)rem * SPARROW_DEC_R0_EIGHTHS / 8 + kDecW - 1) / kDecW) : (rem + 2 * kDecW - 1) / (2 * kDecW);
        if (k >= max_rounds - 1) sz = (rem + kDecW - 1) / kDecW;
        if (sz < kDecMinRange) sz = kDecMinRange;
        const int n = (int64_t)sz * kDecW <= rem ? kDecW : (rem + sz - 1) / sz;
        s.off[k] = off;
        s.size[k] = sz;
        off = n == kDecW ? off + sz * kDecW : T;
        total += n;
        ++k;
    }
    s.off[k] = T;
    s.n_rounds = k;
    s.total = total;
}
// Rounds that a stream of at most t_max tiles can need (host side: sizes the workspace and caps the kernel's table).
__host__ inline int decode_max_rounds(int64_t t_max)
{
    int rounds = 4;
    for (int64_t x = t_max / ((int64_t)kDecW * kDecMinRange); x > 0; x >>= 1) ++rounds;
    return rounds < kDecMaxRounds ? rounds : kDecMaxRounds;
}

__device__ __forceinline__ int ld_acquire(const int32_t *p)
{
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release(int32_t *p, int v)
{
    asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

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

constexpr int kMetaFirst = 1 << 8, kMetaLast = 1 << 9;

// Everything the streaming part of the decode needs (kernel arguments, passed on unchanged).
struct DecodeArgs {
    const uint16_t *q, *k_cache, *v_cache;
    const int32_t *page_table, *seq_lens, *sel_pages, *sel_count;
    int max_sel;
    float *ws_o, *ws_ml;
    int32_t *counters, *sched_ctr;
    uint16_t *out;
    float *lse;
    float scale_log2;
    int n_seq, n_q_heads, n_kv_heads, max_pages;
    int tpp_log2;                // log2 of the 16-token tiles per page (page size 16, 32, 64, 128 -> 0, 1, 2, 3)
    const int32_t *ready;        // fused step only: per-unit flag, non-zero once the unit's page list is written
};

// One warp's share of the decode: streams its ranges of the flat tile stream (s_prefix = list entries before
// sequence i, s_sched = the range table, both in shared memory) through its K/V ring at `ring`.
// kFused: the page lists are being written by the same launch (step.cuh); a look-up waits for its unit's flag.
template <bool kDense, bool kFused>
__device__ __forceinline__ void decode_warp_stream(const DecodeArgs &A, const int32_t *s_prefix, const DecSchedule &s_sched,
                                                   uint8_t *ring)
{
    const uint16_t *__restrict__ q = A.q, *__restrict__ k_cache = A.k_cache, *__restrict__ v_cache = A.v_cache;
    const int32_t *__restrict__ page_table = A.page_table, *__restrict__ seq_lens = A.seq_lens;
    const int32_t *__restrict__ sel_pages = A.sel_pages;
    float *__restrict__ ws_o = A.ws_o, *__restrict__ ws_ml = A.ws_ml;
    int32_t *__restrict__ counters = A.counters, *__restrict__ sched_ctr = A.sched_ctr;
    uint16_t *__restrict__ out = A.out;
    float *__restrict__ lse = A.lse;
    const float scale_log2 = A.scale_log2;
    const int max_sel = A.max_sel, n_seq = A.n_seq, n_q_heads = A.n_q_heads, n_kv_heads = A.n_kv_heads, max_pages = A.max_pages;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r = n_q_heads / n_kv_heads;
    constexpr uint32_t kFull = 0xffffffffu;

    const int T = s_prefix[n_seq] * n_kv_heads;                  // tiles of the whole batch
    const int NR = s_sched.total;                                // ranges of the whole batch
    const int gw = blockIdx.x * kDecWarps + warp;
    // (no CTA-wide barrier below this line: warps run independently)

    // range index -> tiles [a, b);  tile -> index of the range that holds it
    auto range_bounds = [&](int k, int &a, int &b) {
        const int rd = k / kDecW, j = k - rd * kDecW, sz = s_sched.size[rd];
        a = s_sched.off[rd] + j * sz;
        b = min(a + sz, T);
    };
    auto range_of = [&](int t) {
        int rd = 0;
        while (rd + 1 < s_sched.n_rounds && s_sched.off[rd + 1] <= t) ++rd;
        return rd * kDecW + (t - s_sched.off[rd]) / s_sched.size[rd];
    };

    // Look-up of flat tile p -> (sequence, kv-head, list position) -> logical page -> physical tile, as three stages
    // so that no stage consumes a load issued by the stage before it in the same breath: the warp never stalls on
    // the chain while its K/V ring is running.  A WINDOW is up to 32 consecutive tiles of one range, lane = tile.
    struct Lookup {
        int tile;        // stage C: physical page * Hkv + kv-head = index of the 4 KiB K (and V) tile
        int unit;        // stage A: sequence * Hkv + kv-head
        int info;        // stage A: bit 8 first tile of a segment, bit 9 last; stage B adds bits 0-4 = valid tokens
        int seq, logical, len, phys;
        int sub;         // stage A: 16-token tile inside the page (pages larger than 16 tokens)
    };
    auto stage_a = [&](Lookup &m, int p, bool on, int ra, int rb) {
        m.tile = 0; m.unit = 0; m.info = 0; m.seq = -1; m.logical = 0; m.len = 0; m.phys = 0; m.sub = 0;
        if (on) {
            int lo = 0, hi = n_seq - 1;                          // last sequence whose first tile is <= p ...
            while (lo < hi) {
                const int mid = (lo + hi + 1) >> 1;
                if (s_prefix[mid] * n_kv_heads <= p) lo = mid; else hi = mid - 1;
            }
            while (s_prefix[lo + 1] * n_kv_heads <= p) ++lo;     // ... that is not empty (empty lists share a prefix)
            const int seq = lo, base = s_prefix[seq], c = s_prefix[seq + 1] - base;
            const int rem = p - base * n_kv_heads;
            const int g = rem / c, i = rem - g * c;
            m.seq = seq;
            m.unit = seq * n_kv_heads + g;
            m.info = ((i == 0 || p == ra) ? kMetaFirst : 0) | ((i == c - 1 || p == rb - 1) ? kMetaLast : 0);
            const int pi = i >> A.tpp_log2;                      // list position of the tile's page
            m.sub = i - (pi << A.tpp_log2);
            if (kFused) {                                        // the list is written by this launch: wait for it
                while (ld_acquire(A.ready + m.unit) == 0) __nanosleep(64);
                m.logical = __ldcg(sel_pages + ((int64_t)m.unit) * max_sel + pi);
            } else {
                m.logical = kDense ? pi : __ldg(sel_pages + ((int64_t)m.unit) * max_sel + pi);
            }
            m.len = __ldg(seq_lens + seq);
        }
    };
    auto stage_b = [&](Lookup &m) {
        if (m.seq >= 0) {
            m.phys = __ldg(page_table + (int64_t)m.seq * max_pages + m.logical);
            int valid = m.len - ((m.logical << A.tpp_log2) + m.sub) * kPage;
            valid = valid < 0 ? 0 : (valid > kPage ? kPage : valid);
            m.info |= valid;
        }
    };
    auto stage_c = [&](Lookup &m) { m.tile = ((m.phys * n_kv_heads + (m.unit - m.seq * n_kv_heads)) << A.tpp_log2) + m.sub; };

    // ---- the warp's supply of ranges and windows ----
    int ra = 0, rb = 0, rp = 0;          // current range [ra, rb), next tile not yet in a window
    int rk = 0;                          // its index
    int k_next = gw;                     // lane 0: index of the range after it (round 0: the warp's own, no atomic)
    // Opens the next window: n tiles (0 = the stream is exhausted) of range index wk; runs stage A of its look-ups.
    auto open_window = [&](Lookup &m, int &n, int &wk) {
        if (rp >= rb) {                                          // the range is used up: take the prefetched index
            const int k = __shfl_sync(kFull, k_next, 0);
            if (k >= NR) { n = 0; wk = k; stage_a(m, 0, false, 0, 0); return; }
            range_bounds(k, ra, rb);
            rp = ra;
            rk = k;
            if (lane == 0) k_next = kDecW + atomicAdd(sched_ctr, 1);     // consumed one range from now
        }
        const int rem = rb - rp;
        n = rem > 32 ? (rem < 34 ? 30 : 32) : rem;               // never leaves a window of one tile behind
        wk = rk;
        stage_a(m, rp + lane, lane < n, ra, rb);
        rp += n;
    };

    const int hrow = lane >> 2, col = 2 * (lane & 3);               // this lane's query head and column pair
    uint32_t qa[8][2];                                              // Q fragments of the current unit
    auto load_q = [&](int unit) {
        const uint16_t *qrow = q + ((int64_t)unit * r + hrow) * kDim + col;
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
            qa[kk][0] = hrow < r ? __ldg(reinterpret_cast<const uint32_t *>(qrow + kk * 16)) : 0u;
            qa[kk][1] = hrow < r ? __ldg(reinterpret_cast<const uint32_t *>(qrow + kk * 16 + 8)) : 0u;
        }
    };

    Lookup cur, nxt;
    int cn, ck, nn, nk;                  // tiles and range index of the current and the next window
    int nxt_stage;                       // look-up stages of `nxt` done so far (1 = A, 2 = B, 3 = C)
    open_window(cur, cn, ck);
    int q_unit = __shfl_sync(kFull, cur.unit, 0);
    if (cn > 0) load_q(q_unit);                                     // in flight while the look-up chain completes
    if (cn > 0) { open_window(nxt, nn, nk); nxt_stage = 1; }
    else { nn = 0; nk = ck; nxt_stage = 3; }
    stage_b(cur);
    stage_c(cur);
    auto advance_nxt = [&](int target) {                            // warp-uniform
        if (nxt_stage < 2 && target >= 2) { stage_b(nxt); nxt_stage = 2; }
        if (nxt_stage < 3 && target >= 3) { stage_c(nxt); nxt_stage = 3; }
    };

    const uint32_t ring_u32 = smem_u32(ring);
    auto issue = [&](int tile, int stage) {       // copy one K tile and one V tile into a ring stage
        const uint8_t *ksrc = reinterpret_cast<const uint8_t *>(k_cache + (int64_t)tile * kTileElems);
        const uint8_t *vsrc = reinterpret_cast<const uint8_t *>(v_cache + (int64_t)tile * kTileElems);
        const uint32_t dst = ring_u32 + stage * kStageBytes;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int idx = i * 32 + lane;                          // 16-byte chunk of the tile, row-major
            const uint32_t off = tile_off(idx >> 4, idx & 15);
            cp_async16(dst + off, ksrc + idx * 16);
            cp_async16(dst + kTileBytes + off, vsrc + idx * 16);
        }
    };
    // tile at distance d >= 0 ahead of position j of the current window (-1: past the end of the warp's stream)
    auto tile_ahead = [&](int jj) {
        int t = -1;
        if (jj < cn) t = __shfl_sync(kFull, cur.tile, jj);
        else if (jj - cn < nn) {
            advance_nxt(3);
            t = __shfl_sync(kFull, nxt.tile, jj - cn);
        }
        return t;
    };

    float o[16][2];                 // O[head = lane/4][dims nt*8 + col + {0,1}]
    float m_run = -INFINITY, l_run = 0.f;

#pragma unroll
    for (int j = 0; j < kDecStages - 1; ++j) {
        const int tile = tile_ahead(j);
        if (tile >= 0) issue(tile, j);
        cp_async_commit();
    }
    const int mat = lane >> 3, rr = lane & 7;
    int stage = 0;                                                  // ring stage of the tile being consumed
#pragma unroll 1
    while (cn > 0) {
        // look-up stages B and C of the next window run a third and two thirds of the way through this one
        const int jc = cn >= 24 ? 16 : max(0, min((2 * cn) / 3, cn - 2));
        const int jb = cn >= 24 ? 8 : min(cn / 3, jc);
#pragma unroll 1
        for (int j = 0; j < cn; ++j) {
            if (j == jb) advance_nxt(2);
            if (j == jc) advance_nxt(3);
            __syncwarp();                                           // the stage consumed last is free again
            {
                const int tile = tile_ahead(j + kDecStages - 1);
                int st2 = stage + kDecStages - 1;
                st2 = st2 >= kDecStages ? st2 - kDecStages : st2;
                if (tile >= 0) issue(tile, st2);
                cp_async_commit();
            }
            const int info = __shfl_sync(kFull, cur.info, j);
            const int unit = __shfl_sync(kFull, cur.unit, j);
            if (info & kMetaFirst) {                                // warp-uniform: a new softmax state opens
#pragma unroll
                for (int nt = 0; nt < 16; ++nt) { o[nt][0] = 0.f; o[nt][1] = 0.f; }
                m_run = -INFINITY; l_run = 0.f;
                if (unit != q_unit) {
                    q_unit = unit;
                    load_q(unit);
                }
            }
            cp_async_wait<kDecStages - 1>();                         // this lane's copies of the tile have landed
            __syncwarp();                                            // ... and so have the other lanes'
            const uint32_t kb = ring_u32 + stage * kStageBytes;
            const uint32_t vb = kb + kTileBytes;
            stage = stage + 1 == kDecStages ? 0 : stage + 1;
            const int valid = info & 31;
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

            if (!(info & kMetaLast)) continue;
            // ---- the segment of `unit` inside this range is complete: write it out (a7) ----
            float l_tot = l_run;
            l_tot += __shfl_xor_sync(kFull, l_tot, 1);
            l_tot += __shfl_xor_sync(kFull, l_tot, 2);
            const int seq = unit / n_kv_heads, g = unit - seq * n_kv_heads;
            const int base = s_prefix[seq], c = s_prefix[seq + 1] - base;
            const int u0 = base * n_kv_heads + g * c;                // the unit's tiles are [u0, u0 + c) of the stream
            const int w0 = range_of(u0), w1 = range_of(u0 + c - 1);  // ranges that cover it
            constexpr float kLn2 = 0.6931471805599453f;
            if (w0 == w1) {                                          // covered by this range alone: final result
                if (hrow < r) {
                    const float inv = l_tot > 0.f ? 1.f / l_tot : 0.f;
                    uint32_t *dst = reinterpret_cast<uint32_t *>(out + ((int64_t)unit * r + hrow) * kDim + col);
#pragma unroll
                    for (int nt = 0; nt < 16; ++nt) dst[nt * 4] = pack_bf16(o[nt][0] * inv, o[nt][1] * inv);
                    if (lse && (lane & 3) == 0)
                        lse[(int64_t)unit * r + hrow] = l_tot > 0.f ? (m_run + log2f(l_tot)) * kLn2 : -INFINITY;
                }
                continue;
            }
            {
                const int64_t slot = (int64_t)unit + ck;             // unique: unit + range index increases along the stream
                if (hrow < r) {
                    float *po = ws_o + (slot * r + hrow) * kDim + col;
#pragma unroll
                    for (int nt = 0; nt < 16; ++nt) *reinterpret_cast<float2 *>(po + nt * 8) = make_float2(o[nt][0], o[nt][1]);
                    if ((lane & 3) == 0) *reinterpret_cast<float2 *>(ws_ml + (slot * r + hrow) * 2) = make_float2(m_run, l_tot);
                }
            }
            // release / acquire through ONE atomic of lane 0 (no fence per lane): the warp barrier orders the lanes'
            // partial stores before lane 0's acq_rel atomic (cumulative at gpu scope), and the warp barrier after the
            // shuffle that hands its result round orders that acquire before the other lanes' reads of the slots
            __syncwarp();
            int old = 0;
            if (lane == 0)
                asm volatile("atom.acq_rel.gpu.global.add.s32 %0, [%1], 1;" : "=r"(old) : "l"(counters + unit) : "memory");
            old = __shfl_sync(kFull, old, 0);
            __syncwarp();                                            // a shuffle is not a memory-ordering operation; the warp barrier is
            if (old != w1 - w0) continue;                            // not the last segment to arrive
            if (lane == 0) counters[unit] = 0;                       // restore the zero for the next call
            const int nseg = w1 - w0 + 1;
            const int64_t row0 = ((int64_t)unit + w0) * r;           // slot row of segment s, head h: row0 + s * r + h
            // Every dependent round trip costs 1-2 us while the K/V stream saturates HBM, so the merge is written for
            // few rounds: the (m, l) pairs of all segments and heads (lane = segment) and the o rows of the first two
            // segments (lane = 4 channels) are requested together; each further pair of segments is one more round.
            float m_star[kMaxGroup], l_star[kMaxGroup], wgt[kMaxGroup];
            float4 acc[kMaxGroup];
            const float *src = ws_o + row0 * kDim + lane * 4;
            float2 ml[kMaxGroup];
#pragma unroll
            for (int h = 0; h < kMaxGroup; ++h) {
                ml[h] = make_float2(-INFINITY, 0.f);
                if (h < r && lane < nseg) ml[h] = __ldcg(reinterpret_cast<const float2 *>(ws_ml + (row0 + (int64_t)lane * r + h) * 2));
            }
            float4 pa[kMaxGroup], pb[kMaxGroup];                     // o rows of segments i and i + 1
            auto load_pair = [&](int i) {
#pragma unroll
                for (int h = 0; h < kMaxGroup; ++h) {
                    pa[h] = make_float4(0.f, 0.f, 0.f, 0.f);
                    pb[h] = pa[h];
                    if (h < r) {
                        pa[h] = __ldcg(reinterpret_cast<const float4 *>(src + ((int64_t)i * r + h) * kDim));
                        if (i + 1 < nseg) pb[h] = __ldcg(reinterpret_cast<const float4 *>(src + ((int64_t)(i + 1) * r + h) * kDim));
                    }
                }
            };
            load_pair(0);
#pragma unroll
            for (int h = 0; h < kMaxGroup; ++h) {
                m_star[h] = ml[h].y > 0.f ? ml[h].x : -INFINITY;
                acc[h] = make_float4(0.f, 0.f, 0.f, 0.f);
            }
            for (int s0 = 32; s0 < nseg; s0 += 32) {                 // more than 32 segments (long dense units only)
                const int s = s0 + lane;
#pragma unroll
                for (int h = 0; h < kMaxGroup; ++h) {
                    if (h < r && s < nseg) {
                        const float2 t = __ldcg(reinterpret_cast<const float2 *>(ws_ml + (row0 + (int64_t)s * r + h) * 2));
                        if (t.y > 0.f) m_star[h] = fmaxf(m_star[h], t.x);
                    }
                }
            }
#pragma unroll
            for (int h = 0; h < kMaxGroup; ++h) {
#pragma unroll
                for (int of = 16; of > 0; of >>= 1) m_star[h] = fmaxf(m_star[h], __shfl_xor_sync(kFull, m_star[h], of));
                wgt[h] = ml[h].y > 0.f ? fast_exp2(ml[h].x - m_star[h]) : 0.f;      // empty partial: weight 0, never NaN
                l_star[h] = ml[h].y * wgt[h];
            }
            for (int s0 = 0; s0 < nseg; s0 += 32) {
                if (s0 > 0) {
                    const int s = s0 + lane;
#pragma unroll
                    for (int h = 0; h < kMaxGroup; ++h) {
                        wgt[h] = 0.f;
                        if (h < r && s < nseg) {
                            const float2 t = __ldcg(reinterpret_cast<const float2 *>(ws_ml + (row0 + (int64_t)s * r + h) * 2));
                            if (t.y > 0.f) {
                                wgt[h] = fast_exp2(t.x - m_star[h]);
                                l_star[h] = fmaf(t.y, wgt[h], l_star[h]);
                            }
                        }
                    }
                }
                const int cnt = min(32, nseg - s0);
                for (int i = 0; i < cnt; i += 2) {
                    if (s0 + i > 0) load_pair(s0 + i);
#pragma unroll
                    for (int h = 0; h < kMaxGroup; ++h) {
                        if (h < r) {
                            const float wa = __shfl_sync(kFull, wgt[h], i);
                            const float wb = __shfl_sync(kFull, wgt[h], (i + 1) & 31);
                            if (wa > 0.f) {
                                acc[h].x = fmaf(pa[h].x, wa, acc[h].x); acc[h].y = fmaf(pa[h].y, wa, acc[h].y);
                                acc[h].z = fmaf(pa[h].z, wa, acc[h].z); acc[h].w = fmaf(pa[h].w, wa, acc[h].w);
                            }
                            if (i + 1 < cnt && wb > 0.f) {
                                acc[h].x = fmaf(pb[h].x, wb, acc[h].x); acc[h].y = fmaf(pb[h].y, wb, acc[h].y);
                                acc[h].z = fmaf(pb[h].z, wb, acc[h].z); acc[h].w = fmaf(pb[h].w, wb, acc[h].w);
                            }
                        }
                    }
                }
            }
#pragma unroll
            for (int h = 0; h < kMaxGroup; ++h) {
                if (h < r) {
                    float ls = l_star[h];
#pragma unroll
                    for (int of = 16; of > 0; of >>= 1) ls += __shfl_xor_sync(kFull, ls, of);
                    const float inv = ls > 0.f ? 1.f / ls : 0.f;
                    uint2 pk;
                    pk.x = pack_bf16(acc[h].x * inv, acc[h].y * inv);
                    pk.y = pack_bf16(acc[h].z * inv, acc[h].w * inv);
                    *reinterpret_cast<uint2 *>(out + ((int64_t)unit * r + h) * kDim + lane * 4) = pk;
                    if (lse && lane == 0)
                        lse[(int64_t)unit * r + h] = ls > 0.f ? (m_star[h] + log2f(ls)) * kLn2 : -INFINITY;
                }
            }
        }
        // ---- window turn ----
        advance_nxt(3);
        cur = nxt; cn = nn; ck = nk;
        if (cn > 0) { open_window(nxt, nn, nk); nxt_stage = 1; }
        else { nn = 0; nxt_stage = 3; }
    }
    cp_async_wait<0>();
}

template <bool kDense>
__global__ void __launch_bounds__(kDecThreads, 1)
decode_kernel(const DecodeArgs A, int max_rounds)
{
    chain_entry();
    extern __shared__ __align__(1024) uint8_t smem[];
    int32_t *s_prefix = reinterpret_cast<int32_t *>(smem + kDecRingBytes);     // [n_seq + 1] tiles per kv-head before sequence i
    __shared__ int s_scan[kDecWarps];
    __shared__ DecSchedule s_sched;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n_seq = A.n_seq, n_kv_heads = A.n_kv_heads, max_sel = A.max_sel;
    const int32_t *__restrict__ seq_lens = A.seq_lens;
    constexpr uint32_t kFull = 0xffffffffu;



    // ---- prologue: list length of every sequence -> exclusive prefix in shared memory; the range table ----
    {
        const int per = (n_seq + kDecThreads - 1) / kDecThreads;
        const int s0 = min(tid * per, n_seq), s1 = min(s0 + per, n_seq);
        auto count_of = [&](int s) {
            int c;
            const int page_tokens = kPage << A.tpp_log2;
            if (kDense) c = (__ldg(seq_lens + s) + page_tokens - 1) / page_tokens;
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
        if (tid == kDecThreads - 1) {
            s_prefix[n_seq] = run;
            decode_schedule(run * n_kv_heads, max_rounds, s_sched);
        }
        __syncthreads();
    }
    decode_warp_stream<kDense, false>(A, s_prefix, s_sched, smem + warp * (kDecStages * kStageBytes));
    // ---- the last warp out restores the scheduler's zeros for the next call ----
    if (lane == 0) {
        const int done = atomicAdd(A.sched_ctr + 1, 1);
        if (done == kDecW - 1) {
            A.sched_ctr[0] = 0;
            A.sched_ctr[1] = 0;
        }
    }
}

}  // namespace sparrow
