// decode.cuh -- kernel (c): split-K flash-decode over a page list with the log-sum-exp merge fused in.
// SURVEY.md 8(a) a6-a8; PAPER.md:140 (attention over the KV budget B), :131-135 (dense), north_star (c).
//
// Work decomposition ("stream-K" over pages): the (page, kv-head) tiles of the whole batch form ONE flat stream,
// ordered (sequence, kv-head, list position); its length T = Hkv * sum_i cnt_i is known from sel_count (or from
// seq_lens for the dense entry).  A persistent grid of one CTA per SM cuts it into equal contiguous PIECES, whatever
// the mix of lengths and budgets (optionally followed by a self-scheduled tail of small pieces: SPARROW_DEC_STATIC_*,
// off by default).  Inside a CTA the work is warp-specialised:
//
//   * ONE LOOK-UP WARP walks the CTA's stream.  It resolves flat tile -> (sequence, kv-head, list position) -> logical
//     page -> physical tile in windows of 32 tiles (lane = tile; three look-up stages, three windows in flight, so that
//     no stage consumes a load issued by the stage before it in the same breath) and publishes one 16-byte descriptor
//     per tile in a shared-memory ring, far ahead of the consumers.
//   * EIGHT CONSUMER WARPS share a CTA-wide ring of kDecStages = 16 stages of 8 KiB (the K tile and the V tile of a
//     page).  A tile is fetched by TMA: two cp.async.bulk.tensor.2d boxes of 32 rows x 128 B (SWIZZLE_128B, mbarrier
//     complete_tx), issued by one lane of the consumer that has just freed the stage (tile i + 16 follows tile i), so the
//     copy issue is spread over the eight warps.  The consumers take the stream two tiles at a time from a counter in
//     shared memory -- whoever is free takes the next chunk -- each with its own online-softmax state for the unit
//     (sequence, kv-head) it is in.  When a consumer is handed a tile of another unit it parks its state in shared
//     memory; the consumer whose tiles complete the CTA's PART of the unit merges the parked states and writes the
//     result: final (straight to `out`) when the unit lies inside the piece, otherwise the piece's partial, in slot
//     unit + piece id of a small fp32 workspace -- the warp that completes the unit's tile count merges the pieces'
//     partials in stream order (a7; no second launch).
//
// Why this shape (round 2): with one private stream per warp (round 1) a warp's progress is a sum of
// ~50 saturated-HBM latencies; the per-warp finish times spread with sigma ~7 us on a 90 us launch and the kernel
// ends with the slowest of 1184 warps.  Handing the tiles out inside the CTA brings the warps of a CTA to within 2 us
// of one another (traced).  What remains is the spread BETWEEN SMs (equal pieces end +-15 % apart), see DESIGN.md.
// The price of run-time hand-out: which tiles a consumer sums is timing-dependent, so the running maximum under which a
// probability is rounded to bf16 (2^-9 relative per term) and the fp32 summation order differ from call to call: two
// calls agree to the arithmetic's own error (~1e-3 absolute on these inputs, the size of either call's distance from the
// fp64 oracle), not bit for bit.  The page lists, counts, lse to fp32 rounding, and everything integer are reproducible.
// The whole GQA group (r <= 8 query heads) is processed together, so each K/V byte is read from HBM once.
//
// Shared layout of a tile: 32 rows of 128 B, row = (token, half of the head dim), 16-byte chunk index XOR (row & 7) --
// what a 32 x 64 box of the pool's [128-byte rows] view lands as under SWIZZLE_128B: ONE copy per 4 KiB tile (two
// 16 x 64 boxes per tile made the copy issue the limit).  ldmatrix reads it with 2-way bank conflicts (tokens t and
// t + 4 of a half share a bank group); the shared-memory pipe is a third busy at full HBM rate, so they are not the limit.
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

constexpr int kDecConsumers = 8;                                // consumer warps
constexpr int kDecThreads = (kDecConsumers + 1) * 32;           // + the look-up warp
#ifndef SPARROW_DEC_STAGES
#define SPARROW_DEC_STAGES 16
#endif
constexpr int kDecStages = SPARROW_DEC_STAGES;                  // CTA-wide ring depth (tiles in flight per SM)
constexpr int kStageBytes = 2 * kTileBytes;                     // K tile + V tile = 8 KiB
constexpr int kDecRingBytes = kDecStages * kStageBytes;         // 128 KiB
constexpr int kDecChunk = 2;                                    // tiles per claim (kDecConsumers x kDecChunk = the ring: every consumer's tiles are in flight)
static_assert(kDecConsumers * kDecChunk <= kDecStages, "the tiles of every consumer's claim are in the ring together");
constexpr int kMaxGroup = 8;                                    // r <= 8 (rows 0..7 of the m16 tile)
#ifndef SPARROW_DEC_MAXSEQ
#define SPARROW_DEC_MAXSEQ 4096
#endif
constexpr int kDecMaxSeq = SPARROW_DEC_MAXSEQ;                  // prefix table of the batch lives in shared memory
constexpr int kDecGrid = 148;                                   // persistent: one CTA per B200 SM (fewer SMs: fewer CTAs)
constexpr int kAccRow = kDim + 4;                               // one parked head: o[128] | m | l | pad
constexpr int kAccSlots = 2;                                    // parts (the CTA's share of a unit) being parked at once
#ifndef SPARROW_DEC_ACC_GROUP
#define SPARROW_DEC_ACC_GROUP kMaxGroup
#endif
constexpr int kAccGroup = SPARROW_DEC_ACC_GROUP;                   // heads a parking area has room for
constexpr int kDecAccBytes = kAccSlots * kDecConsumers * kAccGroup * kAccRow * 4;   // [slot][consumer][head][kAccRow]
constexpr int kDescRing = 256;                                  // per-tile descriptors the look-up warp runs ahead by
constexpr int kPartRing = 512;                                  // per-part records (piece id, piece bounds) kept beside them
constexpr int kDecDescBytes = kDescRing * 16 + kPartRing * 16;
constexpr int kTailChunk = 32;                                  // tiles of a self-scheduled piece of the stream's tail (= one look-up window)
// share of the stream that is split evenly over the CTAs; the rest is self-scheduled in pieces of kTailChunk tiles.
// Default 1 / 1 = no tail: measured, the tail's extra partials and merges cost more than the balance buys.
#ifndef SPARROW_DEC_STATIC_NUM
#define SPARROW_DEC_STATIC_NUM 1
#endif
#ifndef SPARROW_DEC_STATIC_DEN
#define SPARROW_DEC_STATIC_DEN 1
#endif
// deterministic mode (SPARROW_FLAG_DETERMINISTIC): rounds a consumer may run ahead of the slowest one (0 = no limit)
#ifndef SPARROW_DEC_DET_WINDOW
#define SPARROW_DEC_DET_WINDOW 1
#endif
constexpr int kDetWindow = SPARROW_DEC_DET_WINDOW;
constexpr int kDecMetaBytes = kDecStages * 8 + kDecStages * 4 + 3 * kAccSlots * 4 + kDecConsumers * 4 + 64;   // (+ claim, ready, total)   // full barriers | issued tile per stage | area generation, tile count, consumer mask | consumer positions | claim, ready

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
    const int rho = 2 * t + (c >> 3);                    // 128-byte row of the tile: (token, half)
    return (uint32_t)(rho * 128 + (((c & 7) ^ (rho & 7)) << 4));
}

// One TMA box = one 4 KiB tile: 32 rows x 64 bf16 columns of the [128-byte rows][64] view of a K or V pool (row = (token,
// half of the head dim)), starting at (col, row), into shared memory (SWIZZLE_128B), completing 4096 bytes on `bar`.
__device__ __forceinline__ void tma_box(uint32_t dst, const CUtensorMap *tm, int col, int row, uint32_t bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tm)), "r"(col), "r"(row), "r"(bar) : "memory");
}
// The same tile out of a strided pool: box (64 columns, 2 halves, 16 tokens) at (0, 0, first token, kv-head, page) of the 5-D view.
__device__ __forceinline__ void tma_box5(uint32_t dst, const CUtensorMap *tm, int tok, int head, int page, uint32_t bar)
{
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %2, %3, %4, %5}], [%6];"
                 ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tm)), "r"(0), "r"(tok), "r"(head), "r"(page), "r"(bar) : "memory");
}
__device__ __forceinline__ int lds_volatile(const int32_t *p)
{
    int v;
    asm volatile("ld.volatile.shared.s32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
    return v;
}
// A wait on a shared-memory word that another warp of the CTA will write.  Bounded: a protocol bug becomes a trap (a launch
// failure the caller sees) instead of a hung device.
__device__ __forceinline__ void spin_until(const int32_t *p, int want_ge)
{
    for (uint32_t n = 0; lds_volatile(p) < want_ge; ++n)
        if (n > (1u << 27)) __trap();
}
__device__ __forceinline__ void sts_volatile(int32_t *p, int v)
{
    asm volatile("st.volatile.shared.s32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}

// Everything the decode needs (kernel arguments, passed on unchanged).
struct DecodeArgs {
    const uint16_t *q;
    const int32_t *page_table, *seq_lens, *sel_pages, *sel_count;
    int max_sel;
    float *ws_o, *ws_ml;         // partials of the pieces: [units + pieces][r][128] and [..][r][2] (m, l)
    int32_t *counters;           // [units] tiles of the unit merged so far | tail-piece counter | CTAs done   (all zero between calls)
    uint16_t *out;
    float *lse;
    float scale_log2;
    int n_seq, n_q_heads, n_kv_heads, max_pages;
    int tpp_log2;                // log2 of the 16-token tiles per page (page size 16, 32, 64, 128 -> 0, 1, 2, 3)
    int strided;                 // the pools are not the packed HND layout: tiles are fetched with 5-D boxes (sparrow_shape_t kv_stride_*)
    int deterministic;           // SPARROW_FLAG_DETERMINISTIC: fixed tile hand-out and merge order -- out / lse are bit-reproducible
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
    // the tensor maps are kernel parameters, not data of the kernel before this one: fetch them into the descriptor cache now,
    // so that the first TMA copy (on the launch's critical path: DESIGN.md 6.3, "ramp") does not start with that miss
    if (threadIdx.x == 0) {
        asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&tm_k)) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(reinterpret_cast<uint64_t>(&tm_v)) : "memory");
    }
    if (threadIdx.x == 0) SPARROW_TR(kTraceDecodeCta + blockIdx.x, 0);
    if ((threadIdx.x & 31) == 0) SPARROW_TR(kTraceDecodeWarp + blockIdx.x * (kDecThreads / 32) + (threadIdx.x >> 5), 0);
    chain_wait();
    if (threadIdx.x == 0) SPARROW_TR(kTraceDecodeCta + blockIdx.x, 1);
    extern __shared__ __align__(1024) uint8_t smem[];
    float *s_acc = reinterpret_cast<float *>(smem + kDecRingBytes);                           // [slot][consumer][head][kAccRow]
    int4 *s_desc = reinterpret_cast<int4 *>(smem + kDecRingBytes + kDecAccBytes);             // [kDescRing] per-tile descriptors
    uint64_t *s_full = reinterpret_cast<uint64_t *>(smem + kDecRingBytes + kDecAccBytes + kDecDescBytes);   // [stage] tile has landed
    int32_t *s_issued = reinterpret_cast<int32_t *>(s_full + kDecStages);                     // [stage] latest tile requested into the stage
    int32_t *s_gen = s_issued + kDecStages;                                                   // [slot] parts finished on this parking area
    int32_t *s_count = s_gen + kAccSlots;                                                     // [slot] tiles of the current part parked so far
    int32_t *s_mask = s_count + kAccSlots;                                                    // [slot] consumers that have parked a state
    int32_t *s_pos = s_mask + kAccSlots;                                                      // [consumer] first tile of the claim it is working on
    int32_t *s_claim = s_pos + kDecConsumers;                                                 // chunks claimed by the consumers
    int32_t *s_ready = s_claim + 1;                                                           // descriptors written by the look-up warp
    int32_t *s_prefix = reinterpret_cast<int32_t *>(smem + kDecRingBytes + kDecAccBytes + kDecDescBytes + kDecMetaBytes);   // [n_seq + 1]
    __shared__ int s_scan[kDecThreads / 32];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n_seq = A.n_seq, n_kv_heads = A.n_kv_heads, max_sel = A.max_sel, max_pages = A.max_pages;
    const int r = A.n_q_heads / n_kv_heads;
    constexpr uint32_t kFull = 0xffffffffu;
    const uint32_t ring_u32 = smem_u32(smem);
    const uint32_t full_u32 = smem_u32(s_full);

    // ---- prologue: barriers and flags; list length of every sequence -> exclusive prefix in shared memory ----
    if (tid == 0) {
        for (int s = 0; s < kDecStages; ++s) mbar_init(full_u32 + 8 * s, 1);    // the issuing lane's arrive.expect_tx; the copies complete the bytes
        fence_mbar_init();
        *s_claim = 0;
        *s_ready = 0;
    }
    if (tid < kAccSlots) { s_gen[tid] = 0; s_count[tid] = 0; s_mask[tid] = 0; }
    if (tid < kDecStages) s_issued[tid] = -1;
    if (tid < kDecConsumers) s_pos[tid] = 0;
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
    if (threadIdx.x == 0) SPARROW_TR(kTraceDecodeCta + blockIdx.x, 2);
    if (T == 0) return;
    // The stream is cut into PIECES.  Its first kStatic part is split evenly: CTA b owns piece b, a contiguous range.  The
    // rest, the tail, is cut into pieces of kTailChunk tiles that the CTAs take from one global counter as they run out of
    // work: SMs are not served equally by the memory system (equal ranges end +-15 % apart, traced), and the tail evens
    // them out to within a piece.  Piece ids increase along the stream: b for the static pieces, G + j for tail piece j.
    const int G = (int)gridDim.x;
    const int T0 = (int)((int64_t)T * SPARROW_DEC_STATIC_NUM / SPARROW_DEC_STATIC_DEN);
    CtaRanges cr;
    cr.per = T0 / G;
    cr.extra = T0 - cr.per * G;
    const int ra = cr.begin(blockIdx.x), rb = cr.begin(blockIdx.x + 1);         // this CTA's static piece [ra, rb)
    int32_t *tail_ctr = A.counters + n_seq * n_kv_heads, *done_ctr = tail_ctr + 1;
    int4 *s_part = s_desc + kDescRing;                           // [kPartRing] x = piece id, y = piece begin, z = piece end (stream tiles)
    int32_t *s_total = s_ready + 1;                              // tiles of this CTA's stream, once known (INT_MAX before)
    if (tid == 0) sts_volatile(s_total, 0x7fffffff);
    __syncthreads();
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
        // =========================================================== LOOK-UP WARP ===========================================
        // It lines up the CTA's stream: its static piece, then tail pieces as it gets them.  flat tile p -> (sequence,
        // kv-head, list position) -> logical page -> physical tile, as three stages so that no stage consumes a load
        // issued by the stage before it in the same breath; a WINDOW is up to 32 consecutive tiles of one piece, lane =
        // tile.  The result is one 16-byte descriptor per tile in a ring the consumers read:
        //   x = index of the 4 KiB K (and V) tile in the pools          y = unit (sequence * Hkv + kv-head)
        //   z = valid tokens (bits 0-4) | part number (bits 8..)        w = tiles of the part
        // A PART is a run of the CTA's stream inside one unit and one piece: the granule the consumers reduce together.
        struct Lookup {
            int tile, unit, meta, len_part;
            int seq, logical, len, phys, sub;
        };
        int part_base = 0;                                       // parts started before the window being looked up
        auto stage_a = [&](Lookup &m, int p, bool on, int id, int cb, int ce) {
            bool starts = false;                                 // this tile is the first of a part
            m.tile = 0; m.unit = 0; m.meta = 0; m.len_part = 0; m.seq = -1; m.logical = 0; m.len = 0; m.phys = 0; m.sub = 0;
            if (on) {
                const int seq = seq_of(p), base = s_prefix[seq], c = s_prefix[seq + 1] - base;
                const int rem = p - base * n_kv_heads;
                const int g = rem / c, i = rem - g * c;
                const int u0 = base * n_kv_heads + g * c;        // the unit is tiles [u0, u0 + c) of the stream
                m.seq = seq;
                m.unit = seq * n_kv_heads + g;
                m.len_part = min(u0 + c, ce) - max(u0, cb);
                starts = i == 0 || p == cb;
                const int pi = i >> A.tpp_log2;                  // list position of the tile's page
                m.sub = i - (pi << A.tpp_log2);
                m.logical = kDense ? pi : __ldg(A.sel_pages + ((int64_t)m.unit) * max_sel + pi);
                m.len = __ldg(A.seq_lens + seq);
            }
            // parts are numbered densely along the CTA's stream (the parking areas are handed out in that order)
            const uint32_t sm = __ballot_sync(kFull, starts);
            const int part = part_base + __popc(sm & (0xffffffffu >> (31 - lane))) - 1;
            m.meta = part << 8;
            if (starts) s_part[part & (kPartRing - 1)] = make_int4(id, cb, ce, 0);
            part_base += __popc(sm);
        };
        auto stage_b = [&](Lookup &m) {
            if (m.seq >= 0) {
                m.phys = __ldg(A.page_table + (int64_t)m.seq * max_pages + m.logical);
                int valid = m.len - ((m.logical << A.tpp_log2) + m.sub) * kPage;
                m.meta |= valid < 0 ? 0 : (valid > kPage ? kPage : valid);
            }
        };
        auto stage_c = [&](Lookup &m) { m.tile = ((m.phys * n_kv_heads + (m.unit - m.seq * n_kv_heads)) << A.tpp_log2) + m.sub; };

        // The windows of the CTA's stream, in order: those of the static piece, then one per tail piece taken.  The claim of
        // a tail piece is requested one window before it is needed (its round trip to the L2 is never waited for).
        // The static piece is walked LAST PART FIRST when its last unit runs on into the next CTA's piece: [p_tail, rb), then
        // [ra, p_tail).  The neighbour starts with the other half of that unit, so both halves -- and the cross-piece merge
        // (a7), several dependent round trips -- are done early in the launch instead of forming every CTA's tail; what a
        // CTA ends with is a unit that lies inside its piece and is written straight to `out`.
        int p_tail = ra;
        if (rb > ra) {
            const int seq = seq_of(rb - 1), base = s_prefix[seq], c = s_prefix[seq + 1] - base;
            const int g = (rb - 1 - base * n_kv_heads) / c;
            const int u0 = base * n_kv_heads + g * c;            // the unit that holds the piece's last tile is tiles [u0, u0 + c)
            if (u0 > ra && u0 + c > rb) p_tail = u0;
        }
        int sp = p_tail, seg_end = rb;                           // next tile of the static piece not yet in a window; end of the segment being walked
        bool wrapped = p_tail == ra;                             // the second segment [ra, p_tail) has been entered (or does not exist)
        int j_next = -1;                                         // lane 0: tail piece claimed ahead (-1: none requested yet)
        auto prefetch_claim = [&]() {
            if (sp >= seg_end && wrapped && lane == 0 && j_next < 0) j_next = atomicAdd(tail_ctr, 1);
        };
        auto next_window = [&](Lookup &m) -> int {               // opens the next window (look-up stage A); returns its tiles, 0 = none
            int p0, n, id, cb, ce;
            if (sp < seg_end) {
                p0 = sp; n = min(32, seg_end - sp); id = (int)blockIdx.x; cb = ra; ce = rb;
                sp += n;
                if (sp == seg_end && !wrapped) { wrapped = true; sp = ra; seg_end = p_tail; }
            } else {
                prefetch_claim();
                const int j = __shfl_sync(kFull, j_next, 0);
                j_next = -1;
                if ((int64_t)T0 + (int64_t)j * kTailChunk >= T) return 0;
                p0 = T0 + j * kTailChunk; n = min(kTailChunk, T - p0); id = G + j; cb = p0; ce = p0 + n;
            }
            stage_a(m, p0 + lane, lane < n, id, cb, ce);
            return n;
        };
        // three windows in flight: `cur` (stages A, B done; C when it is published), `nxt` (A, B), `nn2` (A)
        Lookup cur, nxt, nx2;
        int w0 = 0;                                              // first tile (CTA-relative) of window `cur`
        int cn = next_window(cur);
        int nn = cn > 0 ? next_window(nxt) : 0;
        int n2 = nn > 0 ? next_window(nx2) : 0;
        if (n2 > 0) prefetch_claim();
        if (cn > 0) stage_b(cur);
        if (nn > 0) stage_b(nxt);
#pragma unroll 1
        while (cn > 0) {
            stage_c(cur);
            // room in the ring: the entries this window overwrites must be older than every consumer's current claim (a
            // consumer reads the descriptors of its claim's tiles, and of the tiles one ring further on when it refills
            // their stages).  The consumers are NOT within a fixed distance of one another: a consumer held up on tile j
            // blocks only the chain of its own stage (j, j + 16, ...), the others run on until each has picked a chunk on
            // that stage pair -- up to 7 x 8 claims ahead -- so every consumer publishes where it is.
            for (uint32_t n = 0;; ++n) {
                int lo = lane < kDecConsumers ? lds_volatile(s_pos + lane) : 0x7fffffff;
#pragma unroll
                for (int of = 4; of > 0; of >>= 1) lo = min(lo, __shfl_xor_sync(kFull, lo, of));
                lo = __shfl_sync(kFull, lo, 0);
                if (w0 + 32 - kDescRing <= lo) break;
                __nanosleep(100);
                if (n > (1u << 24)) __trap();
            }
            if (lane < cn) s_desc[(w0 + lane) & (kDescRing - 1)] = make_int4(cur.tile, cur.unit, cur.meta, cur.len_part);
            __threadfence_block();
            __syncwarp();
            if (lane == 0) sts_volatile(s_ready, w0 + cn);
            // shift the pipeline: stage B of the window after next, stage A of a new one, the claim of the one after that
            w0 += cn;
            cur = nxt; cn = nn;
            nxt = nx2; nn = n2;
            if (nn > 0) {
                stage_b(nxt);
                n2 = next_window(nx2);
                if (n2 > 0) prefetch_claim();
            } else {
                n2 = 0;
            }
        }
        if (lane == 0) sts_volatile(s_total, w0);                // the CTA's stream ends here
        if (lane == 0) { SPARROW_TR(kTraceDecodeCta + blockIdx.x, 3); SPARROW_TR(kTraceDecodeWarp + blockIdx.x * (kDecThreads / 32) + warp, 1); }
        return;
    }

    // =============================================================== CONSUMERS ===========================================
    const int hrow = lane >> 2, col = 2 * (lane & 3);               // this lane's query head and column pair
    const int mat = lane >> 3, rr = lane & 7;
    const float scale_log2 = A.scale_log2;
    constexpr float kLn2 = 0.6931471805599453f;

    // Does tile `it` of the CTA's stream exist?  Warp-uniform (every lane calls it and keeps the same cached bounds): the
    // look-up warp runs hundreds of tiles ahead, so the shared-memory words it publishes are re-read only when the cached
    // bound is reached -- and the fence that makes the descriptors behind a new bound visible is paid there, not per tile.
    int ready_seen = 0;                                             // descriptors [0, ready_seen) are published and visible to this warp
    int total_seen = 0x7fffffff;                                    // the length of the CTA's stream, once this warp has seen it
    auto exists = [&](int it) -> bool {
        if (it < ready_seen) return true;
        if (it >= total_seen) return false;
        for (uint32_t n = 0;; ++n) {
            const int rd = lds_volatile(s_ready);
            if (rd > it) { __threadfence_block(); ready_seen = rd; return true; }
            const int tt = lds_volatile(s_total);
            if (tt <= it) { total_seen = tt; return false; }
            if (n > (1u << 27)) __trap();
        }
    };
    // the tile `it` of the stream goes to stage it % kDecStages; issued by ONE lane (after exists(it) returned true)
    auto issue = [&](int it) {
        const int tile = s_desc[it & (kDescRing - 1)].x;
        const int stage = it % kDecStages;
        const uint32_t bar = full_u32 + 8 * stage, dst = ring_u32 + stage * kStageBytes;
        sts_volatile(s_issued + stage, it);
        mbar_arrive_expect_tx(bar, kStageBytes);
        if (!A.strided) {
            const int row = tile * 2 * kPage;
            tma_box(dst, &tm_k, 0, row, bar);
            tma_box(dst + kTileBytes, &tm_v, 0, row, bar);
        } else {                                                    // tile = ((page * Hkv + head) << tpp_log2) + sub
            const int sub = tile & ((1 << A.tpp_log2) - 1), ph = tile >> A.tpp_log2;
            const int page = ph / n_kv_heads, head = ph - page * n_kv_heads;
            tma_box5(dst, &tm_k, sub * kPage, head, page, bar);
            tma_box5(dst + kTileBytes, &tm_v, sub * kPage, head, page, bar);
        }
    };
    for (int it = warp; it < kDecStages; it += kDecConsumers) {     // first fill of the ring: consumer w issues tiles w, w + 8, ...
        const bool ex = exists(it);
        if (ex && lane == 0) issue(it);
    }

    uint32_t qa[8][2];                                              // Q fragments of the unit this consumer is in
    int q_unit = -1;
    float o[16][2];                 // O[head = lane/4][dims nt*8 + col + {0,1}] of the part being accumulated
    float m_run = -INFINITY, l_run = 0.f;

    // PARK: this consumer is done with a part (it has been handed a tile of another one, or the stream is exhausted).
    // Its state goes to the part's parking area; the consumer whose tiles complete the part merges the parked states
    // in consumer order and writes the result.  WHICH tiles a consumer took is decided at run time (whoever is free
    // takes the next chunk), so the result can differ from run to run within the arithmetic's error (see the file header).
    auto park = [&](int part, int unit, int n_mine, int part_len, int4 piece) {
        const int slot = part & (kAccSlots - 1);
        // The parking areas are handed out strictly in part order (part P gets area P mod 2 once part P - 2 is finished):
        // a later part can then never hold an area an earlier part is waiting for, and the earliest unfinished part --
        // whose tiles have all been consumed -- can always complete.
        if (lane == 0) {
            spin_until(s_gen + slot, part / kAccSlots);
            __threadfence_block();
        }
        __syncwarp();
        float l_tot = l_run;
        l_tot += __shfl_xor_sync(kFull, l_tot, 1);
        l_tot += __shfl_xor_sync(kFull, l_tot, 2);
        float *area = s_acc + slot * (kDecConsumers * kAccGroup * kAccRow);
        float m_new = m_run, l_new = l_tot;
        if (n_mine < part_len) {                                    // (a consumer that took the whole part keeps it in registers)
            if (hrow < r) {
                float *row = area + (warp * kAccGroup + hrow) * kAccRow;
#pragma unroll
                for (int nt = 0; nt < 16; ++nt) *reinterpret_cast<float2 *>(row + nt * 8 + col) = make_float2(o[nt][0], o[nt][1]);
                if ((lane & 3) == 0) *reinterpret_cast<float2 *>(row + kDim) = make_float2(m_run, l_tot);
            }
            __threadfence_block();
            __syncwarp();
            int last = 0, mask = 0;
            if (lane == 0) {
                atomicOr(s_mask + slot, 1 << warp);
                __threadfence_block();
                last = atomicAdd(s_count + slot, n_mine) + n_mine == part_len;
                if (last) { __threadfence_block(); mask = lds_volatile(s_mask + slot); }
            }
            last = __shfl_sync(kFull, last, 0);
            if (!last) return;
            mask = __shfl_sync(kFull, mask, 0);
            // ---- merge the parked states (consumer order) ----
            m_new = -INFINITY; l_new = 0.f;
#pragma unroll
            for (int nt = 0; nt < 16; ++nt) { o[nt][0] = 0.f; o[nt][1] = 0.f; }
            if (hrow < r) {
                for (int w2 = 0; w2 < kDecConsumers; ++w2) {
                    if (!((mask >> w2) & 1)) continue;
                    const float2 ml = *reinterpret_cast<const float2 *>(area + (w2 * kAccGroup + hrow) * kAccRow + kDim);
                    if (ml.y > 0.f) m_new = fmaxf(m_new, ml.x);
                }
                for (int w2 = 0; w2 < kDecConsumers; ++w2) {
                    if (!((mask >> w2) & 1)) continue;
                    const float *row = area + (w2 * kAccGroup + hrow) * kAccRow;
                    const float2 ml = *reinterpret_cast<const float2 *>(row + kDim);
                    const float wgt = ml.y > 0.f ? fast_exp2(ml.x - m_new) : 0.f;       // empty state: weight 0, never NaN
                    l_new = fmaf(ml.y, wgt, l_new);
#pragma unroll
                    for (int nt = 0; nt < 16; ++nt) {
                        const float2 a = *reinterpret_cast<const float2 *>(row + nt * 8 + col);
                        o[nt][0] = fmaf(a.x, wgt, o[nt][0]);
                        o[nt][1] = fmaf(a.y, wgt, o[nt][1]);
                    }
                }
            }
            __syncwarp();
        }
        if (lane == 0) {                                            // the parking area goes to the part after next
            sts_volatile(s_count + slot, 0);
            sts_volatile(s_mask + slot, 0);
            __threadfence_block();
            sts_volatile(s_gen + slot, part / kAccSlots + 1);
        }
        // ---- o / (m_new, l_new) in registers are the part's result: the piece's share of the unit ----
        const int seq = unit / n_kv_heads, g = unit - seq * n_kv_heads;
        const int c = s_prefix[seq + 1] - s_prefix[seq];
        const int u0 = s_prefix[seq] * n_kv_heads + g * c, u1 = u0 + c;
        if (u0 >= piece.y && u1 <= piece.z) {                       // the unit lies inside this piece: final result
            if (hrow < r) {
                const float inv = l_new > 0.f ? 1.f / l_new : 0.f;
                uint32_t *dst = reinterpret_cast<uint32_t *>(A.out + ((int64_t)unit * r + hrow) * kDim + col);
#pragma unroll
                for (int nt = 0; nt < 16; ++nt) dst[nt * 4] = pack_bf16(o[nt][0] * inv, o[nt][1] * inv);
                if (A.lse && (lane & 3) == 0)
                    A.lse[(int64_t)unit * r + hrow] = l_new > 0.f ? (m_new + log2f(l_new)) * kLn2 : -INFINITY;
            }
            return;
        }
        // ---- the unit spans pieces (a7).  The pieces that hold tiles of the unit, in stream order: static pieces id_a..id_b,
        // then tail pieces id_c..id_d; piece p's partial lives in slot unit + p of the workspace.
        int id_a = 0, id_b = -1, id_c = 0, id_d = -1;
        if (u0 < T0) { id_a = cr.owner(u0); id_b = cr.owner(min(u1, T0) - 1); }
        if (u1 > T0) { id_c = G + (max(u0, T0) - T0) / kTailChunk; id_d = G + (u1 - 1 - T0) / kTailChunk; }
        const int n_a = id_b - id_a + 1, nseg = n_a + (id_d - id_c + 1);
        auto piece_of = [&](int s) { return s < n_a ? id_a + s : id_c + (s - n_a); };
        // FAST PATH: if every other piece of the unit has already been counted, this part completes the unit: fold the others'
        // partials into the registers and write the result -- one acquire load and one round trip for the rows, instead of
        // store -> release atomic -> load -> store (four dependent trips, all at the very end of a CTA's stream, where they
        // are the launch's tail: the piece that ends a CTA's range is usually the LAST of its unit to finish, its neighbour
        // having started with it).
        // (The fold below starts from this part's registers and takes the other pieces in stream order; the slow path folds
        // every piece in stream order.  Which of the two runs, and for which piece, is a matter of timing -- two summation
        // orders for one unit.  Deterministic mode therefore has a fast path of its own, after this one.)
        bool completes = false;
        {
            int cur = 0;
            if (lane == 0) asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(cur) : "l"(A.counters + unit) : "memory");
            cur = __shfl_sync(kFull, cur, 0);
            __syncwarp();                                           // orders lane 0's acquire before the other lanes' loads
            completes = cur + part_len == c;
            if (completes && !A.deterministic) {
                float m_f = m_new, l_f = l_new;
                for (int s2 = 0; s2 < nseg; ++s2) {
                    const int pid = piece_of(s2);
                    if (pid == piece.x) continue;
                    float2 ml2 = make_float2(-INFINITY, 0.f);
                    const int64_t row = ((int64_t)unit + pid) * r + (hrow < r ? hrow : 0);
                    if (hrow < r) ml2 = __ldcg(reinterpret_cast<const float2 *>(A.ws_ml + row * 2));
                    const bool has = ml2.y > 0.f;                   // (an empty partial contributes nothing, never NaN)
                    const float m2 = has ? fmaxf(m_f, ml2.x) : m_f;
                    const float w_old = has ? fast_exp2(m_f - m2) : 1.f, w_new = has ? fast_exp2(ml2.x - m2) : 0.f;   // own part empty: exp2(-inf) = 0
#pragma unroll
                    for (int half = 0; half < 2; ++half) {          // the row in two halves: 8 loads in flight per lane (register budget)
                        float2 v[8];
#pragma unroll
                        for (int nt = 0; nt < 8; ++nt)
                            v[nt] = has ? __ldcg(reinterpret_cast<const float2 *>(A.ws_o + row * kDim + col + (half * 8 + nt) * 8)) : make_float2(0.f, 0.f);
#pragma unroll
                        for (int nt = 0; nt < 8; ++nt) {
                            o[half * 8 + nt][0] = fmaf(v[nt].x, w_new, o[half * 8 + nt][0] * w_old);
                            o[half * 8 + nt][1] = fmaf(v[nt].y, w_new, o[half * 8 + nt][1] * w_old);
                        }
                    }
                    l_f = fmaf(ml2.y, w_new, l_f * w_old);
                    m_f = m2;
                }
                if (hrow < r) {
                    const float inv = l_f > 0.f ? 1.f / l_f : 0.f;
                    uint32_t *dst = reinterpret_cast<uint32_t *>(A.out + ((int64_t)unit * r + hrow) * kDim + col);
#pragma unroll
                    for (int nt = 0; nt < 16; ++nt) dst[nt * 4] = pack_bf16(o[nt][0] * inv, o[nt][1] * inv);
                    if (A.lse && (lane & 3) == 0)
                        A.lse[(int64_t)unit * r + hrow] = l_f > 0.f ? (m_f + log2f(l_f)) * kLn2 : -INFINITY;
                }
                if (lane == 0) A.counters[unit] = 0;                // restore the zero for the next call (nobody else is left to touch it)
                return;
            }
        }
        if (completes) {
            // DETERMINISTIC FAST PATH: the same saving (no store / atomic / re-load of this part), but the fold is the slow
            // path's, operation for operation: pieces in stream order from an empty state, this part's registers taking
            // their place in that order.  Pieces before it are folded into a temporary, a half row at a time (register
            // budget); the (m, l) recurrence is recomputed for each half, so both halves see identical weights.
            int own = 0;
            while (piece_of(own) != piece.x) ++own;
            const int64_t row_of0 = (int64_t)unit * r + (hrow < r ? hrow : 0);
            float m_f = -INFINITY, l_f = 0.f;
#pragma unroll
            for (int half = 0; half < 2; ++half) {
                float2 acc[8];
#pragma unroll
                for (int nt = 0; nt < 8; ++nt) acc[nt] = make_float2(0.f, 0.f);
                float m_a = -INFINITY, l_a = 0.f;
                for (int s2 = 0; s2 < own; ++s2) {                  // pieces before this one
                    const int64_t row = row_of0 + (int64_t)piece_of(s2) * r;
                    float2 ml2 = make_float2(-INFINITY, 0.f);
                    if (hrow < r) ml2 = __ldcg(reinterpret_cast<const float2 *>(A.ws_ml + row * 2));
                    if (!(ml2.y > 0.f)) continue;                   // empty partial: contributes nothing (as in the slow path)
                    float2 v[8];
#pragma unroll
                    for (int nt = 0; nt < 8; ++nt) v[nt] = __ldcg(reinterpret_cast<const float2 *>(A.ws_o + row * kDim + col + (half * 8 + nt) * 8));
                    const float m2 = fmaxf(m_a, ml2.x);
                    const float w_old = fast_exp2(m_a - m2), w_new = fast_exp2(ml2.x - m2);
                    l_a = fmaf(ml2.y, w_new, l_a * w_old);
#pragma unroll
                    for (int nt = 0; nt < 8; ++nt) {
                        acc[nt].x = fmaf(v[nt].x, w_new, acc[nt].x * w_old);
                        acc[nt].y = fmaf(v[nt].y, w_new, acc[nt].y * w_old);
                    }
                    m_a = m2;
                }
                if (l_new > 0.f) {                                  // this part, from the registers
                    const float m2 = fmaxf(m_a, m_new);
                    const float w_old = fast_exp2(m_a - m2), w_new = fast_exp2(m_new - m2);
                    l_a = fmaf(l_new, w_new, l_a * w_old);
#pragma unroll
                    for (int nt = 0; nt < 8; ++nt) {
                        o[half * 8 + nt][0] = fmaf(o[half * 8 + nt][0], w_new, acc[nt].x * w_old);
                        o[half * 8 + nt][1] = fmaf(o[half * 8 + nt][1], w_new, acc[nt].y * w_old);
                    }
                    m_a = m2;
                } else {
#pragma unroll
                    for (int nt = 0; nt < 8; ++nt) { o[half * 8 + nt][0] = acc[nt].x; o[half * 8 + nt][1] = acc[nt].y; }
                }
                for (int s2 = own + 1; s2 < nseg; ++s2) {           // pieces after this one
                    const int64_t row = row_of0 + (int64_t)piece_of(s2) * r;
                    float2 ml2 = make_float2(-INFINITY, 0.f);
                    if (hrow < r) ml2 = __ldcg(reinterpret_cast<const float2 *>(A.ws_ml + row * 2));
                    if (!(ml2.y > 0.f)) continue;
                    float2 v[8];
#pragma unroll
                    for (int nt = 0; nt < 8; ++nt) v[nt] = __ldcg(reinterpret_cast<const float2 *>(A.ws_o + row * kDim + col + (half * 8 + nt) * 8));
                    const float m2 = fmaxf(m_a, ml2.x);
                    const float w_old = fast_exp2(m_a - m2), w_new = fast_exp2(ml2.x - m2);
                    l_a = fmaf(ml2.y, w_new, l_a * w_old);
#pragma unroll
                    for (int nt = 0; nt < 8; ++nt) {
                        o[half * 8 + nt][0] = fmaf(v[nt].x, w_new, o[half * 8 + nt][0] * w_old);
                        o[half * 8 + nt][1] = fmaf(v[nt].y, w_new, o[half * 8 + nt][1] * w_old);
                    }
                    m_a = m2;
                }
                m_f = m_a; l_f = l_a;
            }
            if (hrow < r) {
                const float inv = l_f > 0.f ? 1.f / l_f : 0.f;
                uint32_t *dst = reinterpret_cast<uint32_t *>(A.out + ((int64_t)unit * r + hrow) * kDim + col);
#pragma unroll
                for (int nt = 0; nt < 16; ++nt) dst[nt * 4] = pack_bf16(o[nt][0] * inv, o[nt][1] * inv);
                if (A.lse && (lane & 3) == 0)
                    A.lse[(int64_t)unit * r + hrow] = l_f > 0.f ? (m_f + log2f(l_f)) * kLn2 : -INFINITY;
            }
            if (lane == 0) A.counters[unit] = 0;                    // restore the zero for the next call
            return;
        }
        // SLOW PATH: park the partial in slot unit + piece id and add this part's tiles to the unit's counter.  Release /
        // acquire through ONE atomic of lane 0: the warp barrier orders the lanes' partial stores before the acq_rel atomic
        // (cumulative at gpu scope), and the barrier after it orders that acquire before the other lanes' reads of the other
        // pieces' slots (ld.global.cg below).  Whoever completes the unit merges the partials in stream order.
        {
            const int64_t gslot = (int64_t)unit + piece.x;          // unique: unit + piece id increases along the stream
            if (hrow < r) {
                float *po = A.ws_o + (gslot * r + hrow) * kDim + col;
#pragma unroll
                for (int nt = 0; nt < 16; ++nt) *reinterpret_cast<float2 *>(po + nt * 8) = make_float2(o[nt][0], o[nt][1]);
                if ((lane & 3) == 0) *reinterpret_cast<float2 *>(A.ws_ml + (gslot * r + hrow) * 2) = make_float2(m_new, l_new);
            }
        }
        __syncwarp();
        int old = 0;
        if (lane == 0)
            asm volatile("atom.acq_rel.gpu.global.add.s32 %0, [%1], %2;" : "=r"(old) : "l"(A.counters + unit), "r"(part_len) : "memory");
        old = __shfl_sync(kFull, old, 0);
        __syncwarp();
        if (old + part_len != c) return;                            // the unit is not complete yet
        if (lane == 0) A.counters[unit] = 0;                        // restore the zero for the next call
        // One pass in stream order, four heads at once (lane = 4 dims of each): the rows and (m, l) pairs of two pieces
        // and four heads are requested together and folded into running (m, l, o) per head, so a unit that spans two
        // pieces -- the usual case -- costs ONE round trip to the L2.  (Head by head with the maxima first it was 2 r
        // dependent round trips, ~9 us at r = 5, all of it at the very end of the launch: traced, profiles/r2_decode.md.)
        constexpr int kSegs = 2, kHeads = 4;                        // heads in groups of four: 8 rows + 8 pairs in flight per lane
        for (int h0 = 0; h0 < r; h0 += kHeads) {
            float4 acc[kHeads];
            float m_acc[kHeads], l_acc[kHeads];
#pragma unroll
            for (int h = 0; h < kHeads; ++h) { acc[h] = make_float4(0.f, 0.f, 0.f, 0.f); m_acc[h] = -INFINITY; l_acc[h] = 0.f; }
            for (int s0 = 0; s0 < nseg; s0 += kSegs) {
                float4 v[kHeads][kSegs];
                float2 ml[kHeads][kSegs];
#pragma unroll
                for (int k = 0; k < kSegs; ++k) {
                    const bool on = s0 + k < nseg;
                    const int64_t row0 = ((int64_t)unit + piece_of(on ? s0 + k : s0)) * r + h0;
#pragma unroll
                    for (int h = 0; h < kHeads; ++h) {
                        v[h][k] = make_float4(0.f, 0.f, 0.f, 0.f);
                        ml[h][k] = make_float2(-INFINITY, 0.f);
                        if (on && h0 + h < r) {
                            v[h][k] = __ldcg(reinterpret_cast<const float4 *>(A.ws_o + (row0 + h) * kDim + lane * 4));
                            ml[h][k] = __ldcg(reinterpret_cast<const float2 *>(A.ws_ml + (row0 + h) * 2));
                        }
                    }
                }
#pragma unroll
                for (int k = 0; k < kSegs; ++k) {
#pragma unroll
                    for (int h = 0; h < kHeads; ++h) {
                        if (!(ml[h][k].y > 0.f)) continue;              // empty partial (or no such piece / head): contributes nothing, never NaN
                        const float m_new2 = fmaxf(m_acc[h], ml[h][k].x);
                        const float w_old = fast_exp2(m_acc[h] - m_new2), w_new = fast_exp2(ml[h][k].x - m_new2);   // first piece: w_old = exp2(-inf) = 0
                        l_acc[h] = fmaf(ml[h][k].y, w_new, l_acc[h] * w_old);
                        acc[h].x = fmaf(v[h][k].x, w_new, acc[h].x * w_old); acc[h].y = fmaf(v[h][k].y, w_new, acc[h].y * w_old);
                        acc[h].z = fmaf(v[h][k].z, w_new, acc[h].z * w_old); acc[h].w = fmaf(v[h][k].w, w_new, acc[h].w * w_old);
                        m_acc[h] = m_new2;
                    }
                }
            }
#pragma unroll
            for (int h = 0; h < kHeads; ++h) {
                if (h0 + h >= r) break;
                const float inv = l_acc[h] > 0.f ? 1.f / l_acc[h] : 0.f;
                uint2 pk;
                pk.x = pack_bf16(acc[h].x * inv, acc[h].y * inv);
                pk.y = pack_bf16(acc[h].z * inv, acc[h].w * inv);
                *reinterpret_cast<uint2 *>(A.out + ((int64_t)unit * r + h0 + h) * kDim + lane * 4) = pk;
                if (A.lse && lane == 0)
                    A.lse[(int64_t)unit * r + h0 + h] = l_acc[h] > 0.f ? (m_acc[h] + log2f(l_acc[h])) * kLn2 : -INFINITY;
            }
        }
    };

    int part = -1, unit = 0, n_mine = 0, part_len = 0;              // the part this consumer is accumulating
    int4 piece = make_int4(0, 0, 0, 0);                             // ... and the piece it belongs to (id, begin, end)
    int n_claims = 0;                                               // deterministic mode: chunks this consumer has taken
#pragma unroll 1
    while (true) {
        int cidx = 0;
        if (A.deterministic) {
            // Fixed hand-out: consumer w takes chunks w, w + 8, w + 16 ... of the CTA's stream -- which tiles a consumer
            // sums, and in which order, is then a function of the inputs alone.  (Chunk c lives in stages 2c % 16 and
            // 2c % 16 + 1, so every consumer refills its own two stages; the ring, the descriptors and the parking
            // protocol are unchanged.)
            cidx = warp + n_claims * kDecConsumers;
#if SPARROW_DEC_DET_WINDOW > 0
            // Drift throttle.  With private tile sequences the consumers drift apart like random walks (each waits out its
            // own memory latencies), and the CTA ends with its slowest warp running alone at two tiles in flight.  A
            // consumer therefore starts round k only once every consumer has started round k - kDetWindow: the leaders'
            // landed tiles wait a little, the bandwidth they would have drawn goes to the laggards.  The slowest consumer
            // never waits here, so the order in which parts complete (park) is unaffected.
            if (n_claims > kDetWindow) {
                const int need = (n_claims - kDetWindow) * kDecConsumers * kDecChunk;      // first tile of round k - window
                for (uint32_t n = 0;; ++n) {
                    int lo = lane < kDecConsumers ? lds_volatile(s_pos + lane) : 0x7fffffff;
#pragma unroll
                    for (int of = 4; of > 0; of >>= 1) lo = min(lo, __shfl_xor_sync(kFull, lo, of));
                    lo = __shfl_sync(kFull, lo, 0);
                    if (lo >= need) break;
                    if (n > (1u << 27)) __trap();
                }
            }
#endif
            ++n_claims;
        } else {
            if (lane == 0) cidx = atomicAdd(s_claim, 1);
            cidx = __shfl_sync(kFull, cidx, 0);
        }
        const int it0 = cidx * kDecChunk;
        if (lane == 0) sts_volatile(s_pos + warp, it0);
        const int n_it = exists(it0) ? (exists(it0 + 1) ? 2 : 1) : 0;   // tiles of this claim that exist
        if (n_it == 0) {
            if (lane == 0) sts_volatile(s_pos + warp, 0x7fffffff);
            break;
        }
#pragma unroll 1
        for (int it = it0; it < it0 + n_it; ++it) {
            const int4 d = s_desc[it & (kDescRing - 1)];
            if ((d.z >> 8) != part) {                               // a tile of another part: park the state of the old one
                if (part >= 0) park(part, unit, n_mine, part_len, piece);
                part = d.z >> 8; unit = d.y; n_mine = 0; part_len = d.w;
                piece = s_part[part & (kPartRing - 1)];
#pragma unroll
                for (int nt = 0; nt < 16; ++nt) { o[nt][0] = 0.f; o[nt][1] = 0.f; }
                m_run = -INFINITY; l_run = 0.f;
                if (unit != q_unit) {
                    q_unit = unit;
                    const uint16_t *qrow = A.q + ((int64_t)unit * r + hrow) * kDim + col;
#pragma unroll
                    for (int kk = 0; kk < 8; ++kk) {
                        qa[kk][0] = hrow < r ? __ldg(reinterpret_cast<const uint32_t *>(qrow + kk * 16)) : 0u;
                        qa[kk][1] = hrow < r ? __ldg(reinterpret_cast<const uint32_t *>(qrow + kk * 16 + 8)) : 0u;
                    }
                }
            }
            ++n_mine;
            const int valid = d.z & 31;
            const int stage = it % kDecStages;
            // A consumer may be handed tile `it` while the stage still holds tile it - kDecStages (another consumer's):
            // a parity wait is only meaningful once the barrier has moved on to this tile's phase, i.e. once the tile has
            // been requested (before that, "the phase of the other parity" reads as complete).
            spin_until(s_issued + stage, it);
            mbar_wait(full_u32 + 8 * stage, (it / kDecStages) & 1);
            if (it == 0 && lane == 0) SPARROW_TR(kTraceDecodeCta + blockIdx.x, 4);
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
            // ---- the stage is free: every lane has read it; the consumer that used it refills it with the tile one ring
            // further on (generic-proxy accesses to the stage -- the reads, the zeroing -- are ordered before the copy
            // engine's writes by the proxy fence) ----
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            const bool more = exists(it + kDecStages);
            if (more && lane == 0) issue(it + kDecStages);
        }
    }
    if (part >= 0) park(part, unit, n_mine, part_len, piece);
    // ---- the last CTA out restores the tail counter's zero for the next call (every CTA's look-up warp has made its last
    // claim before its consumers see the end of the stream) ----
    if (warp == 0 && lane == 0) {
        const int done = atomicAdd(done_ctr, 1);
        if (done == G - 1) {
            *tail_ctr = 0;
            *done_ctr = 0;
        }
    }
    if (lane == 0) SPARROW_TR(kTraceDecodeWarp + blockIdx.x * (kDecThreads / 32) + warp, 1);
}

}  // namespace sparrow
