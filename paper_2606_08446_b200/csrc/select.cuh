// select.cuh -- kernel (b): fused page scoring + per-(sequence, kv-head) top-k page selection.
// SURVEY.md 8(a) a2-a5; PAPER.md:138-147 ("landmark scores", Top-k), north_star (b).
//
// Grid = (page slices, kv-heads, sequences).  Every CTA scores a slice of pages_per_cta logical pages (phase A, the
// HBM stream: 512 B of summary per candidate page, gathered through the page table); the LAST CTA of a
// (sequence, kv-head) to finish -- found with one atomic counter -- runs the top-k over that unit's scores
// (phase B: radix select on order-preserving keys + ordered compaction).  So the summary stream is spread
// over all SMs no matter how few (sequence, head) units there are, selection stays fused in the launch, and the
// hardware's CTA scheduler balances the SMs.  (Round 2 built and measured four persistent forms of this kernel --
// resident CTAs pulling 256-page items from a counter; per-warp static ranges with a queue of completed units;
// per-CTA ranges with the octets handed out inside the CTA; one 1024-thread CTA per SM -- and each lost 2-8 us to
// this one at cfg2 / cfg5: static ranges end 6-8 us apart because CTAs that share an SM are not served equally, and
// work stealing fine enough to fix that costs a dependent round trip per 4 KiB.  profiles/r2_select.md.)
//
// Phase B starts its radix select at the first bit in which the unit's keys differ (scores of one unit share sign,
// exponent and often more: a fixed top-down pass spends its first passes on bits that split nothing), 8 bits per
// pass with one histogram bin per thread: typically two passes instead of four, and one packed scan in the
// compaction instead of two.
//
// Score (reading R5): s[p] = sum_{h in group} sum_d max(q_h[d]*mn[d], q_h[d]*mx[d])
//                          = sum_d ( Q+[d]*mx[d] + Q-[d]*mn[d] ),  Q+ = sum_h max(q_h,0), Q- = sum_h min(q_h,0)
// i.e. one 256-long fp32 dot product per page, independent of the GQA ratio r.
//
// Phase A data path: a CTA owns `pages_per_cta` consecutive logical pages of one (sequence, kv-head); its 8 warps
// take 32-page warp-chunks round-robin, with the page-table entries of the next warp-chunk prefetched.  One load
// instruction of a warp reads the whole 512-byte summary of ONE page (lane = 16-byte chunk: lanes 0-15 the min
// vector, 16-31 the max vector), and kSelBatch such loads are issued back to back before the first is consumed
// (kSelBatch x 16 B in flight per lane, kSelBatch x 4 KiB per CTA).  Each lane needs only its 8 entries of Q-/Q+
// in registers.  The per-page partial sums are combined with a transpose-reduce (8 values over 32 lanes in 9
// shuffles).  (A bulk-copy ring was tried in round 1 and dropped: at 512 B per request the copy engine's request
// rate, not HBM, became the limit.)
#pragma once
#include "common.cuh"

namespace sparrow {

constexpr int kSelThreads = 256;
constexpr int kSelWarps = kSelThreads / 32;
constexpr int kSelPagesPerWarp = 32;                    // one warp-chunk: one lane per page-table entry
constexpr int kSelBatch = 8;                            // summaries in flight per warp
#ifndef SPARROW_SEL_MIN_BLOCKS
#define SPARROW_SEL_MIN_BLOCKS 4
#endif
constexpr int kSelMinBlocks = SPARROW_SEL_MIN_BLOCKS;   // CTAs / SM the register budget is held to
constexpr int kSelCtaPagesMin = kSelWarps * kSelPagesPerWarp;                // pages_per_cta is a multiple of this
constexpr int kSelMaxPages = 16384;  // keys of one unit live in shared memory (64 KiB): 262144 tokens
constexpr int kSelRadixBits = 8;     // bits per radix-select pass: one histogram bin per thread of the CTA
constexpr int kSelBins = 1 << kSelRadixBits;
static_assert(kSelBins == kSelThreads, "the radix-select scan gives every thread one bin");

// fp32 -> uint32 whose unsigned order is the float order (larger score = larger key); never 0 for a real score
__device__ __forceinline__ uint32_t order_key(float f)
{
    uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// exclusive prefix sum of one int per thread over the CTA; *total = sum.  warp_sums: kSelWarps ints of smem.
__device__ __forceinline__ int block_excl_scan(int v, int *warp_sums, int *total)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    __syncthreads();                       // previous users of warp_sums are done
    if (lane == 31) warp_sums[w] = inc;
    __syncthreads();
    int before = 0, tot = 0;
#pragma unroll
    for (int i = 0; i < kSelWarps; ++i) {
        const int s = warp_sums[i];
        if (i < w) before += s;
        tot += s;
    }
    *total = tot;
    return before + inc - v;
}

__device__ __forceinline__ float dot8(const float (&qr)[8], const uint4 v, float acc)
{
    acc = fmaf(qr[0], bf16_lo(v.x), acc); acc = fmaf(qr[1], bf16_hi(v.x), acc);
    acc = fmaf(qr[2], bf16_lo(v.y), acc); acc = fmaf(qr[3], bf16_hi(v.y), acc);
    acc = fmaf(qr[4], bf16_lo(v.z), acc); acc = fmaf(qr[5], bf16_hi(v.z), acc);
    acc = fmaf(qr[6], bf16_lo(v.w), acc); acc = fmaf(qr[7], bf16_hi(v.w), acc);
    return acc;
}

// Phase B: top-k of one (sequence, kv-head) unit by the whole CTA (a5).  The unit's candidate scores are in `ws`
// (global, written by the CTAs that scored its slices; visible through the arrival atomic).  Exact, no sort:
//   1. keys -> shared memory (forced pages get the sentinel 0), with the minimum and maximum candidate key;
//   2. radix select for the k-th best key, 8 bits per pass, starting at the highest bit in which minimum and maximum
//      differ (everything above it is common to all keys).  Invariant: the k-th best key has (key & mask) == prefix and
//      is the kk-th best inside that class.  Stops when the class is taken whole (kk == its size) or no bit is left;
//   3. ordered compaction: forced pages, keys above the class, and the first need_eq keys of the class in page order
//      are emitted in ascending page order -- the lower-index tie-break (R10) falls out of the scan order.
__device__ __forceinline__ void unit_topk(const SeqPlan &pl, const float *__restrict__ ws, int32_t *__restrict__ out, int max_sel,
                                          int32_t *__restrict__ sel_count_slot, uint32_t *s_keys, int *s_hist, int *s_warp,
                                          uint32_t *s_red, int *s_bcast, int tr_slot)
{
    (void)tr_slot;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n_pages = pl.n_pages;
    uint32_t kmin = 0xffffffffu, kmax = 0u;
    for (int p = tid; p < n_pages; p += kSelThreads) {
        uint32_t key = 0u;
        if (!pl.forced(p)) {
            key = order_key(__ldcg(ws + p));
            kmin = min(kmin, key);
            kmax = max(kmax, key);
        }
        s_keys[p] = key;
    }
    s_hist[tid] = 0;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        kmin = min(kmin, __shfl_xor_sync(0xffffffffu, kmin, o));
        kmax = max(kmax, __shfl_xor_sync(0xffffffffu, kmax, o));
    }
    if (lane == 0) { s_red[warp] = kmin; s_red[kSelWarps + warp] = kmax; }
    __syncthreads();
#pragma unroll
    for (int w2 = 0; w2 < kSelWarps; ++w2) {
        kmin = min(kmin, s_red[w2]);
        kmax = max(kmax, s_red[kSelWarps + w2]);
    }

    if (threadIdx.x == 0) SPARROW_TR(tr_slot, 7);
    uint32_t prefix = 0, mask = 0;
    int need_eq = 0;                 // how many keys of the final class are taken (lowest page index first, R10)
    if (pl.k > 0) {
        int kk = pl.k;
        const uint32_t diff = kmin ^ kmax;
        int top = diff ? 31 - __clz(diff) : -1;          // highest bit still to be resolved (-1: all candidate keys are equal)
        mask = top < 0 ? 0xffffffffu : (top >= 31 ? 0u : ~((2u << top) - 1u));
        prefix = kmax & mask;
        need_eq = kk;
        int pass = 0;
        while (top >= 0) {
            const int shift = top >= kSelRadixBits - 1 ? top - (kSelRadixBits - 1) : 0;
            const uint32_t dmask = (1u << (top - shift + 1)) - 1u;       // digits of this pass: bits [top, shift]
            for (int p = tid; p < n_pages; p += kSelThreads) {
                const uint32_t key = s_keys[p];
                if (key != 0u && (key & mask) == prefix) atomicAdd(&s_hist[(key >> shift) & dmask], 1);
            }
            __syncthreads();
            // suffix sums over the 256 bins, one bin per thread: S[t] = sum_{j >= t} hist[j]
            const int h = s_hist[tid];
            s_hist[tid] = 0;                             // ready for the next pass
            int suf = h;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int v = __shfl_down_sync(0xffffffffu, suf, o);
                if (lane + o < 32) suf += v;
            }
            if (lane == 0) s_warp[warp] = suf;
            __syncthreads();
            for (int w2 = warp + 1; w2 < kSelWarps; ++w2) suf += s_warp[w2];
            int *bc = s_bcast + 3 * (pass & 1);          // alternate slots: the next pass may write before a slow thread has read
            if (suf >= kk && suf - h < kk) {             // exactly one bin holds the kk-th best key
                bc[0] = tid;
                bc[1] = kk - (suf - h);
                bc[2] = h;
            }
            __syncthreads();
            prefix |= (uint32_t)bc[0] << shift;
            mask |= dmask << shift;
            kk = bc[1];
            need_eq = kk;
            if (kk == bc[2]) break;                      // the whole class is taken: no need to split it further
            top = shift - 1;
            ++pass;
        }
    }

    if (threadIdx.x == 0) SPARROW_TR(tr_slot, 6);
    // Ordered compaction.  Thread t owns the contiguous pages [t*ipt, (t+1)*ipt).  One scan carries both counts: the
    // pages a thread surely emits (low 16 bits) and its members of the final class (high bits).
    const int ipt = (n_pages + kSelThreads - 1) / kSelThreads;
    const int p_lo = tid * ipt, p_hi = min(p_lo + ipt, n_pages);
    int n_eq = 0, n_sure = 0;
    for (int p = p_lo; p < p_hi; ++p) {
        const uint32_t key = s_keys[p];
        if (key == 0u) n_sure += pl.forced(p);
        else if (pl.k > 0) {
            const uint32_t c = key & mask;
            n_sure += c > prefix;
            n_eq += c == prefix;
        }
    }
    int tot;
    const int base = block_excl_scan((n_eq << 16) | n_sure, s_warp, &tot);
    const int eq_base = base >> 16;                      // class members in lower pages
    int eq_left = need_eq - eq_base;                     // class members this thread may still take
    eq_left = eq_left < 0 ? 0 : (eq_left > n_eq ? n_eq : eq_left);
    int pos = (base & 0xffff) + (eq_base < need_eq ? eq_base : need_eq);
    for (int p = p_lo; p < p_hi; ++p) {
        const uint32_t key = s_keys[p];
        bool take;
        if (key == 0u) take = pl.forced(p);
        else if (pl.k > 0) {
            const uint32_t c = key & mask;
            take = c > prefix;
            if (c == prefix && eq_left > 0) { take = true; --eq_left; }
        } else take = false;
        if (take) {
            if (pos < max_sel) out[pos] = p;
            ++pos;
        }
    }
    if (sel_count_slot && tid == 0) {
        const int tot_take = (tot & 0xffff) + ((tot >> 16) < need_eq ? (tot >> 16) : need_eq);
        *sel_count_slot = tot_take < max_sel ? tot_take : max_sel;
    }
}

// kMean: the landmark is one vector per page, the mean key (256 B), scored as (sum_h q_h) . mean -- the form the paper's
// cost model charges (D elements per page); otherwise the min/max pair of north_star (512 B).
template <bool kMean>
__global__ void __launch_bounds__(kSelThreads, kSelMinBlocks)
select_kernel(const uint16_t *__restrict__ q, const uint16_t *__restrict__ summaries,
              const int32_t *__restrict__ page_table, const int32_t *__restrict__ seq_lens,
              const SchedDev sched, int32_t *__restrict__ sel_pages, int max_sel, int32_t *__restrict__ sel_count,
              float *__restrict__ scores_ws, int32_t *__restrict__ counters, float *__restrict__ scores_dbg,
              int n_q_heads, int n_kv_heads, int max_pages, int pages_per_cta)
{
    chain_entry();
    // tracing build only: the linear CTA index while it stays below the decode's slot ranges, else "no slot"
    const long long tr_lin = ((long long)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
    const int tr_slot = tr_lin < kTraceDecodeWarp ? (int)tr_lin : kTraceSlots;
    (void)tr_slot;
    if (threadIdx.x == 0) SPARROW_TR(tr_slot, 0);
    extern __shared__ uint32_t s_keys[];                 // [n_pages] (phase B only)
    __shared__ float s_q[2][kDim];                       // [0] = Q- (pairs with min), [1] = Q+ (pairs with max)
    __shared__ int s_hist[256];
    __shared__ int s_warp[kSelWarps];
    __shared__ int s_bcast[4][3];
    __shared__ uint32_t s_red[2 * kSelWarps];
    __shared__ SeqPlan s_plan;

    const int slice = blockIdx.x, g = blockIdx.y, seq = blockIdx.z;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r = n_q_heads / n_kv_heads;
    const int cta_page0 = slice * pages_per_cta;
    const int32_t *pt = page_table + (int64_t)seq * max_pages;

    // Independent global loads first (sequence length, q, the first page-table entries), so that their latencies
    // overlap instead of chaining: only the summary gather depends on them.
    const int L = seq_lens[seq];
    // A CTA whose slice lies past the sequence's last page has nothing to do (the grid is sized for the longest sequence the
    // page table allows: at cfg4 half of the 8192 CTAs): it leaves here, after one load, before the query rows, the plan and
    // the CTA barrier.  (L <= 0: no pages at all; slice 0 still runs on to write the empty list.)
    if (slice > 0 && (int64_t)cta_page0 << sched.page_log2 >= (int64_t)L) return;
    int phys_cur = 0, phys_nxt = 0;                      // table entries of this warp's chunks i, i+1 (lane = page)
    {
        const int p0 = cta_page0 + warp * kSelPagesPerWarp + lane, p1 = p0 + kSelCtaPagesMin;
        if (p0 < max_pages) phys_cur = __ldg(pt + p0);
        if (p1 < max_pages && p1 < cta_page0 + pages_per_cta) phys_nxt = __ldg(pt + p1);
    }
    float qp = 0.f, qm = 0.f;
    if (tid < kDim) {
        const uint16_t *qs = q + ((int64_t)seq * n_q_heads + g * r) * kDim + tid;
        for (int j = 0; j < r; ++j) {
            const float v = __uint_as_float((uint32_t)__ldg(qs + j * kDim) << 16);
            qp += fmaxf(v, 0.f);
            qm += fminf(v, 0.f);
        }
    }
    // B(L) and the forced-page rule are exact integer arithmetic: one thread evaluates them for the CTA.
    if (tid == 0) s_plan = make_plan(sched, L);
    if (tid < kDim) {
        s_q[0][tid] = kMean ? qp + qm : qm;              // mean landmark: the group's summed query
        s_q[1][tid] = qp;
    }
    __syncthreads();
    if (threadIdx.x == 0) SPARROW_TR(tr_slot, 1);
    const SeqPlan pl = s_plan;
    int32_t *out = sel_pages + ((int64_t)seq * n_kv_heads + g) * max_sel;

    if (pl.dense) {                                      // R13: all pages, no scoring
        if (slice == 0) {
            for (int p = tid; p < pl.n_pages && p < max_sel; p += kSelThreads) out[p] = p;
            if (g == 0 && tid == 0) sel_count[seq] = pl.n_pages < max_sel ? pl.n_pages : max_sel;
        }
        return;
    }
    const int n_chunks = (pl.n_pages + pages_per_cta - 1) / pages_per_cta;
    if (slice >= n_chunks) return;

    // ---------------------------------------------------------------- phase A: score this CTA's pages ----
    float qr[8];                                         // lane = 16-byte chunk of the summary: 8 channels of min or max
#pragma unroll
    for (int e = 0; e < 8; ++e) qr[e] = (&s_q[0][0])[(kMean ? (lane & 15) : lane) * 8 + e];

    const int cta_pages = min(pages_per_cta, pl.n_pages - cta_page0);
    const int n_wc_cta = (cta_pages + kSelPagesPerWarp - 1) / kSelPagesPerWarp;
    const int n_wc = n_wc_cta > warp ? (n_wc_cta - warp + kSelWarps - 1) / kSelWarps : 0;   // warp-chunks of this warp
    float *ws = scores_ws + ((int64_t)seq * n_kv_heads + g) * max_pages;
    const uint4 *sum16 = reinterpret_cast<const uint4 *>(summaries);     // summaries in 16-byte units: 32 per (page, head)
#pragma unroll 1
    for (int i = 0; i < n_wc; ++i) {
        const int my_page = cta_page0 + (warp + i * kSelWarps) * kSelPagesPerWarp + lane;
        const bool my_cand = my_page < pl.n_pages && !pl.forced(my_page);
        const uint32_t cand_mask = __ballot_sync(0xffffffffu, my_cand);  // bit j: page chunk base + j is a candidate
        // offset of this lane's page summary in 16-byte units (< 2^32: up to 64 GiB of summaries)
        uint32_t my_off16 = ((uint32_t)phys_cur * (uint32_t)n_kv_heads + (uint32_t)g) * (kMean ? 16u : 32u);
        // Pages that are not candidates (forced, or past the end) read the first candidate's summary instead (an L2
        // hit) and their score is never stored: every load of a batch is then unconditional, which keeps the loads
        // independent of one another (a predicated load is compiled as load-to-temporary + copy, which serialises).
        {
            const uint32_t safe = __shfl_sync(0xffffffffu, my_off16, cand_mask ? __ffs(cand_mask) - 1 : 0);
            if (!my_cand) my_off16 = safe;
        }
        phys_cur = phys_nxt;                             // prefetch the table entries of the warp-chunk after next
        {
            const int p2 = my_page + 2 * kSelCtaPagesMin;
            phys_nxt = (i + 2 < n_wc && p2 < pl.n_pages) ? __ldg(pt + p2) : 0;
        }
        float my_score = 0.f;                            // score of page chunk base + lane, gathered below
        if constexpr (!kMean) {
            auto load_batch = [&](uint4 (&v)[kSelBatch], int b0) {   // the 8 summaries of pages b0 .. b0 + 7: 8 x 512 B
#pragma unroll
                for (int j = 0; j < kSelBatch; ++j) {
                    const uint32_t off = __shfl_sync(0xffffffffu, my_off16, b0 + j) + lane;
                    v[j] = ldg_stream16(sum16 + off);
                }
            };
            auto reduce_batch = [&](const uint4 (&v)[kSelBatch], int b0) {
                float a[kSelBatch];
#pragma unroll
                for (int j = 0; j < kSelBatch; ++j) a[j] = dot8(qr, v[j], 0.f);
                // transpose-reduce: after the three halving steps lane l holds page j = 4*b4 + 2*b3 + b2 (bits of l),
                // summed over the lanes that differ from l in bits 4, 3, 2; two more butterflies finish the sum.
                static_assert(kSelBatch == 8, "transpose-reduce is written for 8 pages per batch");
                const bool hi = lane & 16;
                float k0 = hi ? a[4] : a[0], k1 = hi ? a[5] : a[1], k2 = hi ? a[6] : a[2], k3 = hi ? a[7] : a[3];
                float s0 = hi ? a[0] : a[4], s1 = hi ? a[1] : a[5], s2 = hi ? a[2] : a[6], s3 = hi ? a[3] : a[7];
                k0 += __shfl_xor_sync(0xffffffffu, s0, 16);
                k1 += __shfl_xor_sync(0xffffffffu, s1, 16);
                k2 += __shfl_xor_sync(0xffffffffu, s2, 16);
                k3 += __shfl_xor_sync(0xffffffffu, s3, 16);
                const bool h8 = lane & 8;
                float m0 = h8 ? k2 : k0, m1 = h8 ? k3 : k1;
                float t0 = h8 ? k0 : k2, t1 = h8 ? k1 : k3;
                m0 += __shfl_xor_sync(0xffffffffu, t0, 8);
                m1 += __shfl_xor_sync(0xffffffffu, t1, 8);
                const bool h4 = lane & 4;
                float z = h4 ? m1 : m0, y = h4 ? m0 : m1;
                z += __shfl_xor_sync(0xffffffffu, y, 4);
                z += __shfl_xor_sync(0xffffffffu, z, 2);
                z += __shfl_xor_sync(0xffffffffu, z, 1);
                // lane l now holds the score of batch page j(l) = ((l>>4)&1)*4 + ((l>>3)&1)*2 + ((l>>2)&1); hand it to
                // the lane that owns that page's table entry (lane b0 + j): source lane for j is 16*(j>>2) + 8*((j>>1)&1) + 4*(j&1).
                const int j = lane - b0;
                const int src = ((j >> 2) & 1) * 16 + ((j >> 1) & 1) * 8 + (j & 1) * 4;
                const float got = __shfl_sync(0xffffffffu, z, src & 31);
                if (j >= 0 && j < kSelBatch) my_score = got;
            };
#pragma unroll 1
            for (int b0 = 0; b0 < kSelPagesPerWarp; b0 += kSelBatch) {
                const uint32_t bm = (cand_mask >> b0) & ((1u << kSelBatch) - 1u);
                if (bm == 0) continue;                   // warp-uniform
                uint4 v[kSelBatch];
                load_batch(v, b0);
                reduce_batch(v, b0);
            }
        } else {
            // 256-byte landmarks: one load instruction covers TWO pages (lanes 0-15 | 16-31), a batch of 8 loads 16 pages
#pragma unroll 1
            for (int b0 = 0; b0 < kSelPagesPerWarp; b0 += 2 * kSelBatch) {
                const uint32_t bm = (cand_mask >> b0) & 0xffffu;
                if (bm == 0) continue;                   // warp-uniform
                const int half = lane >> 4;
                uint4 v[kSelBatch];
#pragma unroll
                for (int j = 0; j < kSelBatch; ++j) {
                    const uint32_t off = __shfl_sync(0xffffffffu, my_off16, b0 + 2 * j + half) + (lane & 15);
                    v[j] = ldg_stream16(sum16 + off);
                }
                float a[kSelBatch];
#pragma unroll
                for (int j = 0; j < kSelBatch; ++j) a[j] = dot8(qr, v[j], 0.f);
                // transpose-reduce inside each 16-lane half: lane l ends with value j = 4*bit3 + 2*bit2 + bit1 of l
                const bool h8 = lane & 8;
                float k0 = h8 ? a[4] : a[0], k1 = h8 ? a[5] : a[1], k2 = h8 ? a[6] : a[2], k3 = h8 ? a[7] : a[3];
                float s0 = h8 ? a[0] : a[4], s1 = h8 ? a[1] : a[5], s2 = h8 ? a[2] : a[6], s3 = h8 ? a[3] : a[7];
                k0 += __shfl_xor_sync(0xffffffffu, s0, 8);
                k1 += __shfl_xor_sync(0xffffffffu, s1, 8);
                k2 += __shfl_xor_sync(0xffffffffu, s2, 8);
                k3 += __shfl_xor_sync(0xffffffffu, s3, 8);
                const bool h4 = lane & 4;
                float m0 = h4 ? k2 : k0, m1 = h4 ? k3 : k1;
                float t0 = h4 ? k0 : k2, t1 = h4 ? k1 : k3;
                m0 += __shfl_xor_sync(0xffffffffu, t0, 4);
                m1 += __shfl_xor_sync(0xffffffffu, t1, 4);
                const bool h2 = lane & 2;
                float z = h2 ? m1 : m0, y = h2 ? m0 : m1;
                z += __shfl_xor_sync(0xffffffffu, y, 2);
                z += __shfl_xor_sync(0xffffffffu, z, 1);
                // page b0 + 2j + half is owned by lane b0 + 2j + half: fetch its total from lane 16*half + 8*(j>>2) + 4*((j>>1)&1) + 2*(j&1)
                const int o = lane - b0, jo = o >> 1, ho = o & 1;
                const int src = ho * 16 + ((jo >> 2) & 1) * 8 + ((jo >> 1) & 1) * 4 + (jo & 1) * 2;
                const float got = __shfl_sync(0xffffffffu, z, src & 31);
                if (o >= 0 && o < 2 * kSelBatch) my_score = got;
            }
        }
        if (my_cand) {                                   // one coalesced 128-byte store per warp
            ws[my_page] = my_score;
            if (scores_dbg) scores_dbg[((int64_t)seq * n_kv_heads + g) * max_pages + my_page] = my_score;
        }
    }

    if (threadIdx.x == 0) SPARROW_TR(tr_slot, 2);
    // ------------------------------------------------ last CTA of this (sequence, kv-head)? --------
    // Release / acquire through ONE atomic of thread 0 instead of a fence by every thread: the CTA barrier orders the
    // warps' score stores before thread 0's acq_rel atomic (cumulative at gpu scope), and in the last CTA the barrier
    // after it orders that acquire before the other threads' reads of the scores (ld.global.cg below).
    __syncthreads();
    if (tid == 0) {
        SPARROW_TR(tr_slot, 3);
        int32_t *ctr = counters + seq * n_kv_heads + g;
        int old;
        asm volatile("atom.acq_rel.gpu.global.add.s32 %0, [%1], 1;" : "=r"(old) : "l"(ctr) : "memory");
        const int last = (old == n_chunks - 1);
        if (last) *ctr = 0;                              // restore the zero for the next call
        s_bcast[0][0] = last;
    }
    __syncthreads();
    if (tid == 0) SPARROW_TR(tr_slot, 4);
    if (!s_bcast[0][0]) return;

    // ---------------------------------------------------------------- phase B: top-k of the unit ----
    unit_topk(pl, ws, out, max_sel, g == 0 ? sel_count + seq : nullptr, s_keys, s_hist, s_warp, s_red, &s_bcast[0][0], tr_slot);
#ifdef SPARROW_TRACE
    __syncthreads();
    if (tid == 0) SPARROW_TR(tr_slot, 5);
#endif
}

}  // namespace sparrow
