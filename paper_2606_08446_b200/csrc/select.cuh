// select.cuh -- kernel (b): fused page scoring + per-(sequence, kv-head) top-k page selection.
// SURVEY.md 8(a) a2-a5; PAPER.md:138-147 ("landmark scores", Top-k), north_star (b).
//
// Grid = (page chunks, kv-heads, sequences).  Every CTA scores a chunk of 256 logical pages (phase A, the
// HBM stream: 512 B of summary per candidate page, gathered through the page table); the LAST CTA of a
// (sequence, kv-head) to finish -- found with one atomic counter -- runs the top-k over that unit's scores
// (phase B: radix select on order-preserving keys + ordered compaction).  So the summary stream is spread
// over all SMs no matter how few (sequence, head) units there are, and selection stays fused in the launch.
//
// Score (reading R5): s[p] = sum_{h in group} sum_d max(q_h[d]*mn[d], q_h[d]*mx[d])
//                          = sum_d ( Q+[d]*mx[d] + Q-[d]*mn[d] ),  Q+ = sum_h max(q_h,0), Q- = sum_h min(q_h,0)
// i.e. one 256-long fp32 dot product per page, independent of the GQA ratio r.
#pragma once
#include "common.cuh"

namespace sparrow {

constexpr int kSelThreads = 256;
constexpr int kSelChunk = 256;       // logical pages per CTA in phase A
constexpr int kSelMaxPages = 16384;  // keys of one unit live in shared memory (64 KiB): 262144 tokens

// fp32 -> uint32 whose unsigned order is the float order (larger score = larger key); never 0 for a real score
__device__ __forceinline__ uint32_t order_key(float f)
{
    uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// exclusive prefix of a 0/1 flag over the 256 threads of the CTA; *total = sum.  warp_sums: 8 ints of smem.
__device__ __forceinline__ int block_excl_scan_flag(bool flag, int *warp_sums, int *total)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const uint32_t b = __ballot_sync(0xffffffffu, flag);
    const int within = __popc(b & ((1u << lane) - 1u));
    __syncthreads();                       // previous users of warp_sums are done
    if (lane == 0) warp_sums[w] = __popc(b);
    __syncthreads();
    int before = 0, tot = 0;
#pragma unroll
    for (int i = 0; i < kSelThreads / 32; ++i) {
        const int v = warp_sums[i];
        if (i < w) before += v;
        tot += v;
    }
    *total = tot;
    return before + within;
}

__global__ void __launch_bounds__(kSelThreads)
select_kernel(const uint16_t *__restrict__ q, const uint16_t *__restrict__ summaries,
              const int32_t *__restrict__ page_table, const int32_t *__restrict__ seq_lens,
              const SchedDev sched, int32_t *__restrict__ sel_pages, int max_sel, int32_t *__restrict__ sel_count,
              float *__restrict__ scores_ws, int32_t *__restrict__ counters, float *__restrict__ scores_dbg,
              int n_q_heads, int n_kv_heads, int max_pages)
{
    extern __shared__ uint32_t s_keys[];                 // [max_pages] (phase B only)
    __shared__ float s_q[2][kDim];                       // [0] = Q- (pairs with min), [1] = Q+ (pairs with max)
    __shared__ int s_hist[256];
    __shared__ int s_warp[kSelThreads / 32];
    __shared__ int s_bcast[2];

    const int chunk = blockIdx.x, g = blockIdx.y, seq = blockIdx.z;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r = n_q_heads / n_kv_heads;
    const SeqPlan pl = make_plan(sched, seq_lens[seq]);
    int32_t *out = sel_pages + ((int64_t)seq * n_kv_heads + g) * max_sel;

    if (pl.dense) {                                      // R13: all pages, no scoring
        if (chunk == 0) {
            for (int p = tid; p < pl.n_pages && p < max_sel; p += kSelThreads) out[p] = p;
            if (g == 0 && tid == 0) sel_count[seq] = pl.n_pages < max_sel ? pl.n_pages : max_sel;
        }
        return;
    }
    const int n_chunks = (pl.n_pages + kSelChunk - 1) / kSelChunk;
    if (chunk >= n_chunks) return;

    // ---------------------------------------------------------------- phase A: score this chunk ----
    if (tid < kDim) {
        float qp = 0.f, qm = 0.f;
        const uint16_t *qs = q + ((int64_t)seq * n_q_heads + g * r) * kDim + tid;
        for (int j = 0; j < r; ++j) {
            const float v = __uint_as_float((uint32_t)qs[j * kDim] << 16);
            qp += fmaxf(v, 0.f);
            qm += fminf(v, 0.f);
        }
        s_q[0][tid] = qm;
        s_q[1][tid] = qp;
    }
    __syncthreads();

    // 8 lanes per page: lane sub-id s reads 16-byte chunks {s, 8+s, 16+s, 24+s} of the 512-byte summary
    // (chunks 0-15 = min, 16-31 = max), so each load instruction of a warp reads 4 x 128 contiguous bytes.
    const int s = lane & 7, slot = lane >> 3;
    float qr[4][8];
    const float *sq = &s_q[0][0];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int e = 0; e < 8; ++e) qr[i][e] = sq[(i * 8 + s) * 8 + e];

    const int32_t *pt = page_table + (int64_t)seq * max_pages;
    float *ws = scores_ws + ((int64_t)seq * n_kv_heads + g) * max_pages;
    constexpr int kIters = kSelChunk / (kSelThreads / 32 * 4);      // 8
    int p_of[kIters];
    int phys[kIters];
#pragma unroll
    for (int it = 0; it < kIters; ++it) {
        const int p = chunk * kSelChunk + it * 32 + warp * 4 + slot;
        const bool cand = p < pl.n_pages && !pl.forced(p);
        p_of[it] = cand ? p : -1;
        phys[it] = cand ? pt[p] : 0;
    }
#pragma unroll
    for (int it = 0; it < kIters; ++it) {
        float acc = 0.f;
        if (p_of[it] >= 0) {
            const uint16_t *src = summaries + ((int64_t)phys[it] * n_kv_heads + g) * kSumElems + s * 8;
            uint4 v[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) v[i] = ldg_stream16(src + i * 64);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                acc = fmaf(qr[i][0], bf16_lo(v[i].x), acc); acc = fmaf(qr[i][1], bf16_hi(v[i].x), acc);
                acc = fmaf(qr[i][2], bf16_lo(v[i].y), acc); acc = fmaf(qr[i][3], bf16_hi(v[i].y), acc);
                acc = fmaf(qr[i][4], bf16_lo(v[i].z), acc); acc = fmaf(qr[i][5], bf16_hi(v[i].z), acc);
                acc = fmaf(qr[i][6], bf16_lo(v[i].w), acc); acc = fmaf(qr[i][7], bf16_hi(v[i].w), acc);
            }
        }
        acc += __shfl_xor_sync(0xffffffffu, acc, 1);
        acc += __shfl_xor_sync(0xffffffffu, acc, 2);
        acc += __shfl_xor_sync(0xffffffffu, acc, 4);
        if (s == 0 && p_of[it] >= 0) {
            ws[p_of[it]] = acc;
            if (scores_dbg) scores_dbg[((int64_t)seq * n_kv_heads + g) * max_pages + p_of[it]] = acc;
        }
    }

    // ------------------------------------------------ last CTA of this (sequence, kv-head)? --------
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        int32_t *ctr = counters + seq * n_kv_heads + g;
        const int old = atomicAdd(ctr, 1);
        const int last = (old == n_chunks - 1);
        if (last) *ctr = 0;                              // restore the zero for the next call
        s_bcast[0] = last;
    }
    __syncthreads();
    if (!s_bcast[0]) return;
    __threadfence();

    // ---------------------------------------------------------------- phase B: top-k of the unit ----
    for (int p = tid; p < pl.n_pages; p += kSelThreads)
        s_keys[p] = pl.forced(p) ? 0u : order_key(__ldcg(ws + p));
    __syncthreads();

    uint32_t thr = 0xffffffffu;      // key of the k-th best candidate
    int need_eq = 0;                 // how many candidates with key == thr are taken (lowest page index first, R10)
    if (pl.k > 0) {
        uint32_t prefix = 0, mask = 0;
        int kk = pl.k;               // rank still to resolve inside the current prefix class (1 = best)
        for (int shift = 24; shift >= 0; shift -= 8) {
            s_hist[tid] = 0;
            __syncthreads();
            for (int p = tid; p < pl.n_pages; p += kSelThreads) {
                const uint32_t key = s_keys[p];
                if ((key & mask) == prefix) atomicAdd(&s_hist[(key >> shift) & 255u], 1);
            }
            __syncthreads();
            // suffix sums over the 256 bins: S[t] = sum_{j >= t} hist[j]
            const int h = s_hist[tid];
            int suf = h;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int v = __shfl_down_sync(0xffffffffu, suf, o);
                if (lane + o < 32) suf += v;
            }
            if (lane == 0) s_warp[warp] = suf;
            __syncthreads();
            for (int w2 = warp + 1; w2 < kSelThreads / 32; ++w2) suf += s_warp[w2];
            if (suf >= kk && suf - h < kk) {             // exactly one bin holds the kk-th best key
                s_bcast[0] = tid;
                s_bcast[1] = kk - (suf - h);
            }
            __syncthreads();
            prefix |= (uint32_t)s_bcast[0] << shift;
            mask |= 255u << shift;
            kk = s_bcast[1];
            __syncthreads();
        }
        thr = prefix;
        need_eq = kk;
    }

    // ordered compaction: forced pages, keys above the threshold, and the first need_eq keys equal to it
    int base_out = 0, base_eq = 0;
    for (int p0 = 0; p0 < pl.n_pages; p0 += kSelThreads) {
        const int p = p0 + tid;
        const bool inb = p < pl.n_pages;
        const uint32_t key = inb ? s_keys[p] : 0u;
        const bool f = inb && pl.forced(p);
        const bool eq = inb && !f && key == thr;
        const bool gt = inb && !f && key > thr;
        int tot_eq, tot_take;
        const int eq_rank = base_eq + block_excl_scan_flag(eq, s_warp, &tot_eq);
        const bool take = f || gt || (eq && eq_rank < need_eq);
        const int pos = base_out + block_excl_scan_flag(take, s_warp, &tot_take);
        if (take && pos < max_sel) out[pos] = p;
        base_eq += tot_eq;
        base_out += tot_take;
    }
    if (g == 0 && tid == 0) sel_count[seq] = base_out < max_sel ? base_out : max_sel;
}

}  // namespace sparrow
