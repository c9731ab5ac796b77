// step.cuh -- the whole sparse decode step in ONE persistent launch: budget + forced pages (a2, a3), page scoring
// (a4), per-(sequence, kv-head) top-k (a5), split-K flash-decode over the selected pages with the LSE merge (a6, a7).
// SURVEY.md 8(a); PAPER.md:138-147 (landmark scores -> Top-k -> attention over the budget), :109-121 (B(L)).
//
// Why one launch: select and decode are two short HBM streams (cfg2: 160 MB + 538 MB, ~25 us + ~80 us at the
// roofline); as two kernels each pays its own ramp-up, its own tail (the top-k of the last units with HBM idle, the
// last merges) and a launch gap.  Here the same 148 x 8 warps first stream the summaries, and every warp moves on to
// the K/V stream as soon as its share of the scoring is done; the only synchronisation is one flag per
// (sequence, kv-head) unit, set when the unit's page list is written and waited for by the decode look-ups that need
// it.  MEASURED (profiles/r1_v7_cfg2.md): exact and parity-green, but not faster than the two launches
// yet -- all units finish scoring together and the single-warp top-k (13-40 us) then holds every decoder up -- so the
// two-launch form stays the library's default and this kernel is the opt-in single-launch form.
//
// Scoring phase (per warp, no CTA-wide barrier): the candidate pages of the batch form a flat stream of 32-page
// warp-chunks, ordered (sequence, kv-head, chunk), cut into equal contiguous ranges.  A chunk's summaries (512 B per
// page: min | max) are gathered through the page table with 16-byte cp.async into the warp's K/V ring (idle in this
// phase) used as four 4 KiB slots of 8 pages, three in flight while the fourth is scored; page-table entries are
// fetched two chunks ahead.  The score is the R5 closed form
//   s[p] = sum_d ( Q+[d]*mx[d] + Q-[d]*mn[d] ),  Q+ = sum_h max(q_h,0), Q- = sum_h min(q_h,0)
// (lane = one 16-byte piece of the summary = 8 channels of min or of max; transpose-reduce over the warp).
// The warp that completes a unit (one atomic counter per unit) runs its top-k alone (warp_topk below) in its own
// shared-memory scratch (one CTA-wide scratch behind a lock when eight do not fit), then releases the unit's flag.
// Sequences that are dense under the schedule (R13) write the identity list chunk by chunk and skip the scoring.
//
// Decode phase: decode_warp_stream<false, true> of decode.cuh, unchanged but for the flag wait.
// The grid must be co-resident (a waiting warp relies on the warp that owns the unit's last chunk to be running):
// the launch is cooperative, one CTA per SM.
#pragma once
#include "decode.cuh"
#include "select.cuh"

namespace sparrow {

struct StepArgs {
    DecodeArgs dec;              // dec.sel_pages / dec.ready alias sel_pages / ready below (read side)
    const uint16_t *summaries;
    int32_t *sel_pages;          // [n_seq][Hkv][max_sel] written here
    int32_t *sel_count;          // [n_seq]
    float *scores_ws;            // [units][ws_stride] fp32, ws_stride = max_pages rounded up to 32 (rows own their 128-byte lines)
    int ws_stride;
    float *scores_dbg;           // optional, same shape
    int32_t *sel_counters;       // [units] chunks scored so far (zero between calls)
    int32_t *ready;              // [units] page list written (zero between calls)
    int max_rounds;              // cap of the decode range table
    int scratch_stride;          // top-k scratch: keys per warp (each warp its own), or 0 = one scratch per CTA behind a lock
};

// sum of 8 per-lane partial dot products over the warp: afterwards lane l holds the total of value
// j(l) = 4*bit4(l) + 2*bit3(l) + bit2(l); the caller fetches value j from lane 16*(j>>2) + 8*((j>>1)&1) + 4*(j&1).
__device__ __forceinline__ float transpose_reduce8(const float (&a)[8], int lane)
{
    constexpr uint32_t kFull = 0xffffffffu;
    const bool hi = lane & 16;
    float k0 = hi ? a[4] : a[0], k1 = hi ? a[5] : a[1], k2 = hi ? a[6] : a[2], k3 = hi ? a[7] : a[3];
    float s0 = hi ? a[0] : a[4], s1 = hi ? a[1] : a[5], s2 = hi ? a[2] : a[6], s3 = hi ? a[3] : a[7];
    k0 += __shfl_xor_sync(kFull, s0, 16);
    k1 += __shfl_xor_sync(kFull, s1, 16);
    k2 += __shfl_xor_sync(kFull, s2, 16);
    k3 += __shfl_xor_sync(kFull, s3, 16);
    const bool h8 = lane & 8;
    float m0 = h8 ? k2 : k0, m1 = h8 ? k3 : k1;
    float t0 = h8 ? k0 : k2, t1 = h8 ? k1 : k3;
    m0 += __shfl_xor_sync(kFull, t0, 8);
    m1 += __shfl_xor_sync(kFull, t1, 8);
    const bool h4 = lane & 4;
    float z = h4 ? m1 : m0, y = h4 ? m0 : m1;
    z += __shfl_xor_sync(kFull, y, 4);
    z += __shfl_xor_sync(kFull, z, 2);
    z += __shfl_xor_sync(kFull, z, 1);
    return z;
}

// Top-k of one (sequence, kv-head) unit by ONE warp (a5): scores of the unit's candidate pages in `ws` (global,
// written by the scoring warps); s_keys (16-byte aligned, >= n_pages rounded up to 4 entries) and s_hist (256) are
// this warp's scratch.  Writes the ascending list: forced pages, every key above the k-th, and the first ties of
// the k-th in page order (R10).  Every scan handles 4 consecutive pages per lane (one 16-byte shared-memory access).
//   1. one cp.async round brings all the scores in; keys = order-preserving uint32 of the fp32 score (exact order)
//   2. a histogram over 256 LINEAR bins of the score range (monotone in the score, so it never reorders keys, and
//      unlike the top bits of a float it spreads the keys: no atomic pile-up) finds the bin of the k-th key
//   3. keys of higher bins become kSure, of lower bins kNever; an 8-bit radix select over the exact keys that are
//      left (few) finds the k-th key itself;  4. ordered compaction.
constexpr uint32_t kKeyForced = 0u, kKeyNever = 1u, kKeySure = 0xffffffffu;     // no finite score has these keys

__device__ __forceinline__ float key_to_float(uint32_t key)
{
    return __uint_as_float((key & 0x80000000u) ? (key & 0x7fffffffu) : ~key);
}

// suffix scan over the 256 bins of s_hist: finds the bin holding the kk-th key counted from the top.
// Returns the bin; kk becomes the rank inside that bin, hcnt the bin's population.
__device__ __forceinline__ int find_bin(const int *s_hist, int &kk, int &hcnt, int lane)
{
    constexpr uint32_t kFull = 0xffffffffu;
    int h[8], tot = 0;                   // lane owns bins [8*lane, 8*lane + 8)
#pragma unroll
    for (int i = 0; i < 8; ++i) { h[i] = s_hist[lane * 8 + i]; tot += h[i]; }
    int inc = tot;                       // inclusive suffix sum over lanes
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_down_sync(kFull, inc, o);
        if (lane + o < 32) inc += v;
    }
    int run = inc - tot, bin = -1, kk_new = 0, hc = 0;
#pragma unroll
    for (int i = 7; i >= 0; --i) {
        if (run < kk && run + h[i] >= kk) { bin = lane * 8 + i; kk_new = kk - run; hc = h[i]; }
        run += h[i];
    }
    const uint32_t who = __ballot_sync(kFull, bin >= 0);             // exactly one lane holds it
    const int src = who ? __ffs(who) - 1 : 0;
    kk = __shfl_sync(kFull, kk_new, src);
    hcnt = __shfl_sync(kFull, hc, src);
    return __shfl_sync(kFull, bin, src);
}

__device__ __forceinline__ void warp_topk(const SeqPlan &pl, const float *__restrict__ ws, uint32_t *s_keys, int *s_hist,
                                          int32_t *__restrict__ out, int max_sel, int lane)
{
    constexpr uint32_t kFull = 0xffffffffu;
    const int n_pages = pl.n_pages;
    const int n4 = (n_pages + 3) >> 2;
    uint4 *k4 = reinterpret_cast<uint4 *>(s_keys);
    {   // 1. scores -> keys
        const uint32_t dst = smem_u32(s_keys);
        for (int v = lane; v < n4; v += 32) cp_async16(dst + v * 16, ws + v * 4);    // rows are 128-byte aligned and padded
        cp_async_commit();
        cp_async_wait<0>();
        __syncwarp();
    }
    uint32_t kmin = 0xffffffffu, kmax = 0u;
#pragma unroll 2
    for (int v = lane; v < n4; v += 32) {
        uint4 x = k4[v];
        uint32_t e[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int p = v * 4 + i;
            const bool cand = p < n_pages && !pl.forced(p);
            e[i] = cand ? order_key(__uint_as_float(e[i])) : kKeyForced;
            if (cand) { kmin = min(kmin, e[i]); kmax = max(kmax, e[i]); }
        }
        k4[v] = make_uint4(e[0], e[1], e[2], e[3]);
    }
#pragma unroll
    for (int of = 16; of > 0; of >>= 1) {
        kmin = min(kmin, __shfl_xor_sync(kFull, kmin, of));
        kmax = max(kmax, __shfl_xor_sync(kFull, kmax, of));
    }
    __syncwarp();

    uint32_t prefix = 0, mask = 0;
    int need_eq = 0;
    if (pl.k > 0) {
        // 2. linear bins: bin(key) = floor((score - vmin) * scale), monotone in the score
        const float vmin = key_to_float(kmin), vmax = key_to_float(kmax);
        const float scale = vmax > vmin ? 255.f / (vmax - vmin) : 0.f;
        auto lin_bin = [&](uint32_t key) {
            const int b = (int)((key_to_float(key) - vmin) * scale);
            return b < 0 ? 0 : (b > 255 ? 255 : b);
        };
#pragma unroll
        for (int i = 0; i < 8; ++i) s_hist[i * 32 + lane] = 0;
        __syncwarp();
#pragma unroll 2
        for (int v = lane; v < n4; v += 32) {
            const uint4 x = k4[v];
            const uint32_t e[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
            for (int i = 0; i < 4; ++i)
                if (e[i] != kKeyForced) atomicAdd(&s_hist[lin_bin(e[i])], 1);
        }
        __syncwarp();
        int kk = pl.k, hcnt = 0;
        const int bstar = find_bin(s_hist, kk, hcnt, lane);
        need_eq = kk;
        __syncwarp();
        // 3. classify by bin; radix select over the exact keys of the k-th key's bin (the rewrite rides on pass 0)
        const bool whole = kk == hcnt;                               // the bin is taken whole: no exact pass needed
        for (int pass = 0; pass < 4; ++pass) {
            const int shift = 24 - 8 * pass;
#pragma unroll
            for (int i = 0; i < 8; ++i) s_hist[i * 32 + lane] = 0;
            __syncwarp();
#pragma unroll 2
            for (int v = lane; v < n4; v += 32) {
                const uint4 x = k4[v];
                uint32_t e[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    if (pass == 0 && e[i] != kKeyForced) {
                        const int b = lin_bin(e[i]);
                        if (b > bstar || (whole && b == bstar)) e[i] = kKeySure;
                        else if (b < bstar) e[i] = kKeyNever;
                    }
                    const bool in_class = e[i] != kKeyForced && e[i] != kKeyNever && e[i] != kKeySure;
                    if (!whole && in_class && (e[i] & mask) == prefix) atomicAdd(&s_hist[(e[i] >> shift) & 255u], 1);
                }
                if (pass == 0) k4[v] = make_uint4(e[0], e[1], e[2], e[3]);
            }
            __syncwarp();
            if (whole) break;
            const int bin = find_bin(s_hist, kk, hcnt, lane);
            prefix |= (uint32_t)bin << shift;
            mask |= 255u << shift;
            need_eq = kk;
            __syncwarp();
            if (kk == hcnt) break;                                   // the whole class is taken
        }
        if (whole) { need_eq = 0; prefix = 0xffffffffu; mask = 0xffffffffu; }   // nothing of the class is left to pick
    }
    __syncwarp();

    // 4. ordered compaction: lane owns pages 4v .. 4v + 3; exclusive scans over the lanes keep page order
    int pos = 0, eq_seen = 0;
    for (int v0 = 0; v0 < n4; v0 += 32) {
        const int v = v0 + lane;
        uint32_t e[4] = {kKeyNever, kKeyNever, kKeyNever, kKeyNever};
        if (v < n4) {
            const uint4 x = k4[v];
            e[0] = x.x; e[1] = x.y; e[2] = x.z; e[3] = x.w;
        }
        bool take[4], eq[4];
        int n_eq = 0;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int p = v * 4 + i;
            take[i] = false; eq[i] = false;
            if (p < n_pages) {
                if (e[i] == kKeyForced) take[i] = pl.forced(p);
                else if (e[i] == kKeySure) take[i] = true;
                else if (e[i] != kKeyNever && pl.k > 0) {
                    const uint32_t c = e[i] & mask;
                    take[i] = c > prefix;
                    eq[i] = c == prefix;
                }
            }
            n_eq += eq[i];
        }
        int eq_inc = n_eq;                                           // ties: rank in page order
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(kFull, eq_inc, o);
            if (lane >= o) eq_inc += t;
        }
        int rank = eq_seen + eq_inc - n_eq, n_take = 0;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            if (eq[i]) { if (rank < need_eq) take[i] = true; ++rank; }
            n_take += take[i];
        }
        int tk_inc = n_take;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(kFull, tk_inc, o);
            if (lane >= o) tk_inc += t;
        }
        int idx = pos + tk_inc - n_take;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            if (take[i]) {
                if (idx < max_sel) out[idx] = v * 4 + i;
                ++idx;
            }
        }
        pos += __shfl_sync(kFull, tk_inc, 31);
        eq_seen += __shfl_sync(kFull, eq_inc, 31);
    }
}

// One 32-page warp-chunk of the scoring stream as its warp sees it.
struct ChunkDesc {
    int unit, seq, g, ci, nwc;   // warp-uniform: (sequence, kv-head), chunk index inside the unit, chunks of the unit
    SeqPlan pl;                  // warp-uniform
    uint32_t cand_mask;          // bit j: page 32*ci + j is a candidate
    int my_page, phys;           // lane = page: logical page and its page-table entry
    bool my_cand;
};

__global__ void __launch_bounds__(kDecThreads, 1)
step_kernel(const StepArgs S, const SchedDev sched)
{
    chain_entry();
    extern __shared__ __align__(1024) uint8_t smem[];
    const DecodeArgs &A = S.dec;
    const int n_seq = A.n_seq, n_kv_heads = A.n_kv_heads, max_sel = A.max_sel, max_pages = A.max_pages;
    int32_t *s_prefix = reinterpret_cast<int32_t *>(smem + kDecRingBytes);     // [n_seq + 1] list entries before sequence i
    int32_t *s_wc = s_prefix + (n_seq + 1);                                    // [n_seq + 1] 32-page chunks before sequence i
    uint32_t *s_keys = reinterpret_cast<uint32_t *>(                          // top-k scratch, 16-byte aligned
        (reinterpret_cast<uintptr_t>(s_wc + (n_seq + 1)) + 15) & ~(uintptr_t)15);
    __shared__ int s_scan[2][kDecWarps];
    __shared__ DecSchedule s_sched;
    __shared__ int s_hist[kDecWarps][256];
    __shared__ int s_lock;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r = A.n_q_heads / n_kv_heads;
    constexpr uint32_t kFull = 0xffffffffu;

    // ---- prologue: per sequence, list length (from the plan: no dependence on the scoring) and chunk count ----
    {
        const int per = (n_seq + kDecThreads - 1) / kDecThreads;
        const int s0 = min(tid * per, n_seq), s1 = min(s0 + per, n_seq);
        auto counts_of = [&](int s, int &cnt, int &wc) {
            const SeqPlan pl = make_plan(sched, __ldg(A.seq_lens + s));
            cnt = pl.count < max_sel ? pl.count : max_sel;
            wc = (pl.n_pages + 31) >> 5;
            if (blockIdx.x == 0) S.sel_count[s] = cnt;
        };
        int sum_c = 0, sum_w = 0;
        for (int s = s0; s < s1; ++s) { int c, w; counts_of(s, c, w); sum_c += c; sum_w += w; }
        int inc_c = sum_c, inc_w = sum_w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int tc = __shfl_up_sync(kFull, inc_c, o), tw = __shfl_up_sync(kFull, inc_w, o);
            if (lane >= o) { inc_c += tc; inc_w += tw; }
        }
        if (lane == 31) { s_scan[0][warp] = inc_c; s_scan[1][warp] = inc_w; }
        if (tid == 0) s_lock = 0;
        __syncthreads();
        int run_c = inc_c - sum_c, run_w = inc_w - sum_w;
        for (int w = 0; w < warp; ++w) { run_c += s_scan[0][w]; run_w += s_scan[1][w]; }
        for (int s = s0; s < s1; ++s) {
            int c, w;
            counts_of(s, c, w);
            s_prefix[s] = run_c; s_wc[s] = run_w;
            run_c += c; run_w += w;
        }
        if (tid == kDecThreads - 1) {
            s_prefix[n_seq] = run_c; s_wc[n_seq] = run_w;
            decode_schedule(run_c * n_kv_heads, S.max_rounds, s_sched);
        }
        __syncthreads();
    }
    const int gw = blockIdx.x * kDecWarps + warp;
    uint8_t *ring = smem + warp * (kDecStages * kStageBytes);
    const uint32_t ring_u32 = smem_u32(ring);
    // (no CTA-wide barrier below this line)

    // =========================================================== scoring phase ===========================
    {
        const int WC = s_wc[n_seq] * n_kv_heads;                     // warp-chunks of the whole batch
        const int per = (WC + kDecW - 1) / kDecW;
        const int a = min(gw * per, WC), b = min(a + per, WC);
        const uint4 *sum16 = reinterpret_cast<const uint4 *>(S.summaries);

        // Q- (lanes 0-15) or Q+ (lanes 16-31), this lane's 8 channels, and the description of the chunk being scored (d),
        // of the next one (dn: its summaries are being requested) and of the one after (dnn: its page-table entries
        // are in flight, a whole chunk ahead of their first use)
        float qc[8], qn[8], qnn[8];
        ChunkDesc d, dn, dnn;
        d.unit = -1; d.seq = -1; dn.unit = -1; dn.seq = -1; dnn.unit = -1; dnn.seq = -1;
        // describe chunk c; `prev` = the description before it (plan and q are reused when they can be)
        auto describe = [&](int c, ChunkDesc &d, const ChunkDesc &prev, float (&qd)[8], const float (&qprev)[8]) {
            int lo = 0, hi = n_seq - 1;
            while (lo < hi) {
                const int mid = (lo + hi + 1) >> 1;
                if (s_wc[mid] * n_kv_heads <= c) lo = mid; else hi = mid - 1;
            }
            while (s_wc[lo + 1] * n_kv_heads <= c) ++lo;
            d.seq = lo;
            d.nwc = s_wc[lo + 1] - s_wc[lo];
            const int rem = c - s_wc[lo] * n_kv_heads;
            d.g = rem / d.nwc;
            d.ci = rem - d.g * d.nwc;
            d.unit = d.seq * n_kv_heads + d.g;
            d.pl = d.seq == prev.seq ? prev.pl : make_plan(sched, __ldg(A.seq_lens + d.seq));
            d.my_page = d.ci * 32 + lane;
            d.my_cand = !d.pl.dense && d.my_page < d.pl.n_pages && !d.pl.forced(d.my_page);
            d.cand_mask = __ballot_sync(kFull, d.my_cand);
            d.phys = d.my_cand ? __ldg(A.page_table + (int64_t)d.seq * max_pages + d.my_page) : 0;
            if (d.unit == prev.unit) {
#pragma unroll
                for (int e = 0; e < 8; ++e) qd[e] = qprev[e];
            } else {
                const uint16_t *qs = A.q + ((int64_t)d.unit * r) * kDim + (lane & 15) * 8;
                const bool want_max = lane >= 16;
#pragma unroll
                for (int e = 0; e < 8; ++e) qd[e] = 0.f;
                for (int h = 0; h < r; ++h) {
                    const uint4 v = __ldg(reinterpret_cast<const uint4 *>(qs + h * kDim));
                    const uint32_t w4[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
                    for (int e = 0; e < 4; ++e) {
                        const float lo_f = bf16_lo(w4[e]), hi_f = bf16_hi(w4[e]);
                        qd[2 * e] += want_max ? fmaxf(lo_f, 0.f) : fminf(lo_f, 0.f);
                        qd[2 * e + 1] += want_max ? fmaxf(hi_f, 0.f) : fminf(hi_f, 0.f);
                    }
                }
            }
        };
        // The warp's ring (2 x 8 KiB) is used as four 4 KiB slots; slot qi holds quarter qi of a chunk = the summaries
        // of its pages [8*qi, 8*qi + 8).  Three quarters are in flight while the fourth is being scored.
        static_assert(kDecStages * kStageBytes >= 4 * 4096, "the scoring pipeline needs 16 KiB of ring per warp");
        auto issue_q = [&](const ChunkDesc &d, int qi) {
            const uint32_t off16 = ((uint32_t)d.phys * (uint32_t)n_kv_heads + (uint32_t)d.g) * 32u;
            const uint32_t dst = ring_u32 + qi * 4096 + lane * 16;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const uint32_t o = __shfl_sync(kFull, off16, qi * 8 + j);
                if ((d.cand_mask >> (qi * 8 + j)) & 1u) cp_async16(dst + j * 512, sum16 + o + lane);
            }
        };
        // scores of those 8 pages: lane 8*qi + j receives page j's score
        auto score_q = [&](const ChunkDesc &d, const float (&qd)[8], int qi, float &my_score) {
            const uint32_t bm = (d.cand_mask >> (qi * 8)) & 0xffu;
            if (bm == 0) return;                                     // warp-uniform
            const uint32_t src = ring_u32 + qi * 4096 + lane * 16;
            float acc[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                acc[j] = 0.f;
                if ((bm >> j) & 1u) acc[j] = dot8(qd, lds128(src + j * 512), 0.f);
            }
            const float z = transpose_reduce8(acc, lane);
            const int j = lane - qi * 8;
            const int from = ((j >> 2) & 1) * 16 + ((j >> 1) & 1) * 8 + (j & 1) * 4;
            const float got = __shfl_sync(kFull, z, from & 31);
            if (j >= 0 && j < 8) my_score = got;
        };

        int done_in_unit = 0;
        if (a < b) describe(a, d, dn, qc, qn);
        if (a + 1 < b) describe(a + 1, dn, d, qn, qc);
#pragma unroll
        for (int qi = 0; qi < 3; ++qi) {
            if (a < b) issue_q(d, qi);
            cp_async_commit();
        }
#pragma unroll 1
        for (int c = a; c < b; ++c) {
            const bool more = c + 1 < b;
            if (c + 2 < b) describe(c + 2, dnn, dn, qnn, qn);        // its page-table entries are in flight from here
            float my_score = 0.f;
#pragma unroll
            for (int qi = 0; qi < 4; ++qi) {
                if (qi == 0) issue_q(d, 3);                          // quarter t + 3 goes into the slot freed by t - 1
                else if (more) issue_q(dn, qi - 1);
                cp_async_commit();
                cp_async_wait<3>();
                __syncwarp();
                score_q(d, qc, qi, my_score);
                __syncwarp();
            }
            // ---- results of the chunk ----
            int32_t *list = S.sel_pages + (int64_t)d.unit * max_sel;
            if (d.pl.dense) {                                        // R13: identity list, no scoring
                if (d.my_page < d.pl.n_pages && d.my_page < max_sel) list[d.my_page] = d.my_page;
            } else if (d.my_cand) {
                S.scores_ws[(int64_t)d.unit * S.ws_stride + d.my_page] = my_score;
                if (S.scores_dbg) S.scores_dbg[(int64_t)d.unit * max_pages + d.my_page] = my_score;
            }
            ++done_in_unit;
            auto turn = [&]() {
                d = dn;
                dn = dnn;
#pragma unroll
                for (int e = 0; e < 8; ++e) { qc[e] = qn[e]; qn[e] = qnn[e]; }
            };
            if (more && dn.unit == d.unit) { turn(); continue; }
            // ---- this warp's share of the unit is done: arrive; the last warp to arrive selects ----
            __threadfence();
            __syncwarp();
            int old = 0;
            if (lane == 0) old = atomicAdd(S.sel_counters + d.unit, done_in_unit);
            old = __shfl_sync(kFull, old, 0);
            if (old + done_in_unit == d.nwc) {
                if (lane == 0) S.sel_counters[d.unit] = 0;           // restore the zero for the next call
                __threadfence();
                if (!d.pl.dense) {
                    const bool shared_scratch = S.scratch_stride == 0;
                    if (shared_scratch && lane == 0) { while (atomicCAS(&s_lock, 0, 1) != 0) __nanosleep(32); }
                    __syncwarp();
                    warp_topk(d.pl, S.scores_ws + (int64_t)d.unit * S.ws_stride, s_keys + warp * S.scratch_stride,
                              s_hist[shared_scratch ? 0 : warp], list, max_sel, lane);
                    __syncwarp();
                    if (shared_scratch && lane == 0) { __threadfence_block(); atomicExch(&s_lock, 0); }
                }
                __threadfence();
                __syncwarp();
                if (lane == 0) st_release(S.ready + d.unit, 1);
            }
            done_in_unit = 0;
            turn();
        }
        cp_async_wait<0>();
        __syncwarp();
    }

    // =========================================================== decode phase ============================
    decode_warp_stream<false, true>(A, s_prefix, s_sched, ring);

    // ---- the last warp out restores the zeros of the range scheduler and of the unit flags for the next call ----
    int last = 0;
    if (lane == 0) last = atomicAdd(A.sched_ctr + 1, 1) == kDecW - 1;
    last = __shfl_sync(kFull, last, 0);
    if (last) {
        for (int u = lane; u < n_seq * n_kv_heads; u += 32) S.ready[u] = 0;
        if (lane == 0) { A.sched_ctr[0] = 0; A.sched_ctr[1] = 0; }
    }
}

}  // namespace sparrow
