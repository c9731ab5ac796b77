// accept.cuh -- the paper's divergence statistic: per-token acceptance rate between the dense
// policy P and the sparse policy Q, and its tail quantile per length bin.
//   PAPER.md:76-79 Eq. 1   alpha = E_{x~Q}[min(p(x)/q(x), 1)] = sum_x min(p(x), q(x))
//   PAPER.md:95            approximated from the top-20 tokens and logprobs each policy returns per position (R23:
//                          the sum runs over the tokens present in BOTH lists; a token missing from a list adds 0)
//   PAPER.md:101, :119     tokens are grouped by position in 2K bins; the statistic is the 5-percentile per bin
// Two kernels.  alpha: a CTA stages the lists of 128 positions in shared memory with coalesced loads, then ONE THREAD per
// position compares its 20 x 20 ids out of registers.  Quantile: exact nearest-rank selection (rank ceil(quantile * count)) per
// bin by a 3-pass radix select (11 + 11 + 10 bits) over the fp32 bit patterns (alpha >= 0: bit order = value order);
// each pass is one streaming histogram launch (block-private shared-memory histograms of all bins) and one tiny
// scan launch that picks the digit, keeps the remaining rank and clears the histogram for the next pass / call.
#pragma once
#include "common.cuh"

namespace sparrow {

constexpr int kAccDigits = 2048;                  // histogram bins per pass (11 bits)
constexpr int kAccThreads = 256;

// One thread per position.  The slices of the four [n_pos][top_n] arrays that belong to the CTA's kAlphaThreads consecutive
// positions are contiguous, so the CTA stages them with full-width coalesced loads (all issued before the first use) into
// shared-memory rows of odd stride (conflict-free when thread t reads row t).  A thread then holds P's ids in registers and
// walks Q's: top_n x top_n compares on the integer pipe, ~25 warp instructions per position.  (Round 1's form -- a warp
// per four positions, lane = Q entry, P's row scanned with broadcast reads -- spent 214 warp instructions per position and
// was issue-bound at 0.21 of the copy peak on its bytes; lane-per-entry leaves 12 of 32 lanes idle and pays a shuffle
// reduction per position.)  min(p, q) = exp(min(log p, log q)): one exp per matched pair.  The ids of a list are distinct
// (it is a top-N list).
constexpr int kAlphaThreads = 128;
constexpr int kAlphaMaxTop = 32;

template <int kTop>                                  // kTop = 20: the paper's lists; 32: any top_n <= 32
__global__ void __launch_bounds__(kAlphaThreads)
accept_alpha_kernel(const int32_t *__restrict__ ids_p, const float *__restrict__ logp_p, const int32_t *__restrict__ ids_q,
                    const float *__restrict__ logp_q, int64_t n_pos, int top_n, int vec16, float *__restrict__ alpha)
{
    extern __shared__ int s_acc_all[];               // [4][kAlphaThreads][stride]: ids_p | ids_q | logp_p | logp_q
    const int stride = top_n | 1;
    int *s_idp = s_acc_all, *s_idq = s_idp + kAlphaThreads * stride;
    float *s_lp = reinterpret_cast<float *>(s_idq + kAlphaThreads * stride), *s_lq = s_lp + kAlphaThreads * stride;
    const int64_t pos0 = (int64_t)blockIdx.x * kAlphaThreads;
    const int n_here = (int)min((int64_t)kAlphaThreads, n_pos - pos0);
    const int total = n_here * top_n;
    const int64_t g0 = pos0 * top_n;
    if (vec16) {                                                     // top_n a multiple of 4 and the four arrays 16-byte aligned (host)
        // 16-byte loads: the CTA's slice starts on a 16-byte boundary (128 x top_n words) and a row is a whole number of
        // quads, so a quad never straddles two positions; all four arrays' loads of a quad are issued before its stores
        const int qpr = top_n >> 2;                                  // quads per row
        for (int f = threadIdx.x; f < (total >> 2); f += kAlphaThreads) {
            const int k = f / qpr, at = k * stride + ((f - k * qpr) << 2);
            const int4 a = __ldg(reinterpret_cast<const int4 *>(ids_p + g0) + f), b = __ldg(reinterpret_cast<const int4 *>(ids_q + g0) + f);
            const float4 c = __ldg(reinterpret_cast<const float4 *>(logp_p + g0) + f), d = __ldg(reinterpret_cast<const float4 *>(logp_q + g0) + f);
            s_idp[at] = a.x; s_idp[at + 1] = a.y; s_idp[at + 2] = a.z; s_idp[at + 3] = a.w;
            s_idq[at] = b.x; s_idq[at + 1] = b.y; s_idq[at + 2] = b.z; s_idq[at + 3] = b.w;
            s_lp[at] = c.x; s_lp[at + 1] = c.y; s_lp[at + 2] = c.z; s_lp[at + 3] = c.w;
            s_lq[at] = d.x; s_lq[at + 1] = d.y; s_lq[at + 2] = d.z; s_lq[at + 3] = d.w;
        }
    } else {
        for (int e = threadIdx.x; e < total; e += kAlphaThreads) {   // coalesced: consecutive threads, consecutive words
            const int k = e / top_n, at = k * stride + (e - k * top_n);
            s_idp[at] = ids_p[g0 + e];
            s_idq[at] = ids_q[g0 + e];
            s_lp[at] = logp_p[g0 + e];
            s_lq[at] = logp_q[g0 + e];
        }
    }
    __syncthreads();
    const int t = threadIdx.x;
    if (t >= n_here) return;
    int pid[kTop];
#pragma unroll
    for (int k = 0; k < kTop; ++k) pid[k] = k < top_n ? s_idp[t * stride + k] : -1;      // (token ids are >= 0)
    float acc = 0.f;
    for (int i = 0; i < top_n; ++i) {
        const int idq = s_idq[t * stride + i];
        int j = -1;
#pragma unroll
        for (int k = 0; k < kTop; ++k) j = pid[k] == idq ? k : j;
        if (j >= 0) acc += expf(fminf(s_lp[t * stride + j], s_lq[t * stride + i]));
    }
    alpha[pos0 + t] = acc;
}

// per-bin selection state: [0] prefix (key bits fixed so far), [1] mask, [2] remaining rank (1-based, from the
// smallest), [3] count of the bin.
// One streaming pass over (alpha, position) per radix digit: every block keeps a private histogram of ALL bins in
// shared memory ([n_bins_local][2048] ints; the host cuts the bins into groups of n_bins_local that fit, grid.y =
// group) and flushes its non-zero counters with global atomics.
constexpr int kHistThreads = 1024;                // one CTA per SM (its histograms fill the shared memory): as many warps as fit
__global__ void __launch_bounds__(kHistThreads)
accept_hist_kernel(const float *__restrict__ alpha, const int32_t *__restrict__ positions, int64_t n_pos, int bin_tokens,
                   int n_bins, int bins_per_group, int shift, int digit_bits, const uint32_t *__restrict__ state,
                   int32_t *__restrict__ hist)
{
    extern __shared__ int s_hist[];                                  // [bins_per_group][kAccDigits]
    __shared__ uint32_t s_state[64][2];                              // (prefix, mask) of the group's bins (bins_per_group <= 64)
    const int bin0 = blockIdx.y * bins_per_group;
    const int nb = min(bins_per_group, n_bins - bin0);
    for (int i = threadIdx.x; i < nb * kAccDigits; i += kHistThreads) s_hist[i] = 0;
    if (threadIdx.x < 2 * nb) s_state[threadIdx.x >> 1][threadIdx.x & 1] = state[(bin0 + (threadIdx.x >> 1)) * 4 + (threadIdx.x & 1)];
    __syncthreads();
    const uint32_t dmask = (1u << digit_bits) - 1u;
    const int64_t step = (int64_t)gridDim.x * kHistThreads;
    constexpr int kU = 4;                                            // independent (position, alpha) loads in flight per thread
    for (int64_t i0 = (int64_t)blockIdx.x * kHistThreads + threadIdx.x; i0 < n_pos; i0 += kU * step) {
        int pos[kU];
        uint32_t key[kU];
#pragma unroll
        for (int u = 0; u < kU; ++u) {
            const int64_t i = i0 + u * step;
            pos[u] = i < n_pos ? __ldg(positions + i) : -1;
            key[u] = i < n_pos ? __float_as_uint(__ldg(alpha + i)) : 0u;
        }
#pragma unroll
        for (int u = 0; u < kU; ++u) {
            if (i0 + u * step >= n_pos) continue;
            int b = pos[u] / bin_tokens;
            b = (b < 0 ? 0 : (b >= n_bins ? n_bins - 1 : b)) - bin0;
            if (b < 0 || b >= nb) continue;
            if ((key[u] & s_state[b][1]) == s_state[b][0]) atomicAdd(&s_hist[b * kAccDigits + ((key[u] >> shift) & dmask)], 1);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nb * kAccDigits; i += kHistThreads)
        if (s_hist[i]) atomicAdd(&hist[bin0 * kAccDigits + i], s_hist[i]);
}

// one block per bin: find the digit that holds the wanted rank (ascending), update the state, clear the histogram
__global__ void __launch_bounds__(kAccThreads)
accept_scan_kernel(int32_t *__restrict__ hist, uint32_t *__restrict__ state, int shift, int digit_bits, int first_pass,
                   float quantile, int last_pass, float *__restrict__ bin_quantile, int32_t *__restrict__ bin_count)
{
    __shared__ int s_total;
    __shared__ int s_part[kAccThreads];
    const int bin = blockIdx.x, tid = threadIdx.x;
    constexpr int kPer = kAccDigits / kAccThreads;                   // 8 consecutive digits per thread
    int local[kPer], sum = 0;
#pragma unroll
    for (int i = 0; i < kPer; ++i) {
        local[i] = hist[bin * kAccDigits + tid * kPer + i];
        hist[bin * kAccDigits + tid * kPer + i] = 0;                 // ready for the next pass / call
        sum += local[i];
    }
    s_part[tid] = sum;
    __syncthreads();
    if (tid == 0) {                                                  // exclusive prefix over 256 partial sums
        int run = 0;
        for (int i = 0; i < kAccThreads; ++i) { const int v = s_part[i]; s_part[i] = run; run += v; }
        s_total = run;
    }
    __syncthreads();
    const int total = s_total;
    uint32_t rank;
    if (first_pass) {
        // nearest rank: the smallest value whose empirical CDF reaches `quantile`
        int r = (int)ceil((double)quantile * (double)total);       // fp64: the rank is an exact function of (quantile, count)
        r = r < 1 ? 1 : (r > total ? total : r);
        rank = (uint32_t)r;
        if (tid == 0) { bin_count[bin] = total; state[bin * 4 + 3] = (uint32_t)total; }
    } else {
        rank = state[bin * 4 + 2];
    }
    if (total == 0) {
        if (tid == 0 && last_pass) bin_quantile[bin] = __int_as_float(0x7fc00000);       // empty bin: NaN
        return;
    }
    __syncthreads();                                                 // every thread has read the rank before one rewrites it
    int run = s_part[tid];
#pragma unroll
    for (int i = 0; i < kPer; ++i) {
        if ((uint32_t)run < rank && rank <= (uint32_t)(run + local[i])) {   // exactly one (thread, i) holds the rank
            const uint32_t digit = (uint32_t)(tid * kPer + i);
            const uint32_t prefix = state[bin * 4 + 0] | (digit << shift);
            state[bin * 4 + 0] = prefix;
            state[bin * 4 + 1] = state[bin * 4 + 1] | (((1u << digit_bits) - 1u) << shift);
            state[bin * 4 + 2] = rank - (uint32_t)run;
            if (last_pass) bin_quantile[bin] = __uint_as_float(prefix);
        }
        run += local[i];
    }
}

}  // namespace sparrow
