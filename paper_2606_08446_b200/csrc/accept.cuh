// accept.cuh -- the paper's divergence statistic: per-token acceptance rate between the dense
// policy P and the sparse policy Q, and its tail quantile per length bin.
//   PAPER.md:76-79 Eq. 1   alpha = E_{x~Q}[min(p(x)/q(x), 1)] = sum_x min(p(x), q(x))
//   PAPER.md:95            approximated from the top-20 tokens and logprobs each policy returns per position (R23:
//                          the sum runs over the tokens present in BOTH lists; a token missing from a list adds 0)
//   PAPER.md:101, :119     tokens are grouped by position in 2K bins; the statistic is the 5-percentile per bin
// Two kernels.  alpha: one warp per position, lane = list entry (top_n <= 32): the P list is broadcast entry by entry
// and matched against the lane's Q entry.  Quantile: exact nearest-rank selection (rank ceil(quantile * count)) per
// bin by a 3-pass radix select (11 + 11 + 10 bits) over the fp32 bit patterns (alpha >= 0: bit order = value order);
// each pass is one streaming histogram launch (grid.y = bin, block-private shared-memory histogram) and one tiny
// scan launch that picks the digit, keeps the remaining rank and clears the histogram for the next pass / call.
#pragma once
#include "common.cuh"

namespace sparrow {

constexpr int kAccDigits = 2048;                  // histogram bins per pass (11 bits)
constexpr int kAccThreads = 256;

__global__ void __launch_bounds__(kAccThreads)
accept_alpha_kernel(const int32_t *__restrict__ ids_p, const float *__restrict__ logp_p, const int32_t *__restrict__ ids_q,
                    const float *__restrict__ logp_q, int64_t n_pos, int top_n, float *__restrict__ alpha)
{
    const int lane = threadIdx.x & 31;
    const int64_t pos = (int64_t)blockIdx.x * (kAccThreads / 32) + (threadIdx.x >> 5);
    if (pos >= n_pos) return;
    const bool on = lane < top_n;
    const int idp = on ? ids_p[pos * top_n + lane] : -1;
    const float pp = on ? expf(logp_p[pos * top_n + lane]) : 0.f;
    const int idq = on ? ids_q[pos * top_n + lane] : -2;
    const float qq = on ? expf(logp_q[pos * top_n + lane]) : 0.f;
    float acc = 0.f;
    for (int i = 0; i < top_n; ++i) {
        const int id = __shfl_sync(0xffffffffu, idp, i);
        const float p = __shfl_sync(0xffffffffu, pp, i);
        if (on && idq == id) acc += fminf(p, qq);
    }
#pragma unroll
    for (int of = 16; of > 0; of >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, of);
    if (lane == 0) alpha[pos] = acc;
}

// per-bin selection state: [0] prefix (key bits fixed so far), [1] mask, [2] remaining rank (1-based, from the
// smallest), [3] count of the bin
__global__ void __launch_bounds__(kAccThreads)
accept_hist_kernel(const float *__restrict__ alpha, const int32_t *__restrict__ positions, int64_t n_pos, int bin_tokens,
                   int n_bins, int shift, int digit_bits, const uint32_t *__restrict__ state, int32_t *__restrict__ hist)
{
    __shared__ int s_hist[kAccDigits];
    const int bin = blockIdx.y;
    for (int i = threadIdx.x; i < kAccDigits; i += kAccThreads) s_hist[i] = 0;
    __syncthreads();
    const uint32_t prefix = state[bin * 4 + 0], mask = state[bin * 4 + 1];
    const uint32_t dmask = (1u << digit_bits) - 1u;
    for (int64_t i = (int64_t)blockIdx.x * kAccThreads + threadIdx.x; i < n_pos; i += (int64_t)gridDim.x * kAccThreads) {
        int b = positions[i] / bin_tokens;
        b = b < 0 ? 0 : (b >= n_bins ? n_bins - 1 : b);
        if (b != bin) continue;
        const uint32_t key = __float_as_uint(alpha[i]);
        if ((key & mask) == prefix) atomicAdd(&s_hist[(key >> shift) & dmask], 1);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < kAccDigits; i += kAccThreads)
        if (s_hist[i]) atomicAdd(&hist[bin * kAccDigits + i], s_hist[i]);
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
