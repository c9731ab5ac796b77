// accept.cuh -- the paper's divergence statistic: per-token acceptance rate between the dense
// policy P and the sparse policy Q, and its tail quantile per length bin.
//   PAPER.md:76-79 Eq. 1   alpha = E_{x~Q}[min(p(x)/q(x), 1)] = sum_x min(p(x), q(x))
//   PAPER.md:95            approximated from the top-20 tokens and logprobs each policy returns per position (R23:
//                          the sum runs over the tokens present in BOTH lists; a token missing from a list adds 0)
//   PAPER.md:101, :119     tokens are grouped by position in 2K bins; the statistic is the 5-percentile per bin
// Two kernels.  alpha: a warp stages the lists of four positions in shared memory with coalesced loads, then per
// position lane = Q entry scans P's row with 16-byte broadcast reads.  Quantile: exact nearest-rank selection (rank ceil(quantile * count)) per
// bin by a 3-pass radix select (11 + 11 + 10 bits) over the fp32 bit patterns (alpha >= 0: bit order = value order);
// each pass is one streaming histogram launch (block-private shared-memory histograms of all bins) and one tiny
// scan launch that picks the digit, keeps the remaining rank and clears the histogram for the next pass / call.
#pragma once
#include "common.cuh"

namespace sparrow {

constexpr int kAccDigits = 2048;                  // histogram bins per pass (11 bits)
constexpr int kAccThreads = 256;

// One warp per kAccPosPerWarp consecutive positions.  Their slices of the four [n_pos][top_n] arrays are contiguous, so
// the warp stages them with full-width coalesced loads (all issued before the first use: ~1.5 KiB in flight per
// warp) into shared memory rows padded to 32 entries.  Then, per position, lane = Q entry: it scans P's row four ids
// per 16-byte broadcast read.  (One position per warp with 80-byte loads was latency bound, a 20-step shuffle loop
// shuffle bound; __match_any_sync pairing and a thread-per-position outward search were slower still.)
// min(p, q) = exp(min(log p, log q)): one exp per matched pair.
constexpr int kAccPosPerWarp = 4;

__global__ void __launch_bounds__(kAccThreads)
accept_alpha_kernel(const int32_t *__restrict__ ids_p, const float *__restrict__ logp_p, const int32_t *__restrict__ ids_q,
                    const float *__restrict__ logp_q, int64_t n_pos, int top_n, float *__restrict__ alpha)
{
    constexpr int kW = kAccThreads / 32, kP = kAccPosPerWarp;
    __shared__ __align__(16) int s_idp[kW][kP][32];
    __shared__ int s_idq[kW][kP][32];
    __shared__ float s_lp[kW][kP][32], s_lq[kW][kP][32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t pos0 = ((int64_t)blockIdx.x * kW + warp) * kP;
    if (pos0 >= n_pos) return;
    const int n_here = (int)min((int64_t)kP, n_pos - pos0);
    const int total = n_here * top_n;
#pragma unroll
    for (int k = 0; k < kP; ++k) s_idp[warp][k][lane] = -1;              // padding never matches a token id
    __syncwarp();
    const int64_t g0 = pos0 * top_n;
#pragma unroll
    for (int e0 = 0; e0 < kP * 32; e0 += 32) {
        const int e = e0 + lane;
        if (e < total) {
            const int k = e / top_n, i = e - k * top_n;
            s_idp[warp][k][i] = ids_p[g0 + e];
            s_idq[warp][k][i] = ids_q[g0 + e];
            s_lp[warp][k][i] = logp_p[g0 + e];
            s_lq[warp][k][i] = logp_q[g0 + e];
        }
    }
    __syncwarp();
    for (int k = 0; k < n_here; ++k) {
        float acc = 0.f;
        if (lane < top_n) {
            const int idq = s_idq[warp][k][lane];
            const int4 *row = reinterpret_cast<const int4 *>(s_idp[warp][k]);
            int j = -1;
            for (int i = 0; i < top_n; i += 4) {
                const int4 v = row[i >> 2];
                j = v.x == idq ? i : (v.y == idq ? i + 1 : (v.z == idq ? i + 2 : (v.w == idq ? i + 3 : j)));
            }
            if (j >= 0) acc = expf(fminf(s_lp[warp][k][j], s_lq[warp][k][lane]));
        }
#pragma unroll
        for (int of = 16; of > 0; of >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, of);
        if (lane == 0) alpha[pos0 + k] = acc;
    }
}

// per-bin selection state: [0] prefix (key bits fixed so far), [1] mask, [2] remaining rank (1-based, from the
// smallest), [3] count of the bin.
// One streaming pass over (alpha, position) per radix digit: every block keeps a private histogram of ALL bins in
// shared memory ([n_bins_local][2048] ints; the host cuts the bins into groups of n_bins_local that fit, grid.y =
// group) and flushes its non-zero counters with global atomics.
__global__ void __launch_bounds__(kAccThreads)
accept_hist_kernel(const float *__restrict__ alpha, const int32_t *__restrict__ positions, int64_t n_pos, int bin_tokens,
                   int n_bins, int bins_per_group, int shift, int digit_bits, const uint32_t *__restrict__ state,
                   int32_t *__restrict__ hist)
{
    extern __shared__ int s_hist[];                                  // [bins_per_group][kAccDigits]
    const int bin0 = blockIdx.y * bins_per_group;
    const int nb = min(bins_per_group, n_bins - bin0);
    for (int i = threadIdx.x; i < nb * kAccDigits; i += kAccThreads) s_hist[i] = 0;
    __syncthreads();
    const uint32_t dmask = (1u << digit_bits) - 1u;
    for (int64_t i = (int64_t)blockIdx.x * kAccThreads + threadIdx.x; i < n_pos; i += (int64_t)gridDim.x * kAccThreads) {
        int b = positions[i] / bin_tokens;
        b = (b < 0 ? 0 : (b >= n_bins ? n_bins - 1 : b)) - bin0;
        if (b < 0 || b >= nb) continue;
        const uint32_t key = __float_as_uint(alpha[i]);
        const uint32_t prefix = state[(bin0 + b) * 4 + 0], mask = state[(bin0 + b) * 4 + 1];
        if ((key & mask) == prefix) atomicAdd(&s_hist[b * kAccDigits + ((key >> shift) & dmask)], 1);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < nb * kAccDigits; i += kAccThreads)
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
