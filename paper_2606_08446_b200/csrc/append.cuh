// append.cuh -- decode-step cache update with summarize-on-fill (a1 on page fill, north_star (a)).
// The rollout loop (per generated token, landmark scores -> Top-k -> attention over the budget;
// :109-119: the budget follows the growing length) needs, per step and sequence: the new token's K/V rows written at
// position L of the paged cache, L <- L + 1, and -- when that token fills its page -- the page's min/max summary.
// One CTA per sequence, one warp per kv-head: the warp stores the two 256-byte rows, and if the page is now full it
// reads the page's 16 key rows back (15 from HBM/L2, its own from the store just made) and writes the 512-byte
// summary, exactly as summarize_kernel does.  All warps read L before any of them writes L + 1.
#pragma once
#include "summarize.cuh"

namespace sparrow {

constexpr int kAppendMaxWarps = 8;                 // warps per CTA; more kv-heads than that are looped over

__global__ void __launch_bounds__(kAppendMaxWarps * 32)
append_kernel(const uint16_t *__restrict__ k_new, const uint16_t *__restrict__ v_new, uint16_t *__restrict__ k_cache,
              uint16_t *__restrict__ v_cache, uint16_t *__restrict__ summaries, const int32_t *__restrict__ page_table,
              int32_t *__restrict__ seq_lens, int n_kv_heads, int max_pages, int page_tokens, int landmark, const KvLayout kv)
{
    chain_entry();
    const int seq = blockIdx.x, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int L = seq_lens[seq];                         // tokens cached before this step
    __syncthreads();                                     // every warp has read L
    const int page_l = L / page_tokens, row = L - page_l * page_tokens;
    if (L < 0 || page_l >= max_pages) return;            // no room in the page table: the call leaves the sequence alone
    if (threadIdx.x == 0) seq_lens[seq] = L + 1;
    const int64_t page = page_table[(int64_t)seq * max_pages + page_l];
    for (int g = warp; g < n_kv_heads; g += blockDim.x >> 5) {
        const int64_t tile = page * kv.page + g * kv.head;                               // the page's rows, 256 B each, kv.tok elements apart
        const int64_t src = ((int64_t)seq * n_kv_heads + g) * kDim;
        // 256-byte row = 16 lanes x 16 B: lanes 0-15 copy K, lanes 16-31 copy V
        const int c = lane & 15;
        const uint4 val = *reinterpret_cast<const uint4 *>((lane < 16 ? k_new : v_new) + src + c * 8);
        *reinterpret_cast<uint4 *>((lane < 16 ? k_cache : v_cache) + tile + row * kv.tok + c * 8) = val;
        if (row != page_tokens - 1) continue;            // the page is not full yet
        __syncwarp();                                    // the new key row is visible to the whole warp
        if (landmark == SPARROW_LANDMARK_MEAN) {         // mean-key landmark: same device function as summarize_mean_kernel
            mean_of_page(k_cache + tile, kv.tok, page_tokens, lane, summaries + (page * n_kv_heads + g) * (int64_t)kDim, true);
            continue;
        }
        const int half = lane >> 4;
        uint32_t mn[4] = {0x7f807f80u, 0x7f807f80u, 0x7f807f80u, 0x7f807f80u};
        uint32_t mx[4] = {0xff80ff80u, 0xff80ff80u, 0xff80ff80u, 0xff80ff80u};
        for (int t0 = 0; t0 < page_tokens; t0 += kPage) {
            uint4 v[8];
#pragma unroll
            for (int i = 0; i < 8; ++i)                  // rows t0 + 2i + half; coherent loads (the last row was just written)
                v[i] = __ldcg(reinterpret_cast<const uint4 *>(k_cache + tile + (t0 + 2 * i + half) * kv.tok + c * 8));
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                mn[0] = bf2_min(mn[0], v[i].x); mx[0] = bf2_max(mx[0], v[i].x);
                mn[1] = bf2_min(mn[1], v[i].y); mx[1] = bf2_max(mx[1], v[i].y);
                mn[2] = bf2_min(mn[2], v[i].z); mx[2] = bf2_max(mx[2], v[i].z);
                mn[3] = bf2_min(mn[3], v[i].w); mx[3] = bf2_max(mx[3], v[i].w);
            }
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            mn[j] = bf2_min(mn[j], __shfl_xor_sync(0xffffffffu, mn[j], 16));
            mx[j] = bf2_max(mx[j], __shfl_xor_sync(0xffffffffu, mx[j], 16));
        }
        uint16_t *dst = summaries + (page * n_kv_heads + g) * (int64_t)kSumElems + half * kDim + c * 8;
        *reinterpret_cast<uint4 *>(dst) = half ? make_uint4(mx[0], mx[1], mx[2], mx[3]) : make_uint4(mn[0], mn[1], mn[2], mn[3]);
    }
}

}  // namespace sparrow
