// summarize.cuh -- kernel (a): page summaries = per-channel min/max of K over a page's valid tokens.
// SURVEY.md 8(a) a1; "landmark" PAPER.md:147; north_star (a).  HBM-bound: reads 4 KiB, writes 512 B per
// (page, kv-head).  One warp per (page, kv-head) tile; a half-warp covers one 256-byte key row with
// 16-byte loads, so every load instruction reads two whole rows (512 contiguous bytes).
#pragma once
#include "common.cuh"

namespace sparrow {

constexpr int kSumWarps = 8;

__device__ __forceinline__ uint32_t bf2_min(uint32_t a, uint32_t b)
{
    __nv_bfloat162 r = __hmin2(*reinterpret_cast<__nv_bfloat162 *>(&a), *reinterpret_cast<__nv_bfloat162 *>(&b));
    return *reinterpret_cast<uint32_t *>(&r);
}
__device__ __forceinline__ uint32_t bf2_max(uint32_t a, uint32_t b)
{
    __nv_bfloat162 r = __hmax2(*reinterpret_cast<__nv_bfloat162 *>(&a), *reinterpret_cast<__nv_bfloat162 *>(&b));
    return *reinterpret_cast<uint32_t *>(&r);
}

__global__ void __launch_bounds__(kSumWarps * 32)
summarize_kernel(const uint16_t *__restrict__ k_cache, uint16_t *__restrict__ summaries,
                 const int32_t *__restrict__ page_ids, const int32_t *__restrict__ n_valid,
                 int64_t n_update, int n_kv_heads, int page_tokens, const KvLayout kv)
{
    chain_entry();
    const int lane = threadIdx.x & 31;
    const int64_t tile = (int64_t)blockIdx.x * kSumWarps + (threadIdx.x >> 5);   // (update, kv-head)
    if (tile >= n_update * n_kv_heads) return;
    const int64_t u = tile / n_kv_heads;
    const int g = (int)(tile % n_kv_heads);
    const int64_t page = page_ids ? (int64_t)page_ids[u] : u;
    int valid = n_valid ? n_valid[u] : page_tokens;
    valid = valid < 0 ? 0 : (valid > page_tokens ? page_tokens : valid);

    const uint16_t *src = k_cache + page * kv.page + g * kv.head;     // page_tokens rows of 256 B, kv.tok elements apart
    const int half = lane >> 4;       // which of the two rows of this load
    const int c = lane & 15;          // 16-byte chunk (8 channels) of the row

    // +inf / -inf in both bf16 lanes: identity of min / max (a page with valid == 0 keeps them)
    uint32_t mn[4] = {0x7f807f80u, 0x7f807f80u, 0x7f807f80u, 0x7f807f80u};
    uint32_t mx[4] = {0xff80ff80u, 0xff80ff80u, 0xff80ff80u, 0xff80ff80u};
    for (int t0 = 0; t0 < valid; t0 += kPage) {      // one 16-token tile (4 KiB) at a time
        uint4 v[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) {     // all loads first (8 x 16 B in flight per lane)
            const int t = t0 + 2 * i + half;
            if (t < valid) v[i] = ldg_stream16(src + t * kv.tok + c * 8);
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int t = t0 + 2 * i + half;
            if (t < valid) {
                mn[0] = bf2_min(mn[0], v[i].x); mx[0] = bf2_max(mx[0], v[i].x);
                mn[1] = bf2_min(mn[1], v[i].y); mx[1] = bf2_max(mx[1], v[i].y);
                mn[2] = bf2_min(mn[2], v[i].z); mx[2] = bf2_max(mx[2], v[i].z);
                mn[3] = bf2_min(mn[3], v[i].w); mx[3] = bf2_max(mx[3], v[i].w);
            }
        }
    }
#pragma unroll
    for (int j = 0; j < 4; ++j) {     // combine even and odd rows
        mn[j] = bf2_min(mn[j], __shfl_xor_sync(0xffffffffu, mn[j], 16));
        mx[j] = bf2_max(mx[j], __shfl_xor_sync(0xffffffffu, mx[j], 16));
    }
    // lanes 0-15 store min (256 B), lanes 16-31 store max (256 B): one contiguous 512-byte summary
    uint16_t *dst = summaries + (page * n_kv_heads + g) * (int64_t)kSumElems + half * kDim + c * 8;
    uint4 o = half ? make_uint4(mx[0], mx[1], mx[2], mx[3]) : make_uint4(mn[0], mn[1], mn[2], mn[3]);
    *reinterpret_cast<uint4 *>(dst) = o;
}

// Mean-key landmark (the single vector per page of the paper's cost model): mean[d] = (sum over the
// page's valid tokens of K[t][d]) / valid, accumulated in fp32 (token order) and rounded to bf16 once (nearest even).
// The definition is the exact mean rounded once (reading R24); the fp32 sum is within (valid + 1) 2^-24 mean|k| of it,
// so the stored code is that one or, next to a rounding boundary, its neighbour -- the checker's validity band.
// One warp per (page, kv-head); lane = 4 channels (8 bytes), so a row is one coalesced 256-byte load.
__device__ __forceinline__ void mean_of_page(const uint16_t *__restrict__ src, int64_t row_stride, int valid, int lane,
                                             uint16_t *__restrict__ dst, bool coherent)
{
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    for (int t0 = 0; t0 < valid; t0 += kPage) {
        uint2 v[kPage];
#pragma unroll
        for (int i = 0; i < kPage; ++i) {                // all loads of the tile first
            const uint2 *p = reinterpret_cast<const uint2 *>(src + (t0 + i) * row_stride + lane * 4);
            if (t0 + i < valid) v[i] = coherent ? __ldcg(p) : __ldg(p);
        }
#pragma unroll
        for (int i = 0; i < kPage; ++i) {                // then the adds, in token order
            if (t0 + i < valid) {
                acc[0] += bf16_lo(v[i].x); acc[1] += bf16_hi(v[i].x);
                acc[2] += bf16_lo(v[i].y); acc[3] += bf16_hi(v[i].y);
            }
        }
    }
    const float n = valid > 0 ? (float)valid : 1.f;
    __nv_bfloat162 lo = __floats2bfloat162_rn(acc[0] / n, acc[1] / n), hi = __floats2bfloat162_rn(acc[2] / n, acc[3] / n);
    uint2 o;
    o.x = *reinterpret_cast<uint32_t *>(&lo);
    o.y = *reinterpret_cast<uint32_t *>(&hi);
    *reinterpret_cast<uint2 *>(dst + lane * 4) = o;
}

__global__ void __launch_bounds__(kSumWarps * 32)
summarize_mean_kernel(const uint16_t *__restrict__ k_cache, uint16_t *__restrict__ summaries,
                      const int32_t *__restrict__ page_ids, const int32_t *__restrict__ n_valid,
                      int64_t n_update, int n_kv_heads, int page_tokens, const KvLayout kv)
{
    chain_entry();
    const int lane = threadIdx.x & 31;
    const int64_t tile = (int64_t)blockIdx.x * kSumWarps + (threadIdx.x >> 5);   // (update, kv-head)
    if (tile >= n_update * n_kv_heads) return;
    const int64_t u = tile / n_kv_heads;
    const int g = (int)(tile % n_kv_heads);
    const int64_t page = page_ids ? (int64_t)page_ids[u] : u;
    int valid = n_valid ? n_valid[u] : page_tokens;
    valid = valid < 0 ? 0 : (valid > page_tokens ? page_tokens : valid);
    mean_of_page(k_cache + page * kv.page + g * kv.head, kv.tok, valid, lane, summaries + (page * n_kv_heads + g) * (int64_t)kDim, false);
}

}  // namespace sparrow
