// decode.cuh -- kernel (c): split-K flash-decode over a page list, plus the log-sum-exp merge.
// SURVEY.md 8(a) a6-a8; PAPER.md:140 (attention over the KV budget B), :131-135 (dense), north_star (c).
//
// Work item = (sequence, kv-head, split): a chunk of `chunk_pages` entries of the page list.  The whole GQA
// group (r <= 8 query heads) is processed together, so each K/V byte is read from HBM once per group.
//
// Data path per warp (each warp owns whole pages and its own online-softmax state, no CTA-wide sync in the
// loop): the 4 KiB K tile and 4 KiB V tile of a page are copied global -> shared with 16-byte cp.async
// (512 contiguous bytes per warp instruction) into a per-warp ring of kStages stages.  Shared layout of a tile:
// [half = dim/64][token 0..15][64 dims = 8 chunks of 16 B], chunk index XOR (token & 7) -- the 128-byte swizzle
// (the same pattern a TMA SWIZZLE_128B box {64 dims, 16 tokens, 2 halves} produces), conflict-free for ldmatrix.
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

constexpr int kDecWarps = 4;
constexpr int kDecThreads = kDecWarps * 32;
constexpr int kDecStages = 3;                                   // per-warp ring depth
constexpr int kStageBytes = 2 * kTileBytes;                     // K tile + V tile = 8 KiB
constexpr int kDecSmemBytes = kDecWarps * kDecStages * kStageBytes;   // 96 KiB -> 2 CTAs / SM
constexpr int kMaxGroup = 8;                                    // r <= 8 (rows 0..7 of the m16 tile)
constexpr int kMaxChunkPages = 32 * kDecWarps;                  // one lane per page of a warp's share

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

template <bool kDense>
__global__ void __launch_bounds__(kDecThreads, 2)
decode_kernel(const uint16_t *__restrict__ q, const uint16_t *__restrict__ k_cache, const uint16_t *__restrict__ v_cache,
              const int32_t *__restrict__ page_table, const int32_t *__restrict__ seq_lens,
              const int32_t *__restrict__ sel_pages, int max_sel, const int32_t *__restrict__ sel_count,
              float *__restrict__ ws_o, float *__restrict__ ws_ml, int chunk_pages, int n_splits_max,
              float scale_log2, int n_q_heads, int n_kv_heads, int max_pages)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    const int split = blockIdx.x, g = blockIdx.y, seq = blockIdx.z;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r = n_q_heads / n_kv_heads;

    const int L = seq_lens[seq];
    const int n_pages = (L + kPage - 1) / kPage;
    int cnt = n_pages;
    if (!kDense) { cnt = sel_count[seq]; cnt = cnt < max_sel ? cnt : max_sel; }
    const int i_begin = split * chunk_pages;
    if (i_begin >= cnt) return;                                   // merge only reads ceil(cnt / chunk) splits
    const int i_end = (i_begin + chunk_pages < cnt) ? i_begin + chunk_pages : cnt;

    // this warp's pages: list entries i_begin + warp + kDecWarps * j; lane j keeps (logical, physical) of page j
    const int n_my = (i_end - i_begin - warp + kDecWarps - 1) / kDecWarps;      // may be <= 0
    int my_logical = 0, my_phys = 0;
    if (lane < n_my) {
        const int i = i_begin + warp + kDecWarps * lane;
        my_logical = kDense ? i : sel_pages[((int64_t)seq * n_kv_heads + g) * max_sel + i];
        my_phys = page_table[(int64_t)seq * max_pages + my_logical];
    }

    // Q fragments: row = lane/4 is the query head inside the group (zero beyond r), 8 k-steps of 16 dims
    uint32_t qa[8][2];
    {
        const int hrow = lane >> 2;
        const uint16_t *qrow = q + ((int64_t)seq * n_q_heads + g * r + hrow) * kDim + 2 * (lane & 3);
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
            qa[kk][0] = hrow < r ? *reinterpret_cast<const uint32_t *>(qrow + kk * 16) : 0u;
            qa[kk][1] = hrow < r ? *reinterpret_cast<const uint32_t *>(qrow + kk * 16 + 8) : 0u;
        }
    }

    uint8_t *ring = smem + warp * (kDecStages * kStageBytes);
    const uint32_t ring_u32 = smem_u32(ring);

    auto issue = [&](int j) {       // copy page j of this warp into stage j % kStages (K then V)
        const int phys = __shfl_sync(0xffffffffu, my_phys, j);
        const uint8_t *ksrc = reinterpret_cast<const uint8_t *>(k_cache + ((int64_t)phys * n_kv_heads + g) * kTileElems);
        const uint8_t *vsrc = reinterpret_cast<const uint8_t *>(v_cache + ((int64_t)phys * n_kv_heads + g) * kTileElems);
        const uint32_t dst = ring_u32 + (j % kDecStages) * kStageBytes;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int idx = i * 32 + lane;                          // 16-byte chunk of the tile, row-major
            const uint32_t off = tile_off(idx >> 4, idx & 15);
            cp_async16(dst + off, ksrc + idx * 16);
            cp_async16(dst + kTileBytes + off, vsrc + idx * 16);
        }
    };

    float o[16][2];                 // O[head = lane/4][dims nt*8 + 2*(lane&3) + {0,1}]
#pragma unroll
    for (int nt = 0; nt < 16; ++nt) { o[nt][0] = 0.f; o[nt][1] = 0.f; }
    float m_run = -INFINITY, l_run = 0.f;

#pragma unroll
    for (int j = 0; j < kDecStages - 1; ++j) {
        if (j < n_my) issue(j);
        cp_async_commit();
    }
    const int mat = lane >> 3, rr = lane & 7;
    for (int j = 0; j < n_my; ++j) {
        __syncwarp();                                                // stage (j-1) % kStages is free again
        if (j + kDecStages - 1 < n_my) issue(j + kDecStages - 1);
        cp_async_commit();
        cp_async_wait<kDecStages - 1>();                             // this lane's copies of page j have landed
        __syncwarp();                                                // ... and so have the other lanes'
        const uint32_t kb = ring_u32 + (j % kDecStages) * kStageBytes;
        const uint32_t vb = kb + kTileBytes;
        const int logical = __shfl_sync(0xffffffffu, my_logical, j);

        // ---- S = Q K^T: two n-tiles (tokens 0-7, 8-15), 8 k-steps ----
        float s0a = 0.f, s0b = 0.f, s1a = 0.f, s1b = 0.f;
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
            uint32_t b0, b1, b2, b3;   // matrices: (tok 0-7, chunk 2kk) (tok 0-7, 2kk+1) (tok 8-15, 2kk) (tok 8-15, 2kk+1)
            ldsm_x4(b0, b1, b2, b3, kb + tile_off((mat >> 1) * 8 + rr, 2 * kk + (mat & 1)));
            mma_rows07(s0a, s0b, qa[kk][0], qa[kk][1], b0, b1);
            mma_rows07(s1a, s1b, qa[kk][0], qa[kk][1], b2, b3);
        }
        // ---- online softmax: this lane holds head lane/4, tokens tq, tq+1, tq+8, tq+9 ----
        const int tq = logical * kPage + 2 * (lane & 3);
        float x0 = tq < L ? s0a * scale_log2 : -INFINITY;
        float x1 = tq + 1 < L ? s0b * scale_log2 : -INFINITY;
        float x2 = tq + 8 < L ? s1a * scale_log2 : -INFINITY;
        float x3 = tq + 9 < L ? s1b * scale_log2 : -INFINITY;
        float mx = fmaxf(fmaxf(x0, x1), fmaxf(x2, x3));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
        mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
        const float m_new = fmaxf(m_run, mx);
        const float m_safe = m_new == -INFINITY ? 0.f : m_new;
        const float alpha = fast_exp2(m_run - m_safe);
        const float p0 = fast_exp2(x0 - m_safe), p1 = fast_exp2(x1 - m_safe);
        const float p2 = fast_exp2(x2 - m_safe), p3 = fast_exp2(x3 - m_safe);
        l_run = l_run * alpha + ((p0 + p1) + (p2 + p3));
        m_run = m_new;
        if (!__all_sync(0xffffffffu, alpha == 1.f)) {
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
    }
    cp_async_wait<0>();
    l_run += __shfl_xor_sync(0xffffffffu, l_run, 1);
    l_run += __shfl_xor_sync(0xffffffffu, l_run, 2);

    // ---- combine the warps of this CTA (each warp parks its state in its own, now idle, ring) ----
    __syncwarp();
    float *st_o = reinterpret_cast<float *>(ring);                    // [kMaxGroup][128]
    float *st_ml = st_o + kMaxGroup * kDim;                           // [kMaxGroup][2]
    {
        const int hrow = lane >> 2;
        if (hrow < r) {
#pragma unroll
            for (int nt = 0; nt < 16; ++nt)
                *reinterpret_cast<float2 *>(st_o + hrow * kDim + nt * 8 + 2 * (lane & 3)) = make_float2(o[nt][0], o[nt][1]);
            if ((lane & 3) == 0) { st_ml[hrow * 2] = m_run; st_ml[hrow * 2 + 1] = l_run; }
        }
    }
    __syncthreads();
    const int64_t part = ((int64_t)seq * n_kv_heads + g) * n_splits_max + split;
    for (int hrow = 0; hrow < r; ++hrow) {
        float mw[kDecWarps], m_star = -INFINITY;
#pragma unroll
        for (int w = 0; w < kDecWarps; ++w) {
            mw[w] = reinterpret_cast<const float *>(smem + w * (kDecStages * kStageBytes))[kMaxGroup * kDim + hrow * 2];
            m_star = fmaxf(m_star, mw[w]);
        }
        float acc = 0.f, l_star = 0.f;
#pragma unroll
        for (int w = 0; w < kDecWarps; ++w) {
            const float *so = reinterpret_cast<const float *>(smem + w * (kDecStages * kStageBytes));
            const float wgt = mw[w] == -INFINITY ? 0.f : fast_exp2(mw[w] - m_star);
            acc = fmaf(so[hrow * kDim + tid], wgt, acc);
            l_star = fmaf(so[kMaxGroup * kDim + hrow * 2 + 1], wgt, l_star);
        }
        ws_o[(part * r + hrow) * kDim + tid] = acc;                   // un-normalised partial (a6)
        if (tid == 0) { ws_ml[(part * r + hrow) * 2] = m_star; ws_ml[(part * r + hrow) * 2 + 1] = l_star; }
    }
}

// a7: log-sum-exp merge of the splits of one (sequence, query head); thread = output channel.
template <bool kDense>
__global__ void __launch_bounds__(kDim)
merge_kernel(const float *__restrict__ ws_o, const float *__restrict__ ws_ml, const int32_t *__restrict__ seq_lens,
             const int32_t *__restrict__ sel_count, int max_sel, uint16_t *__restrict__ out, float *__restrict__ lse,
             int chunk_pages, int n_splits_max, int n_q_heads, int n_kv_heads)
{
    const int h = blockIdx.x, seq = blockIdx.y, d = threadIdx.x;
    const int r = n_q_heads / n_kv_heads;
    const int g = h / r, hrow = h % r;
    int cnt;
    if (kDense) cnt = (seq_lens[seq] + kPage - 1) / kPage;
    else { cnt = sel_count[seq]; cnt = cnt < max_sel ? cnt : max_sel; }
    const int n_splits = (cnt + chunk_pages - 1) / chunk_pages;
    const int64_t part0 = ((int64_t)seq * n_kv_heads + g) * n_splits_max;

    float m_star = -INFINITY;
    for (int s = 0; s < n_splits; ++s) {
        const float m = ws_ml[((part0 + s) * r + hrow) * 2];
        const float l = ws_ml[((part0 + s) * r + hrow) * 2 + 1];
        if (l > 0.f) m_star = fmaxf(m_star, m);
    }
    float acc = 0.f, l_star = 0.f;
    for (int s = 0; s < n_splits; ++s) {
        const float m = ws_ml[((part0 + s) * r + hrow) * 2];
        const float l = ws_ml[((part0 + s) * r + hrow) * 2 + 1];
        if (!(l > 0.f)) continue;                                      // empty partial: skip, never NaN
        const float wgt = fast_exp2(m - m_star);
        acc = fmaf(ws_o[((part0 + s) * r + hrow) * kDim + d], wgt, acc);
        l_star = fmaf(l, wgt, l_star);
    }
    const float res = l_star > 0.f ? acc / l_star : 0.f;
    __nv_bfloat16 b = __float2bfloat16_rn(res);
    out[((int64_t)seq * n_q_heads + h) * kDim + d] = *reinterpret_cast<uint16_t *>(&b);
    if (lse && d == 0)
        lse[(int64_t)seq * n_q_heads + h] = l_star > 0.f ? (m_star + log2f(l_star)) * 0.6931471805599453f : -INFINITY;
}

}  // namespace sparrow
