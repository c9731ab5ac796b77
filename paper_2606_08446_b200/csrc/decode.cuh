// decode.cuh -- kernel (c): split-K flash-decode over a page list with the log-sum-exp merge fused in.
// SURVEY.md 8(a) a6-a8; PAPER.md:140 (attention over the KV budget B), :131-135 (dense), north_star (c).
//
// Work decomposition ("stream-K" over pages): the (page, kv-head) tiles of the whole batch form ONE flat stream,
// ordered (sequence, kv-head, list position); its length T = Hkv * sum_i cnt_i is known from sel_count (or from
// seq_lens for the dense entry).  The stream is cut into W equal contiguous ranges, W = warps of a persistent
// grid of one CTA per SM, and every warp streams exactly its range: the HBM stream is balanced to within one tile
// whatever the mix of lengths and budgets, there is no tail wave, and per-unit fixed costs (query fragments, list
// and page-table look-ups) are prefetched behind the running K/V stream instead of sitting in front of it.
// A range that crosses a (sequence, kv-head) boundary simply closes one softmax state and opens the next.
// The whole GQA group (r <= 8 query heads) is processed together, so each K/V byte is read from HBM once.
//
// Split-K merge (a7): a (sequence, kv-head) unit covered by one range is normalised and written straight to `out`;
// otherwise each covering warp parks its un-normalised (o, m, l) in slot unit + warp of a small fp32 workspace
// (unit + warp is strictly increasing along the stream, hence unique) and bumps the unit's counter; the warp
// that arrives last merges the slots in stream order (deterministic) and writes `out` / `lse`.  No second launch.
//
// Data path per warp: the 4 KiB K tile and 4 KiB V tile of a page are copied global -> shared with 16-byte cp.async
// (512 contiguous bytes per warp instruction) into a per-warp ring of kDecStages stages.  Shared layout of a tile:
// [half = dim/64][token 0..15][64 dims = 8 chunks of 16 B], chunk index XOR (token & 7) -- the 128-byte swizzle,
// conflict-free for ldmatrix.
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

constexpr int kDecWarps = 8;
constexpr int kDecThreads = kDecWarps * 32;
constexpr int kDecStages = 3;                                   // per-warp ring depth
constexpr int kStageBytes = 2 * kTileBytes;                     // K tile + V tile = 8 KiB
constexpr int kDecRingBytes = kDecWarps * kDecStages * kStageBytes;   // 192 KiB -> one CTA per SM
constexpr int kMaxGroup = 8;                                    // r <= 8 (rows 0..7 of the m16 tile)
constexpr int kDecMaxSeq = 8192;                                // prefix table of the batch lives in shared memory
constexpr int kDecMinRange = 4;                                 // tiles per warp at least (bounds the number of partials)
constexpr int kDecGrid = 148;                                   // persistent: one CTA per B200 SM

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

constexpr int kMetaFirst = 1 << 8, kMetaLast = 1 << 9;

// Tiles per range for a stream of T tiles cut for W warps.
__host__ __device__ inline int decode_range_tiles(int T, int W)
{
    const int rr = (T + W - 1) / W;
    return rr < kDecMinRange ? kDecMinRange : rr;
}

template <bool kDense>
__global__ void __launch_bounds__(kDecThreads, 1)
decode_kernel(const uint16_t *__restrict__ q, const uint16_t *__restrict__ k_cache, const uint16_t *__restrict__ v_cache,
              const int32_t *__restrict__ page_table, const int32_t *__restrict__ seq_lens,
              const int32_t *__restrict__ sel_pages, int max_sel, const int32_t *__restrict__ sel_count,
              float *__restrict__ ws_o, float *__restrict__ ws_ml, int32_t *__restrict__ counters,
              uint16_t *__restrict__ out, float *__restrict__ lse,
              float scale_log2, int n_seq, int n_q_heads, int n_kv_heads, int max_pages)
{
    extern __shared__ __align__(1024) uint8_t smem[];
    int32_t *s_prefix = reinterpret_cast<int32_t *>(smem + kDecRingBytes);     // [n_seq + 1] list entries before sequence i
    __shared__ int s_scan[kDecWarps];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int r = n_q_heads / n_kv_heads;

    // ---- prologue: list length of every sequence -> exclusive prefix in shared memory ----
    {
        const int per = (n_seq + kDecThreads - 1) / kDecThreads;
        const int s0 = min(tid * per, n_seq), s1 = min(s0 + per, n_seq);
        auto count_of = [&](int s) {
            int c;
            if (kDense) c = (__ldg(seq_lens + s) + kPage - 1) / kPage;
            else { c = __ldg(sel_count + s); c = c < max_sel ? c : max_sel; }
            return c > 0 ? c : 0;
        };
        int sum = 0;
        for (int s = s0; s < s1; ++s) sum += count_of(s);
        int inc = sum;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, inc, o);
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
    const int R = decode_range_tiles(T, gridDim.x * kDecWarps);
    const int gw = blockIdx.x * kDecWarps + warp;
    const int a = gw * R;                                        // this warp streams tiles [a, b)
    if (a >= T) return;                                          // (no CTA-wide barrier below this line)
    const int b = min(a + R, T);
    const int n = b - a;

    // Look-up of flat tile p -> (sequence, kv-head, list position) -> logical page -> physical tile, as three stages
    // so that no stage consumes a load issued by the stage before it in the same breath: the warp never stalls on
    // the chain while its K/V ring is running (the stages of window w + 1 run at tiles 0, 8 and 16 of window w).
    struct Lookup {
        int tile;        // stage C: physical page * Hkv + kv-head = index of the 4 KiB K (and V) tile
        int unit;        // stage A: sequence * Hkv + kv-head
        int info;        // stage A: bit 8 first tile of a segment, bit 9 last; stage B adds bits 0-4 = valid tokens
        int seq, logical, len, phys;
    };
    auto stage_a = [&](Lookup &m, int p) {
        m.tile = 0; m.unit = 0; m.info = 0; m.seq = -1; m.logical = 0; m.len = 0; m.phys = 0;
        if (p < b) {
            int lo = 0, hi = n_seq - 1;                          // last sequence whose first tile is <= p ...
            while (lo < hi) {
                const int mid = (lo + hi + 1) >> 1;
                if (s_prefix[mid] * n_kv_heads <= p) lo = mid; else hi = mid - 1;
            }
            while (s_prefix[lo + 1] * n_kv_heads <= p) ++lo;     // ... that is not empty (empty lists share a prefix)
            const int seq = lo, base = s_prefix[seq], c = s_prefix[seq + 1] - base;
            const int rem = p - base * n_kv_heads;
            const int g = rem / c, i = rem - g * c;
            m.seq = seq;
            m.unit = seq * n_kv_heads + g;
            m.info = ((i == 0 || p == a) ? kMetaFirst : 0) | ((i == c - 1 || p == b - 1) ? kMetaLast : 0);
            m.logical = kDense ? i : __ldg(sel_pages + ((int64_t)m.unit) * max_sel + i);
            m.len = __ldg(seq_lens + seq);
        }
    };
    auto stage_b = [&](Lookup &m) {
        if (m.seq >= 0) {
            m.phys = __ldg(page_table + (int64_t)m.seq * max_pages + m.logical);
            int valid = m.len - m.logical * kPage;
            valid = valid < 0 ? 0 : (valid > kPage ? kPage : valid);
            m.info |= valid;
        }
    };
    auto stage_c = [&](Lookup &m) { m.tile = m.phys * n_kv_heads + (m.unit - m.seq * n_kv_heads); };

    const int hrow = lane >> 2, col = 2 * (lane & 3);               // this lane's query head and column pair
    uint32_t qa[8][2];                                              // Q fragments of the current unit
    auto load_q = [&](int unit) {
        const uint16_t *qrow = q + ((int64_t)unit * r + hrow) * kDim + col;
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
            qa[kk][0] = hrow < r ? __ldg(reinterpret_cast<const uint32_t *>(qrow + kk * 16)) : 0u;
            qa[kk][1] = hrow < r ? __ldg(reinterpret_cast<const uint32_t *>(qrow + kk * 16 + 8)) : 0u;
        }
    };

    Lookup cur, nxt;
    stage_a(cur, a + lane);
    int q_unit = __shfl_sync(0xffffffffu, cur.unit, 0);
    load_q(q_unit);                                                 // in flight while the look-up chain completes
    stage_a(nxt, a + 32 + lane);
    stage_b(cur);
    stage_c(cur);

    const uint32_t ring_u32 = smem_u32(smem + warp * (kDecStages * kStageBytes));
    auto issue = [&](int tile, int stage) {       // copy one K tile and one V tile into a ring stage
        const uint8_t *ksrc = reinterpret_cast<const uint8_t *>(k_cache + (int64_t)tile * kTileElems);
        const uint8_t *vsrc = reinterpret_cast<const uint8_t *>(v_cache + (int64_t)tile * kTileElems);
        const uint32_t dst = ring_u32 + stage * kStageBytes;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int idx = i * 32 + lane;                          // 16-byte chunk of the tile, row-major
            const uint32_t off = tile_off(idx >> 4, idx & 15);
            cp_async16(dst + off, ksrc + idx * 16);
            cp_async16(dst + kTileBytes + off, vsrc + idx * 16);
        }
    };

    float o[16][2];                 // O[head = lane/4][dims nt*8 + col + {0,1}]
    float m_run = -INFINITY, l_run = 0.f;

#pragma unroll
    for (int j = 0; j < kDecStages - 1; ++j) {
        const int tile = __shfl_sync(0xffffffffu, cur.tile, j);
        if (j < n) issue(tile, j);
        cp_async_commit();
    }
    const int mat = lane >> 3, rr = lane & 7;
    int stage = 0;                                                  // j % kDecStages
#pragma unroll 1
    for (int j = 0; j < n; ++j) {
        const int jl = j & 31;
        if (jl == 0 && j > 0) {                                     // window turn
            cur = nxt;
            stage_a(nxt, a + j + 32 + lane);
        } else if (jl == 8) stage_b(nxt);
        else if (jl == 16) stage_c(nxt);
        __syncwarp();                                               // stage (j-1) % kStages is free again
        {
            const int jj = j + kDecStages - 1;
            const int t_cur = __shfl_sync(0xffffffffu, cur.tile, jj & 31);
            const int t_nxt = __shfl_sync(0xffffffffu, nxt.tile, jj & 31);
            int st2 = stage + kDecStages - 1;
            st2 = st2 >= kDecStages ? st2 - kDecStages : st2;
            if (jj < n) issue((jj >> 5) == (j >> 5) ? t_cur : t_nxt, st2);
            cp_async_commit();
        }
        const int info = __shfl_sync(0xffffffffu, cur.info, jl);
        const int unit = __shfl_sync(0xffffffffu, cur.unit, jl);
        if (info & kMetaFirst) {                                    // warp-uniform: a new softmax state opens
#pragma unroll
            for (int nt = 0; nt < 16; ++nt) { o[nt][0] = 0.f; o[nt][1] = 0.f; }
            m_run = -INFINITY; l_run = 0.f;
            if (unit != q_unit) {
                q_unit = unit;
                load_q(unit);
            }
        }
        cp_async_wait<kDecStages - 1>();                             // this lane's copies of tile j have landed
        __syncwarp();                                                // ... and so have the other lanes'
        const uint32_t kb = ring_u32 + stage * kStageBytes;
        const uint32_t vb = kb + kTileBytes;
        stage = stage + 1 == kDecStages ? 0 : stage + 1;

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
        const int valid = info & 31;
        float x0 = col < valid ? s0a * scale_log2 : -INFINITY;
        float x1 = col + 1 < valid ? s0b * scale_log2 : -INFINITY;
        float x2 = col + 8 < valid ? s1a * scale_log2 : -INFINITY;
        float x3 = col + 9 < valid ? s1b * scale_log2 : -INFINITY;
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

        if (!(info & kMetaLast)) continue;
        // ---- the segment of `unit` inside this range is complete: write it out (a7) ----
        float l_tot = l_run;
        l_tot += __shfl_xor_sync(0xffffffffu, l_tot, 1);
        l_tot += __shfl_xor_sync(0xffffffffu, l_tot, 2);
        const int seq = unit / n_kv_heads, g = unit - seq * n_kv_heads;
        const int base = s_prefix[seq], c = s_prefix[seq + 1] - base;
        const int u0 = base * n_kv_heads + g * c;                    // the unit's tiles are [u0, u0 + c) of the stream
        const int w0 = u0 / R, w1 = (u0 + c - 1) / R;                // ranges (warps) that cover it
        constexpr float kLn2 = 0.6931471805599453f;
        if (w0 == w1) {                                              // covered by this warp alone: final result
            if (hrow < r) {
                const float inv = l_tot > 0.f ? 1.f / l_tot : 0.f;
                uint32_t *dst = reinterpret_cast<uint32_t *>(out + ((int64_t)unit * r + hrow) * kDim + col);
#pragma unroll
                for (int nt = 0; nt < 16; ++nt) dst[nt * 4] = pack_bf16(o[nt][0] * inv, o[nt][1] * inv);
                if (lse && (lane & 3) == 0)
                    lse[(int64_t)unit * r + hrow] = l_tot > 0.f ? (m_run + log2f(l_tot)) * kLn2 : -INFINITY;
            }
            continue;
        }
        {
            const int64_t slot = (int64_t)unit + gw;                 // unique: unit + warp increases along the stream
            if (hrow < r) {
                float *po = ws_o + (slot * r + hrow) * kDim + col;
#pragma unroll
                for (int nt = 0; nt < 16; ++nt) *reinterpret_cast<float2 *>(po + nt * 8) = make_float2(o[nt][0], o[nt][1]);
                if ((lane & 3) == 0) *reinterpret_cast<float2 *>(ws_ml + (slot * r + hrow) * 2) = make_float2(m_run, l_tot);
            }
        }
        __threadfence();
        __syncwarp();
        int old = 0;
        if (lane == 0) old = atomicAdd(counters + unit, 1);
        old = __shfl_sync(0xffffffffu, old, 0);
        if (old != w1 - w0) continue;                                // not the last segment to arrive
        if (lane == 0) counters[unit] = 0;                           // restore the zero for the next call
        __threadfence();
        for (int h = 0; h < r; ++h) {                                // lane = 4 output channels
            float m_star = -INFINITY;
            for (int w = w0; w <= w1; ++w) {
                const float2 ml = __ldcg(reinterpret_cast<const float2 *>(ws_ml + (((int64_t)unit + w) * r + h) * 2));
                if (ml.y > 0.f) m_star = fmaxf(m_star, ml.x);
            }
            float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
            float l_star = 0.f;
            for (int w = w0; w <= w1; ++w) {
                const int64_t row = ((int64_t)unit + w) * r + h;
                const float2 ml = __ldcg(reinterpret_cast<const float2 *>(ws_ml + row * 2));
                if (!(ml.y > 0.f)) continue;                         // empty partial: skip, never NaN
                const float wgt = fast_exp2(ml.x - m_star);
                const float4 v = __ldcg(reinterpret_cast<const float4 *>(ws_o + row * kDim + lane * 4));
                acc.x = fmaf(v.x, wgt, acc.x); acc.y = fmaf(v.y, wgt, acc.y);
                acc.z = fmaf(v.z, wgt, acc.z); acc.w = fmaf(v.w, wgt, acc.w);
                l_star = fmaf(ml.y, wgt, l_star);
            }
            const float inv = l_star > 0.f ? 1.f / l_star : 0.f;
            uint2 pk;
            pk.x = pack_bf16(acc.x * inv, acc.y * inv);
            pk.y = pack_bf16(acc.z * inv, acc.w * inv);
            *reinterpret_cast<uint2 *>(out + ((int64_t)unit * r + h) * kDim + lane * 4) = pk;
            if (lse && lane == 0)
                lse[(int64_t)unit * r + h] = l_star > 0.f ? (m_star + log2f(l_star)) * kLn2 : -INFINITY;
        }
    }
    cp_async_wait<0>();
}

}  // namespace sparrow
