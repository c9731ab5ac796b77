// common.cuh -- shared device/host helpers of libsparrow_b200 (sm_100a only).
// Schedule arithmetic (a2, a3 of SURVEY.md 8(a); readings R2-R9, R13 of DESIGN.md) is written here once for the
// library (host helpers and kernels both use it); the CPU oracle has its own, independent statement.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/sparrow.h"

namespace sparrow {

constexpr int kPage = 16;          // tokens per TILE = the paper's page size; a larger page (32, 64, 128
                                   // tokens: Table 4) is 2, 4 or 8 consecutive 16-token tiles
constexpr int kDim = 128;          // head dim
constexpr int kTileElems = kPage * kDim;        // one (page, kv-head) K or V tile: 2048 bf16 = 4 KiB
constexpr int kTileBytes = kTileElems * 2;
constexpr int kSumElems = 2 * kDim;             // one (page, kv-head) summary: min[128] + max[128] = 512 B

// Strides of the K and V pools in elements (sparrow_shape_t kv_stride_*; the head dim is always contiguous): row t of the
// (page, kv-head) tile is at page * .page + head * .head + t * .tok.  Packed HND (the default): tok = 128, head = P * 128,
// page = Hkv * P * 128 -- a tile is 4 KiB contiguous.  NHD (vLLM / FlashInfer's default): head = 128, tok = Hkv * 128.
struct KvLayout {
    int64_t page, head, tok;
};

// Schedule passed to kernels by value (no device memory, graph-capturable).
struct SchedDev {
    int32_t kind, sink_tokens, local_tokens, table_len, bin_tokens;
    int32_t page;                // tokens per page: 16, 32, 64 or 128
    int32_t page_log2;           // its log2: every division by the page size in the plan is a shift
    int64_t fixed_tokens, floor_tokens, f0_ppm, f1_ppm, L0, L1;
    double inv_den;              // LINEAR_FRAC: 1.0 / (1e6 * (L1 - L0)), the quotient estimate's multiplier
    int32_t table[SPARROW_MAX_TABLE_BINS];
};

__host__ __device__ inline int64_t ceil_div64(int64_t a, int64_t b) { return (a + b - 1) / b; }

// floor(a * b / c) for a, b >= 0, c > 0, exact; inv_c = 1.0 / c rounded to fp64 (the host puts it in SchedDev).
// A 128-bit (or even 64-bit) division is hundreds of instructions on the GPU and sits on every CTA's critical path,
// so the quotient is estimated with two fp64 multiplies (off by a unit or two at most while it is below 2^50) and
// then fixed with the exact remainder a*b - q*c, which is tiny and therefore survives 64-bit wrap-around
// arithmetic.  Larger quotients (possible only for host callers: device lengths are int32) take the plain
// 128-bit division.
__host__ __device__ inline int64_t muldiv_floor(int64_t a, int64_t b, int64_t c, double inv_c)
{
    const double est = (double)a * (double)b * inv_c;
#ifndef __CUDA_ARCH__
    if (!(est < 1125899906842624.0)) return (int64_t)(((__int128)a * b) / c);
#endif
    int64_t qv = (int64_t)est;
    int64_t rem = (int64_t)((uint64_t)a * (uint64_t)b - (uint64_t)qv * (uint64_t)c);
    while (rem < 0) { --qv; rem += c; }
    while (rem >= c) { ++qv; rem -= c; }
    return qv;
}

// a2: B(L) in tokens, exact integers (R3).
__host__ __device__ inline int64_t budget_tokens(const SchedDev &s, int64_t L)
{
    int64_t B;
    switch (s.kind) {
    case SPARROW_SCHED_DENSE: B = L; break;
    case SPARROW_SCHED_FIXED: B = s.fixed_tokens; break;
    case SPARROW_SCHED_CLAMP_FRAC:
        B = muldiv_floor(L, s.f0_ppm, 1000000, 1.0e-6);
        if (B < s.floor_tokens) B = s.floor_tokens;
        break;
    case SPARROW_SCHED_LINEAR_FRAC: {
        int64_t Lc = L < s.L0 ? s.L0 : (L > s.L1 ? s.L1 : L);
        int64_t span = s.L1 - s.L0;
        // validated on entry: 0 <= f <= 1e6 ppm and span < 2^31, so num and den stay below 2^51
        const int64_t num = s.f0_ppm * span - (s.f0_ppm - s.f1_ppm) * (Lc - s.L0);
        const int64_t den = 1000000 * span;
        B = muldiv_floor(L, num, den, s.inv_den);
        if (B < s.floor_tokens) B = s.floor_tokens;
        break;
    }
    default: {  // TABLE: pages per length bin, B = pagesize x num_pages
#ifdef __CUDA_ARCH__
        int64_t b = L > 0 ? (int64_t)((uint32_t)(L - 1) / (uint32_t)s.bin_tokens) : 0;   // device lengths are int32
#else
        int64_t b = (L - 1) / s.bin_tokens;
#endif
        if (b < 0) b = 0;
        if (b >= s.table_len) b = s.table_len - 1;
        B = (int64_t)s.table[b] * s.page;
        break;
    }
    }
    return B > L ? L : B;
}

// Everything the selector needs to know about one sequence (a2 + a3).
struct SeqPlan {
    int32_t L, n_pages, k_pages;
    int32_t n_sink;      // sink pages are [0, n_sink)
    int32_t tail0;       // local-window pages + last page are [tail0, n_pages)
    int32_t n_forced;    // |F|
    int32_t k;           // candidates to pick = max(0, K_pages - |F|)   (R2)
    int32_t count;       // pages attended = n_pages if dense else max(K_pages, |F|)
    bool dense;          // K_pages >= n_pages (R13)
    __host__ __device__ bool forced(int p) const { return p < n_sink || p >= tail0; }
};

__host__ __device__ inline SeqPlan make_plan(const SchedDev &s, int64_t L)
{
    SeqPlan pl;
    pl.L = (int32_t)L;
    const int sh = s.page_log2;
    const int64_t pm = s.page - 1;
    pl.n_pages = (int32_t)((L + pm) >> sh);
    int64_t kp = (budget_tokens(s, L) + pm) >> sh;                       // R4: ceil
    pl.k_pages = (int32_t)(kp < pl.n_pages ? kp : pl.n_pages);
    int32_t ns = (int32_t)((s.sink_tokens + pm) >> sh);                  // R8
    pl.n_sink = ns < pl.n_pages ? ns : pl.n_pages;
    int32_t t0 = pl.n_pages - 1;                                         // last page always kept (R9)
    if (s.local_tokens > 0) {
        int64_t lo = L - s.local_tokens;
        if (lo < 0) lo = 0;
        int32_t fl = (int32_t)(lo >> sh);                                // R7: every page overlapping the window
        if (fl < t0) t0 = fl;
    }
    if (t0 < 0) t0 = 0;
    pl.tail0 = t0;
    int32_t tail_from = t0 > pl.n_sink ? t0 : pl.n_sink;
    pl.n_forced = pl.n_sink + (pl.n_pages - tail_from);
    pl.dense = pl.k_pages >= pl.n_pages;
    int32_t k = pl.k_pages - pl.n_forced;
    pl.k = k > 0 ? k : 0;
    pl.count = pl.dense ? pl.n_pages : (pl.k_pages > pl.n_forced ? pl.k_pages : pl.n_forced);
    return pl;
}

// ---- tracing build (-DSPARROW_TRACE; `python -m paper_2606_08446_b200.build --trace`, read by paper_2606_08446_b200/trace.py):
// the kernels drop %globaltimer stamps into a caller-provided buffer [65536 slots][8] of 64-bit words (sparrow_trace_set).
// In the normal build SPARROW_TR() is empty and the kernels carry no trace of it.
//   select_kernel:  slot = linear CTA index (CTAs past slot 55999 leave no stamps: the slots above belong to the decode, and
//                   nothing is ever written past the buffer's 65536 slots); 0 start, 1 prologue done, 2 summary stream done (warp 0), 3 CTA barrier passed,
//                   4 arrival atomic done, 5 top-k done (last CTA of a unit), 7 keys in shared memory, 6 radix select done
//   decode_kernel:  slot = 60000 + CTA; 0 start, 1 dependency wait over, 2 prefix table built, 3 look-up warp finished,
//                   4 first tile landed;   slot = 56000 + 9 x CTA + warp; 0 warp entry, 1 warp exit
#ifdef SPARROW_TRACE
__device__ unsigned long long *g_trace = nullptr;
__device__ __forceinline__ unsigned long long trace_now()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}
#define SPARROW_TR(slot, k)                                                       \
    do {                                                                          \
        const unsigned long long t__ = sparrow::trace_now();                      \
        unsigned long long *g__ = sparrow::g_trace;                               \
        if (g__ && (unsigned)(slot) < (unsigned)sparrow::kTraceSlots) g__[(size_t)(slot) * 8 + (k)] = t__; \
    } while (0)
#else
#define SPARROW_TR(slot, k) do { } while (0)
#endif
constexpr int kTraceSlots = 65536, kTraceDecodeCta = 60000, kTraceDecodeWarp = 56000;

// ---------------------------------------------------------------- small device helpers ----
__device__ __forceinline__ float bf16_lo(uint32_t x) { return __uint_as_float(x << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t x) { return __uint_as_float(x & 0xffff0000u); }

__device__ __forceinline__ uint4 ldg_stream16(const void *p)
{
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ---- programmatic dependent launch: the step's kernels (summarize / append -> select -> decode) are launched with
// cudaLaunchAttributeProgrammaticStreamSerialization, so the next kernel's CTAs can be brought up while this one
// drains.  Every kernel calls chain_entry() first: it lets its dependents start launching and then waits until everything
// before it in the stream has completed and is visible -- nothing is read or written before that point.
// The decode kernel calls chain_wait() only: it leaves room on its SMs (168 registers, one CTA), so a dependent launched
// early would sit beside it for the whole launch, and warps parked in griddepcontrol.wait are not free (measured: the
// step 15 us slower at cfg3 with select's CTAs resident beside the decode CTAs).  Its dependents start when it completes.
__device__ __forceinline__ void chain_wait()
{
#ifndef SPARROW_NO_PDL
    asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
}
__device__ __forceinline__ void chain_entry()
{
#ifndef SPARROW_NO_PDL
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
#endif
    chain_wait();
}

// ---- mbarrier + bulk-copy (TMA) primitives; shared-memory operands are 32-bit shared::cta addresses ----
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
// make freshly initialised barriers visible to the async proxy (the TMA unit completes transactions on them)
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
// (bounded: a protocol bug becomes a trap -- a launch failure the caller sees -- instead of a hung device)
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    for (uint32_t n = 0; !mbar_try_wait(bar, parity); ++n)
        if (n > (1u << 26)) __trap();
}
// 1-D bulk copy global -> shared (UBLKCP): bytes and both addresses multiples of 16; completes `bytes` on `bar`
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ uint4 lds128(uint32_t addr)
{
    uint4 r;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr));
    return r;
}

}  // namespace sparrow
