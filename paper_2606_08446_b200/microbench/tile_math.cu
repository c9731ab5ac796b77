// tile_math.cu -- microbenchmark behind DESIGN.md 6.3 / profiles/r2_decode.md: cycles per 16-token tile of the decode consumer's
// math alone (S = Q K^T, online softmax, O += P V with mma.sync.m16n8k16 bf16 -> fp32 and ldmatrix from a swizzled shared-memory
// tile), per warp, at 1 / 2 / 3 warps per scheduler partition.  No global memory traffic, no hand-out: what the tensor-core path
// itself costs.  Not part of the library (nothing links it).
//   nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -o tile_math paper_2606_08446_b200/microbench/tile_math.cu && ./tile_math
// ("S = Q K^T" alone is not meaningful: with its result unused the compiler hoists most of it; the other rows stand.)
#include <cstdio>
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>
__device__ __forceinline__ void ldsm_x4(uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3, uint32_t addr)
{ asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];" : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr)); }
__device__ __forceinline__ void ldsm_x4_t(uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3, uint32_t addr)
{ asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];" : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr)); }
__device__ __forceinline__ void mma_rows07(float &c0, float &c1, uint32_t a0, uint32_t a2, uint32_t b0, uint32_t b1)
{
    float d2, d3;
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%5}, {%7,%8}, {%0,%1,%9,%9};"
                 : "+f"(c0), "+f"(c1), "=f"(d2), "=f"(d3) : "r"(a0), "r"(0u), "r"(a2), "r"(b0), "r"(b1), "f"(0.f));
}
__device__ __forceinline__ float fast_exp2(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) { __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi); return *reinterpret_cast<uint32_t *>(&v); }
__device__ __forceinline__ uint32_t tile_off(int t, int c) { const int rho = 2 * t + (c >> 3); return (uint32_t)(rho * 128 + (((c & 7) ^ (rho & 7)) << 4)); }

template <int MODE>   // 0 full, 1 S only, 2 PV only, 3 softmax only
__global__ void k(float *out, long long *cyc, int iters)
{
    extern __shared__ __align__(1024) unsigned char smem[];
    for (int i = threadIdx.x; i < 8192 * 4 / 4; i += blockDim.x) reinterpret_cast<uint32_t *>(smem)[i] = 0x3c003c00u + i;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int mat = lane >> 3, rr = lane & 7;
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(smem);
    uint32_t qa[8][2];
    for (int kk = 0; kk < 8; ++kk) { qa[kk][0] = 0x3c003c00u + lane + kk; qa[kk][1] = 0x3c003c01u + lane * 3 + kk; }
    float o[16][2];
    for (int nt = 0; nt < 16; ++nt) { o[nt][0] = 0.f; o[nt][1] = 0.f; }
    float m_run = -INFINITY, l_run = 0.f;
    float s0a = 0.1f * lane, s0b = 0.2f, s1a = 0.3f, s1b = 0.4f;
    long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
        const uint32_t kb = base + ((it + warp) & 3) * 8192, vb = kb + 4096;
        if (MODE == 0 || MODE == 1) {
            s0a = s0b = s1a = s1b = 0.f;
#pragma unroll
            for (int kk = 0; kk < 8; ++kk) {
                uint32_t b0, b1, b2, b3;
                ldsm_x4(b0, b1, b2, b3, kb + tile_off((mat >> 1) * 8 + rr, 2 * kk + (mat & 1)));
                mma_rows07(s0a, s0b, qa[kk][0], qa[kk][1], b0, b1);
                mma_rows07(s1a, s1b, qa[kk][0], qa[kk][1], b2, b3);
            }
        }
        uint32_t pa0 = 0x3c003c00u, pa2 = 0x3c003c00u;
        if (MODE == 0 || MODE == 3) {
            float x0 = s0a * 0.1f, x1 = s0b * 0.1f, x2 = s1a * 0.1f, x3 = s1b * 0.1f;
            float mx = fmaxf(fmaxf(x0, x1), fmaxf(x2, x3));
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 1));
            mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 2));
            const float m_new = fmaxf(m_run, mx);
            const float m_safe = m_new == -INFINITY ? 0.f : m_new;
            const float alpha = fast_exp2(m_run - m_safe);
            const float p0 = fast_exp2(x0 - m_safe), p1 = fast_exp2(x1 - m_safe), p2 = fast_exp2(x2 - m_safe), p3 = fast_exp2(x3 - m_safe);
            l_run = l_run * alpha + ((p0 + p1) + (p2 + p3));
            m_run = m_new;
            if (!__all_sync(0xffffffffu, alpha == 1.f)) {
#pragma unroll
                for (int nt = 0; nt < 16; ++nt) { o[nt][0] *= alpha; o[nt][1] *= alpha; }
            }
            pa0 = pack_bf16(p0, p1); pa2 = pack_bf16(p2, p3);
            if (MODE == 3) { s0a += p0; s0b += p1; s1a += p2; s1b += p3; }
        }
        if (MODE == 0 || MODE == 2) {
#pragma unroll
            for (int jn = 0; jn < 8; ++jn) {
                uint32_t b0, b1, b2, b3;
                ldsm_x4_t(b0, b1, b2, b3, vb + tile_off((mat & 1) * 8 + rr, 2 * jn + (mat >> 1)));
                mma_rows07(o[2 * jn][0], o[2 * jn][1], pa0, pa2, b0, b1);
                mma_rows07(o[2 * jn + 1][0], o[2 * jn + 1][1], pa0, pa2, b2, b3);
            }
        }
    }
    long long t1 = clock64();
    float acc = l_run + s0a + s0b + s1a + s1b;
    for (int nt = 0; nt < 16; ++nt) acc += o[nt][0] + o[nt][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
    if (lane == 0) cyc[blockIdx.x * (blockDim.x / 32) + warp] = t1 - t0;
}
template <int MODE> void run(const char *name, int warps)
{
    float *out; long long *cyc; cudaMalloc(&out, 148 * 1024 * 4); cudaMalloc(&cyc, 148 * 32 * 8);
    cudaFuncSetAttribute(k<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, 32768);
    const int iters = 2000;
    k<MODE><<<148, warps * 32, 32768>>>(out, cyc, iters); cudaDeviceSynchronize();
    k<MODE><<<148, warps * 32, 32768>>>(out, cyc, iters); cudaDeviceSynchronize();
    long long h[32]; cudaMemcpy(h, cyc, warps * 8, cudaMemcpyDeviceToHost);
    printf("%-14s %2d warps/SM: %7.1f cycles per tile per warp  -> %.2f tiles/us/SM at 1.9 GHz (%s)\n", name, warps, (double)h[0] / iters,
           warps * 1900.0 / ((double)h[0] / iters), cudaGetErrorString(cudaGetLastError()));
    cudaFree(out); cudaFree(cyc);
}
int main()
{
    for (int w : {4, 8, 12}) { run<0>("full math", w); run<1>("S = Q K^T", w); run<2>("O += P V", w); run<3>("softmax", w); }
    return 0;
}
