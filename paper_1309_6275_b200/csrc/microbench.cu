// Roofline micro-benchmarks: the denominators the vote kernel and the stencil are
// reported against are measured on the box, not assumed.  Synchronous helpers; not part of the hot path.
#include <stdio.h>

#include "hough_internal.cuh"

namespace {

// kind 0: conflict-free 32-bit shared atomics, one add + one or per step, result unused (the vote's pattern)
__global__ void __launch_bounds__(1024) mb_shared_atomics(int iters, uint32_t* sink)
{
    __shared__ uint32_t s[8192];
    for (int i = threadIdx.x; i < 8192; i += blockDim.x) s[i] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t idx = (warp * 97u) & 255u;                  // row of 32 words; lanes hit 32 distinct banks
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            uint32_t* w = &s[((idx + u * 13u) & 255u) * 32u + lane];
            atomicAdd(w, 1u);
            atomicOr(w, 0x10000u);
        }
        idx += 7u;
    }
    __syncthreads();
    if (s[threadIdx.x] == 0xdeadbeefu) sink[0] = 1;
}

// kind 1: fp32 non-FMA arithmetic, 8 independent chains per thread
__global__ void __launch_bounds__(1024) mb_fp32(int iters, float seed, float* sink)
{
    float a0 = seed + threadIdx.x, a1 = a0 + 1.f, a2 = a0 + 2.f, a3 = a0 + 3.f;
    float a4 = a0 + 4.f, a5 = a0 + 5.f, a6 = a0 + 6.f, a7 = a0 + 7.f;
    const float m = 0.999999f + seed * 1e-9f, c = 1e-3f + seed * 1e-9f;     // register operands, as in the vote sweep
    for (int i = 0; i < iters; ++i) {
        a0 = __fmul_rn(a0, m); a1 = __fadd_rn(a1, c); a2 = __fmul_rn(a2, m); a3 = __fadd_rn(a3, c);
        a4 = __fmul_rn(a4, m); a5 = __fadd_rn(a5, c); a6 = __fmul_rn(a6, m); a7 = __fadd_rn(a7, c);
        a0 = __fadd_rn(a0, c); a1 = __fmul_rn(a1, m); a2 = __fadd_rn(a2, c); a3 = __fmul_rn(a3, m);
        a4 = __fadd_rn(a4, c); a5 = __fmul_rn(a5, m); a6 = __fadd_rn(a6, c); a7 = __fmul_rn(a7, m);
    }
    const float r = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (r == 12345.678f) sink[0] = r;
}

__global__ void __launch_bounds__(512) mb_read(const uint4* __restrict__ src, size_t n16, uint32_t* sink)
{
    uint32_t acc = 0;
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    for (; i + 3 * stride < n16; i += 4 * stride) {
        const uint4 a = src[i], b = src[i + stride], c = src[i + 2 * stride], d = src[i + 3 * stride];
        acc += a.x ^ a.y ^ a.z ^ a.w ^ b.x ^ b.y ^ b.z ^ b.w ^ c.x ^ c.y ^ c.z ^ c.w ^ d.x ^ d.y ^ d.z ^ d.w;
    }
    for (; i < n16; i += stride) { const uint4 a = src[i]; acc += a.x ^ a.y ^ a.z ^ a.w; }
    if (acc == 0x12345u) sink[0] = acc;
}

__global__ void __launch_bounds__(512) mb_write(uint4* __restrict__ dst, size_t n16)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += stride)
        dst[i] = make_uint4((uint32_t)i, 1u, 2u, 3u);
}

// kind 4: packed fp32x2 non-FMA arithmetic (FMUL2 / FADD2 with register operands), 8 independent chains per thread
__device__ __forceinline__ uint64_t mb_pk(float lo, float hi)
{
    uint64_t r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__global__ void __launch_bounds__(1024) mb_fp32x2(int iters, float seed, float* sink)
{
    uint64_t a[8];
    for (int i = 0; i < 8; ++i) a[i] = mb_pk(seed + threadIdx.x + i, seed + threadIdx.x + i + 0.5f);
    const uint64_t m = mb_pk(0.999999f + seed * 1e-9f, 0.999998f), c = mb_pk(1e-3f + seed * 1e-9f, 2e-3f);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; i += 2) {                         // a product never feeds a sum: ptxas would contract
            asm volatile("mul.rn.f32x2 %0, %0, %1;" : "+l"(a[i]) : "l"(m));
            asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(a[i + 1]) : "l"(c));
            asm volatile("mul.rn.f32x2 %0, %0, %1;" : "+l"(a[i]) : "l"(m));
            asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(a[i + 1]) : "l"(c));
        }
    }
    uint64_t x = 0;
    for (int i = 0; i < 8; ++i) x ^= a[i];
    if (x == 0x12345ull) sink[0] = 1.f;
}

// kinds 5, 6: what one SM can store towards L2 (the buffer is small enough to stay in L2: no DRAM limit).  Every
// block rewrites its own 128 KB; kind 5 fully coalesced 128-bit stores, kind 6 the pattern of the vote flush (256-bit
// stores, lane pairs write 64 contiguous bytes of rows 1 KB apart).
template <bool FLUSH_PATTERN>
__global__ void __launch_bounds__(1024) mb_store(unsigned char* buf, int iters)
{
    unsigned char* base = buf + (size_t)blockIdx.x * 131072;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int it = 0; it < iters; ++it) {
        if (!FLUSH_PATTERN) {
            for (int o = threadIdx.x * 16; o < 131072; o += 1024 * 16) *reinterpret_cast<uint4*>(base + o) = make_uint4(it, 1, 2, 3);
        } else {
            for (int g = 0; g < 4; ++g)
                for (int kb = warp; kb < 16; kb += 32) {
                    unsigned char* q = base + g * 32768 + (lane & ~1) * 1024 + kb * 64 + (lane & 1) * 32;
                    asm volatile("st.global.cs.v8.b32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1};" :: "l"(q), "r"(it) : "memory");
                    asm volatile("st.global.cs.v8.b32 [%0], {%1,%1,%1,%1,%1,%1,%1,%1};" :: "l"(q + 1024), "r"(it) : "memory");
                }
        }
    }
}

}  // namespace

extern "C" int hough_microbench(int kind, size_t bytes, double* host_rate)
{
    if (!host_rate || kind < 0 || kind > 6) return HOUGH_EINVAL;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return HOUGH_ECUDA;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaEvent_t t0 = nullptr, t1 = nullptr;
    uint32_t* sink = nullptr;
    if (cudaEventCreate(&t0) != cudaSuccess || cudaEventCreate(&t1) != cudaSuccess ||
        cudaMalloc((void**)&sink, 16) != cudaSuccess) {
        if (t0) cudaEventDestroy(t0);
        if (t1) cudaEventDestroy(t1);
        cudaFree(sink);
        return HOUGH_ECUDA;
    }
    void* buf = nullptr;
    double work = 0.0;
    float best_ms = 1e30f;
    const int reps = 5;
    if (kind == 5 || kind == 6) bytes = (size_t)sms * 131072;
    if (kind == 2 || kind == 3 || kind == 5 || kind == 6) {
        if (bytes < (1u << 20)) bytes = (size_t)1 << 30;
        if (cudaMalloc(&buf, bytes) != cudaSuccess) {
            cudaGetLastError();
            cudaFree(sink); cudaEventDestroy(t0); cudaEventDestroy(t1);
            return HOUGH_ENOMEM;
        }
        cudaMemset(buf, 1, bytes);
    }
    for (int rep = 0; rep < reps + 1; ++rep) {
        cudaEventRecord(t0);
        if (kind == 0) {
            const int iters = 4096;
            mb_shared_atomics<<<sms * 2, 1024>>>(iters, sink);
            work = (double)sms * 2 * 1024 * iters * 16;
        } else if (kind == 1) {
            const int iters = 8192;
            mb_fp32<<<sms * 2, 1024>>>(iters, 1.0f, (float*)sink);
            work = (double)sms * 2 * 1024 * iters * 16;
        } else if (kind == 4) {
            const int iters = 8192;
            mb_fp32x2<<<sms * 2, 1024>>>(iters, 1.0f, (float*)sink);
            work = (double)sms * 2 * 1024 * iters * 16;          // packed instructions (two operations each)
        } else if (kind == 5 || kind == 6) {
            const int iters = 2000;
            if (kind == 5) mb_store<false><<<sms, 1024>>>((unsigned char*)buf, iters);
            else mb_store<true><<<sms, 1024>>>((unsigned char*)buf, iters);
            work = (double)sms * 131072.0 * iters;               // bytes, all SMs together
        } else if (kind == 2) {
            mb_read<<<sms * 8, 512>>>((const uint4*)buf, bytes / 16, sink);
            work = (double)bytes;
        } else {
            mb_write<<<sms * 8, 512>>>((uint4*)buf, bytes / 16);
            work = (double)bytes;
        }
        cudaEventRecord(t1);
        cudaEventSynchronize(t1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, t0, t1);
        if (rep > 0 && ms < best_ms) best_ms = ms;
    }
    cudaError_t err = cudaGetLastError();
    cudaFree(buf); cudaFree(sink);
    cudaEventDestroy(t0); cudaEventDestroy(t1);
    if (err != cudaSuccess) return HOUGH_ECUDA;
    *host_rate = work / ((double)best_ms * 1e-3);
    return HOUGH_OK;
}
