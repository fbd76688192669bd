// ubench.cu -- FP32 pipe micro-benchmark behind gx_ubench_fp32 (include/gx.h): the measured peak that
// bench.py reports next to the nominal one (roofline.peak_measured).  Each thread runs `iters` rounds of
// 16 independent dependency chains of one instruction kind, so that the pipe, not latency, is the limit.
#include <cuda_runtime.h>

#include "../../include/gx.h"
#include "dft_packed.cuh"

namespace {

typedef unsigned long long u64;
__device__ __forceinline__ u64 pk(float a, float b) { u64 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a), "f"(b)); return r; }

template <int KIND> __global__ void fp32_kernel(float* sink, int iters, float seed) {
    constexpr int CH = 16;
    float a[CH];
    u64 p[CH];
    const float x = seed + 1e-7f * threadIdx.x, y = 1.0f + 1e-6f * seed;
#pragma unroll
    for (int c = 0; c < CH; ++c) { a[c] = x + c; p[c] = pk(x + c, y - c); }
    const u64 px = pk(x, y), py = pk(y, x);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int c = 0; c < CH; ++c) {
            if (KIND == 0) asm volatile("add.f32 %0, %0, %1;" : "+f"(a[c]) : "f"(x));
            if (KIND == 1) asm volatile("mul.f32 %0, %0, %1;" : "+f"(a[c]) : "f"(y));
            if (KIND == 2) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(a[c]) : "f"(y), "f"(x));
            if (KIND == 3) asm volatile("add.f32x2 %0, %0, %1;" : "+l"(p[c]) : "l"(px));
            if (KIND == 4) asm volatile("mul.f32x2 %0, %0, %1;" : "+l"(p[c]) : "l"(py));
            if (KIND == 5) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p[c]) : "l"(py), "l"(px));
        }
    }
    float s = 0.f;
#pragma unroll
    for (int c = 0; c < CH; ++c) s += a[c] + (float)(p[c] & 0xffff);
    if (s == 123.456f) sink[0] = s;
}

// batched 16-point complex DFTs held in registers, the building block of the x passes: `iters` transforms per
// thread back to back (each followed by one twiddle multiplication, as in a two-pass FFT), scalar or packed
// (two transforms per thread in FADD2/FFMA2 form)
template <bool PACKED> __global__ void dft16_kernel(float* sink, int iters, float seed) {
    using namespace gx;
    if constexpr (PACKED) {
        pk::c2 v[16];
#pragma unroll
        for (int i = 0; i < 16; ++i)
            v[i] = pk::make_c2(pk::pk2(seed + i + threadIdx.x * 1e-3f, seed - i), pk::pk2(0.5f * i, seed * i - threadIdx.x * 1e-3f));
        for (int it = 0; it < iters; ++it) {
            pk::dft<16, +1>(v);
#pragma unroll
            for (int i = 1; i < 16; ++i) v[i] = pk::cmul_s(v[i], 0.0624f, 0.0012f * i);
        }
        float s = 0.f;
#pragma unroll
        for (int i = 0; i < 16; ++i) s += pk::lo(v[i].re) + pk::hi(v[i].im);
        if (s == 123.456f) sink[0] = s;
    } else {
        float2 v[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) v[i] = make_float2(seed + i + threadIdx.x * 1e-3f, 0.5f * i - seed);
        for (int it = 0; it < iters; ++it) {
            dft<16, +1>(v);
#pragma unroll
            for (int i = 1; i < 16; ++i) v[i] = cmul(v[i], make_float2(0.0624f, 0.0012f * i));
        }
        float s = 0.f;
#pragma unroll
        for (int i = 0; i < 16; ++i) s += v[i].x + v[i].y;
        if (s == 123.456f) sink[0] = s;
    }
}

}  // namespace

extern "C" int gx_ubench_dft16(int packed, int threads_per_block, int blocks_per_sm, int iters, double* ms, double* transforms) {
    if (threads_per_block < 32 || threads_per_block > 1024 || blocks_per_sm < 1 || iters < 1 || !ms || !transforms) return GX_ERR_ARG;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return GX_ERR_CUDA;
    float* sink = nullptr;
    if (cudaMalloc(&sink, 4) != cudaSuccess) return GX_ERR_ALLOC;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int grid = nsm * blocks_per_sm;
    void (*k)(float*, int, float) = packed ? dft16_kernel<true> : dft16_kernel<false>;
    k<<<grid, threads_per_block>>>(sink, iters / 8 + 1, 0.37f);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) {
        cudaEventRecord(e0);
        k<<<grid, threads_per_block>>>(sink, iters, 0.37f);
        cudaEventRecord(e1);
        e = cudaEventSynchronize(e1);
    }
    float t = 0.f;
    if (e == cudaSuccess) cudaEventElapsedTime(&t, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    if (e != cudaSuccess) return GX_ERR_CUDA;
    *ms = t;
    *transforms = (double)grid * threads_per_block * (double)iters * (packed ? 2.0 : 1.0);
    return GX_OK;
}

extern "C" int gx_ubench_fp32(int kind, int threads_per_block, int blocks_per_sm, int iters, double* ms, double* lane_ops) {
    if (kind < 0 || kind > 5 || threads_per_block < 32 || threads_per_block > 1024 || blocks_per_sm < 1 || iters < 1 || !ms ||
        !lane_ops)
        return GX_ERR_ARG;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
        return GX_ERR_CUDA;
    float* sink = nullptr;
    if (cudaMalloc(&sink, 4) != cudaSuccess) return GX_ERR_ALLOC;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int grid = nsm * blocks_per_sm;
    void (*k)(float*, int, float) = kind == 0 ? fp32_kernel<0> : kind == 1 ? fp32_kernel<1> : kind == 2 ? fp32_kernel<2>
                                   : kind == 3 ? fp32_kernel<3> : kind == 4 ? fp32_kernel<4> : fp32_kernel<5>;
    k<<<grid, threads_per_block>>>(sink, iters / 8 + 1, 0.5f);      // warm-up
    if (cudaGetLastError() != cudaSuccess) {                         // e.g. too many registers for this block size
        cudaEventDestroy(e0);
        cudaEventDestroy(e1);
        cudaFree(sink);
        return GX_ERR_CUDA;
    }
    cudaEventRecord(e0);
    k<<<grid, threads_per_block>>>(sink, iters, 0.5f);
    cudaEventRecord(e1);
    cudaError_t e = cudaEventSynchronize(e1);
    float t = 0.f;
    cudaEventElapsedTime(&t, e0, e1);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(sink);
    if (e != cudaSuccess) return GX_ERR_CUDA;
    *ms = t;
    *lane_ops = (double)grid * threads_per_block * (double)iters * 16.0 * (kind >= 3 ? 2.0 : 1.0);
    return GX_OK;
}
