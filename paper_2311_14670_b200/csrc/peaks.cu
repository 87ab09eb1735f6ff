// peaks.cu -- register-only instruction chains that measure the arithmetic peaks the hot kernels are judged against
// (DESIGN.md "Measurement"): MEASURED_PEAKS.json has HBM and bf16 entries only, so the FP64 FMA, FP64 tensor-core (DMMA) and
// FP32 FMA peaks are measured in the same process, at the clocks of the same run.
//   kind 0: DFMA   -- 16 independent fma.rn.f64 chains per thread            (2 flop per instruction and lane)
//   kind 1: DMMA   -- 8 independent mma.sync.m8n8k4.f64 accumulator chains   (512 flop per warp instruction)
//   kind 2: FFMA   -- 16 independent fma.rn.f32 chains per thread
//   kind 3: FFMA2  -- 16 independent fma.rn.f32x2 chains per thread (packed: 4 flop per instruction and lane; theta_f32.cu)
#include "internal.h"

#include <cuda_runtime.h>

namespace {

__global__ void __launch_bounds__(256) peak_dfma_kernel(int iters, double* sink) {
    double a[16];
    const double x = 1.0 + 1e-9 * threadIdx.x, y = 1e-12 * (blockIdx.x + 1);
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = (double)i;
    for (int k = 0; k < iters; ++k) {
#pragma unroll
        for (int i = 0; i < 16; ++i) a[i] = fma(a[i], x, y);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += a[i];
    if (s == 123.456) sink[0] = s;
}

__global__ void __launch_bounds__(256) peak_dmma_kernel(int iters, double* sink) {
    double c[8][2];
    const double a = 1.0 + 1e-9 * threadIdx.x, b = 1e-3 * ((threadIdx.x & 7) + 1);
#pragma unroll
    for (int i = 0; i < 8; ++i) { c[i][0] = (double)i; c[i][1] = -(double)i; }
    for (int k = 0; k < iters; ++k) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1])
                         : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
    if (s == 123.456) sink[0] = s;
}

__global__ void __launch_bounds__(256) peak_ffma_kernel(int iters, double* sink) {
    float a[16];
    const float x = 1.0f + 1e-6f * threadIdx.x, y = 1e-6f * (blockIdx.x + 1);
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = (float)i;
    for (int k = 0; k < iters; ++k) {
#pragma unroll
        for (int i = 0; i < 16; ++i) a[i] = fmaf(a[i], x, y);
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += a[i];
    if (s == 123.456f) sink[0] = s;
}

__global__ void __launch_bounds__(256) peak_ffma2_kernel(int iters, double* sink) {
    float2 a[16];
    const float2 x = make_float2(1.0f + 1e-6f * threadIdx.x, 1.0f - 1e-6f * threadIdx.x), y = make_float2(1e-6f * (blockIdx.x + 1), -1e-6f);
#pragma unroll
    for (int i = 0; i < 16; ++i) a[i] = make_float2((float)i, (float)-i);
    for (int k = 0; k < iters; ++k) {
#pragma unroll
        for (int i = 0; i < 16; ++i) a[i] = __ffma2_rn(a[i], x, y);
    }
    float s = 0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += a[i].x + a[i].y;
    if (s == 123.456f) sink[0] = s;
}

}  // namespace

cudaError_t launch_peak(int kind, int iters, int nsm, double* sink, cudaStream_t st, double* flop) {
    const int blocks = nsm * 8, threads = 256;
    if (kind == 0) {
        peak_dfma_kernel<<<blocks, threads, 0, st>>>(iters, sink);
        *flop = 2.0 * 16 * (double)iters * blocks * threads;
    } else if (kind == 1) {
        peak_dmma_kernel<<<blocks, threads, 0, st>>>(iters, sink);
        *flop = 512.0 * 8 * (double)iters * blocks * (threads / 32);      // m8n8k4: 2*8*8*4 flop per warp instruction
    } else if (kind == 2) {
        peak_ffma_kernel<<<blocks, threads, 0, st>>>(iters, sink);
        *flop = 2.0 * 16 * (double)iters * blocks * threads;
    } else if (kind == 3) {
        peak_ffma2_kernel<<<blocks, threads, 0, st>>>(iters, sink);
        *flop = 4.0 * 16 * (double)iters * blocks * threads;
    } else
        return cudaErrorInvalidValue;
    count_launch();
    return cudaGetLastError();
}
