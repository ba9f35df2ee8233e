// Measured non-tensor arithmetic peak (roofline denominator): independent FMA chains in registers.
#include <cuda_runtime.h>

#include "../../include/pairhmm_b200.h"

namespace {
constexpr int PEAK_ITERS = 8192;
template <int KIND> __global__ void __launch_bounds__(256) k_peak(float* out, float a, float b) {
    float f[16];
    double d[8];
    unsigned long long p[8];
#pragma unroll
    for (int i = 0; i < 16; i++) f[i] = threadIdx.x * 0.001f + i;
#pragma unroll
    for (int i = 0; i < 8; i++) {
        d[i] = f[i];
        p[i] = ((unsigned long long)__float_as_uint(f[2 * i + 1]) << 32) | __float_as_uint(f[2 * i]);
    }
    const unsigned long long a2 = ((unsigned long long)__float_as_uint(a) << 32) | __float_as_uint(a);
    const unsigned long long b2 = ((unsigned long long)__float_as_uint(b) << 32) | __float_as_uint(b);
    for (int it = 0; it < PEAK_ITERS; it++) {
        if (KIND == 0) {
#pragma unroll
            for (int i = 0; i < 16; i++) f[i] = fmaf(f[i], a, b);
        } else if (KIND == 1) {
#pragma unroll
            for (int i = 0; i < 8; i++) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(p[i]) : "l"(a2), "l"(b2));
        } else {
#pragma unroll
            for (int i = 0; i < 8; i++) d[i] = fma(d[i], (double)a, (double)b);
        }
    }
    float r = 0;
#pragma unroll
    for (int i = 0; i < 16; i++) r += f[i];
#pragma unroll
    for (int i = 0; i < 8; i++) r += (float)d[i] + __uint_as_float((unsigned)p[i]) + __uint_as_float((unsigned)(p[i] >> 32));
    if (r == 123.456f) out[0] = r;
}
}  // namespace

extern "C" int phmm_measure_peak(int device, int kind, int reps, double* out_tflops) {
    if (!out_tflops || kind < 0 || kind > 2) return PHMM_E_ARG;
    if (reps < 1) reps = 3;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess || cudaSetDevice(device) != cudaSuccess) return PHMM_E_CUDA;
    float* out = nullptr;
    if (cudaMalloc(&out, 4) != cudaSuccess) return PHMM_E_NOMEM;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int grid = prop.multiProcessorCount * 8, tpb = 256;
    const double lane_fma = (double)grid * tpb * PEAK_ITERS * (kind == 2 ? 8.0 : 16.0);
    double best = 0;
    for (int r = 0; r <= reps; r++) {  // first launch is warm-up
        cudaEventRecord(e0);
        if (kind == 0) k_peak<0><<<grid, tpb>>>(out, 0.999f, 0.001f);
        else if (kind == 1) k_peak<1><<<grid, tpb>>>(out, 0.999f, 0.001f);
        else k_peak<2><<<grid, tpb>>>(out, 0.999f, 0.001f);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(out); return PHMM_E_CUDA; }
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        const double tf = 2.0 * lane_fma / (ms * 1e-3) / 1e12;
        if (r > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    *out_tflops = best;
    return cudaGetLastError() == cudaSuccess ? PHMM_OK : PHMM_E_CUDA;
}
