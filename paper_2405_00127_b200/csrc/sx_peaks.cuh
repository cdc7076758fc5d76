// sx_peaks.cuh -- issue-rate microbenchmarks behind sx_measure_issue_peaks: the measured ceilings R_fp32 and R_mufu of
// the roofline T_roof = max(B_alg / BW_hbm, I_fp32 / R_fp32, I_mufu / R_mufu) that bench.py reports.
//
//   k_peak_ffma   independent FFMA chains (8 per thread), all SMs, 1024 threads per SM: FP32 lane-operations per second
//   k_peak_mix    the same number of FFMA interleaved with integer ALU instructions (the stroke kernels are such a mix:
//                 the fma and alu pipes issue side by side): warp instructions issued per second x 32 lanes
//   k_peak_mufu   independent MUFU.RSQ chains: special-function lane-operations per second
// Timed with CUDA events on the default stream after a warm-up launch; the best of 5 launches is reported.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sx {

constexpr int kPeakThreads = 256, kPeakBlocksPerSM = 4, kPeakIters = 4096;

__global__ void __launch_bounds__(kPeakThreads) k_peak_ffma(float* out, float a, float b) {
    float x0 = threadIdx.x, x1 = x0 + 1.0f, x2 = x0 + 2.0f, x3 = x0 + 3.0f, x4 = x0 + 4.0f, x5 = x0 + 5.0f, x6 = x0 + 6.0f, x7 = x0 + 7.0f;
#pragma unroll 8
    for (int i = 0; i < kPeakIters; i++) {
        x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
        x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
    }
    out[blockIdx.x * kPeakThreads + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

__global__ void __launch_bounds__(kPeakThreads) k_peak_mix(float* out, float a, float b, uint32_t m) {
    float x0 = threadIdx.x, x1 = x0 + 1.0f, x2 = x0 + 2.0f, x3 = x0 + 3.0f;
    uint32_t y0 = threadIdx.x, y1 = y0 + 1u, y2 = y0 + 2u, y3 = y0 + 3u;
#pragma unroll 8
    for (int i = 0; i < kPeakIters; i++) {
        x0 = fmaf(x0, a, b); y0 = (y0 ^ m) + (y0 >> 3);
        x1 = fmaf(x1, a, b); y1 = (y1 ^ m) + (y1 >> 3);
        x2 = fmaf(x2, a, b); y2 = (y2 ^ m) + (y2 >> 3);
        x3 = fmaf(x3, a, b); y3 = (y3 ^ m) + (y3 >> 3);
    }
    out[blockIdx.x * kPeakThreads + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + __uint_as_float(((y0 ^ y1) ^ (y2 ^ y3)) & 0x3fffffffu);
}

__global__ void __launch_bounds__(kPeakThreads) k_peak_mufu(float* out, float a) {
    float x0 = threadIdx.x + a, x1 = x0 + 1.0f, x2 = x0 + 2.0f, x3 = x0 + 3.0f, x4 = x0 + 4.0f, x5 = x0 + 5.0f, x6 = x0 + 6.0f, x7 = x0 + 7.0f;
#pragma unroll 4
    for (int i = 0; i < kPeakIters; i++) {
        asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(x0)); asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(x1));
        asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(x2)); asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(x3));
        asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(x4)); asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(x5));
        asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(x6)); asm volatile("rsqrt.approx.ftz.f32 %0, %0;" : "+f"(x7));
    }
    out[blockIdx.x * kPeakThreads + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

// h_out3: [0] FFMA lane-ops/s, [1] issued lane-ops/s of the FFMA + integer mix, [2] MUFU lane-ops/s
inline cudaError_t measure_issue_peaks(int device, double* h_out3) {
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return e;
    int sms = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    const int blocks = sms * kPeakBlocksPerSM;
    float* out = nullptr;
    e = cudaMalloc(&out, (size_t)blocks * kPeakThreads * sizeof(float));
    if (e != cudaSuccess) return e;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0); cudaEventCreate(&t1);
    const double threads = (double)blocks * kPeakThreads;
    const double ops[3] = {threads * kPeakIters * 8.0, threads * kPeakIters * 12.0, threads * kPeakIters * 8.0};  // mix: 4 FFMA + 4 x (LOP3, SHF/IADD) per iteration
    for (int k = 0; k < 3; k++) {
        float best = 1e30f;
        for (int rep = 0; rep < 6; rep++) {
            cudaEventRecord(t0, 0);
            if (k == 0) k_peak_ffma<<<blocks, kPeakThreads>>>(out, 0.999f, 0.001f);
            else if (k == 1) k_peak_mix<<<blocks, kPeakThreads>>>(out, 0.999f, 0.001f, 0x9e3779b9u);
            else k_peak_mufu<<<blocks, kPeakThreads>>>(out, 1.5f);
            cudaEventRecord(t1, 0);
            e = cudaEventSynchronize(t1);
            if (e != cudaSuccess) break;
            float ms = 0.0f;
            cudaEventElapsedTime(&ms, t0, t1);
            if (rep > 0 && ms < best) best = ms;
        }
        if (e != cudaSuccess) break;
        h_out3[k] = ops[k] / (best * 1e-3);
    }
    cudaEventDestroy(t0); cudaEventDestroy(t1);
    cudaFree(out);
    return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace sx
