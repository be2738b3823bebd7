// probes.cu -- bench hooks of include/flare_probes.h (libflare_probes.so): FP64 DMMA / DFMA issue peaks and an
// HBM copy, the roofline denominators bench.py reports against.  Not part of libflare_b200.so.
#include <cuda_runtime.h>

#include "../../include/flare_probes.h"

namespace {

__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

__global__ void k_probe_dmma(double* out, int iters, double a, double b) {
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; i++) { c[i][0] = threadIdx.x; c[i][1] = i; }
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++) dmma884(c[i][0], c[i][1], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
    if (s == 123.456) out[0] = s;
}

__global__ void k_probe_dfma(double* out, int iters, double a, double b) {
    double c[8];
#pragma unroll
    for (int i = 0; i < 8; i++) c[i] = threadIdx.x + i;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++) c[i] = fma(c[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += c[i];
    if (s == 123.456) out[0] = s;
}

__global__ void k_probe_copy(const double2* __restrict__ src, double2* __restrict__ dst, size_t n16) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n16; i += (size_t)gridDim.x * blockDim.x)
        dst[i] = src[i];
}

template <class Launch>
double best_ms(Launch&& launch, int reps) {
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return -1.0;
    launch();
    cudaDeviceSynchronize();
    float best = 1e30f;
    for (int r = 0; r < reps; r++) {
        cudaEventRecord(e0);
        launch();
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return cudaGetLastError() == cudaSuccess ? (double)best : -1.0;
}

int sm_count(int device) {
    cudaDeviceProp p;
    if (cudaSetDevice(device) != cudaSuccess || cudaGetDeviceProperties(&p, device) != cudaSuccess) return -1;
    return p.multiProcessorCount;
}

}  // namespace

extern "C" {
#pragma GCC visibility push(default)

double flare_probe_fp64_dmma_tflops(int device) {
    const int sms = sm_count(device);
    if (sms <= 0) return -1.0;
    double* out = nullptr;
    if (cudaMalloc(&out, 8) != cudaSuccess) return -1.0;
    const int blocks = sms * 2, threads = 256, iters = 1 << 14;
    const double ms = best_ms([&] { k_probe_dmma<<<blocks, threads>>>(out, iters, 1.0000001, 1e-9); }, 5);
    cudaFree(out);
    if (ms <= 0.0) return -1.0;
    const double flops = 512.0 * 8 * (double)iters * blocks * (threads / 32);  // 512 flop per DMMA.8x8x4
    return flops / (ms * 1e-3) * 1e-12;
}

double flare_probe_fp64_dfma_tflops(int device) {
    const int sms = sm_count(device);
    if (sms <= 0) return -1.0;
    double* out = nullptr;
    if (cudaMalloc(&out, 8) != cudaSuccess) return -1.0;
    const int blocks = sms * 4, threads = 256, iters = 1 << 14;
    const double ms = best_ms([&] { k_probe_dfma<<<blocks, threads>>>(out, iters, 1.0000001, 1e-9); }, 5);
    cudaFree(out);
    if (ms <= 0.0) return -1.0;
    const double flops = 2.0 * 8 * (double)iters * blocks * threads;
    return flops / (ms * 1e-3) * 1e-12;
}

double flare_probe_hbm_copy_gbs(int device, size_t bytes) {
    const int sms = sm_count(device);
    if (sms <= 0 || bytes < 16) return -1.0;
    const size_t n16 = bytes / 16;
    double2 *a = nullptr, *b = nullptr;
    if (cudaMalloc(&a, n16 * 16) != cudaSuccess) return -1.0;
    if (cudaMalloc(&b, n16 * 16) != cudaSuccess) { cudaFree(a); return -1.0; }
    cudaMemset(a, 0, n16 * 16);
    const double ms = best_ms([&] { k_probe_copy<<<sms * 16, 512>>>(a, b, n16); }, 5);
    cudaFree(a);
    cudaFree(b);
    if (ms <= 0.0) return -1.0;
    return 2.0 * (double)n16 * 16.0 / (ms * 1e-3) * 1e-9;
}

#pragma GCC visibility pop
}  // extern "C"
