// peaks.cu -- measured fp64 roofs of the device the library runs on: the denominators of the
// "alu" rooflines bench.py reports for the passes that are bound by fp64 arithmetic (spread, gather, real space).
// Register-resident chains, no memory traffic: DFMA (vector pipe) and mma.sync.m8n8k4.f64 (tensor path).
#include "pce_internal.h"

__global__ void __launch_bounds__(256) k_peak_dfma(double* out, int iters, double a, double b)
{
    double acc[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) acc[i] = threadIdx.x * 1e-3 + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) acc[i] = fma(acc[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 16; ++i) s += acc[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) k_peak_dmma(double* out, int iters, double a, double b)
{
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; ++i) { c[i][0] = threadIdx.x * 1e-3; c[i][1] = i; }
    const double A = a + threadIdx.x * 1e-9, B = b;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(A), "d"(B));
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// tflops[0] = DFMA chains, tflops[1] = fp64 mma (2 flops per multiply-add), best of 3 timed launches each
extern "C" int pce_measure_fp64_peaks(double tflops[2])
{
    if (!tflops) return PCE_EINVAL;
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return PCE_ECUDA;
    const int threads = 256, blocks = nsm * 4, iters = 20000;
    double* out = nullptr;
    if (cudaMalloc(&out, (size_t)blocks * threads * sizeof(double)) != cudaSuccess) return PCE_ENOMEM;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    for (int which = 0; which < 2; ++which) {
        float best = 1e30f;
        for (int rep = 0; rep < 4; ++rep) {
            cudaEventRecord(e0);
            if (which == 0) k_peak_dfma<<<blocks, threads>>>(out, iters, 0.999, 1e-3);
            else k_peak_dmma<<<blocks, threads>>>(out, iters, 0.999, 1e-3);
            cudaEventRecord(e1);
            cudaEventSynchronize(e1);
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        const double fl = (which == 0) ? 2.0 * 16 * iters * (double)blocks * threads : 2.0 * 256 * 8 * iters * (double)blocks * threads / 32;
        tflops[which] = fl / (best * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    return cudaGetLastError() == cudaSuccess ? PCE_OK : PCE_ECUDA;
}

// ---------------------------------------------------------------- test hook: poison shared memory
// Fills the whole dynamic shared memory of every SM with NaN bit patterns (several CTA waves of the largest size), so that a
// kernel of this library that reads shared memory it never wrote shows up as NaN in the next result instead of passing by luck.
__global__ void __launch_bounds__(256) k_poison_smem(int n_words, double* sink)
{
    extern __shared__ unsigned long long psm[];
    for (int i = threadIdx.x; i < n_words; i += blockDim.x) psm[i] = 0x7ff8dead0000beefull;
    __syncthreads();
    if (sink && psm[(threadIdx.x * 7) % n_words] == 1ull) sink[0] = 1.0;  // keeps the stores alive
}

extern "C" int pce_debug_poison_shared_memory(void* stream)
{
    int dev = 0, nsm = 0, max_smem = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess)
        return PCE_ECUDA;
    if (cudaFuncSetAttribute(k_poison_smem, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem) != cudaSuccess) return PCE_ECUDA;
    k_poison_smem<<<nsm * 4, 256, (size_t)max_smem, (cudaStream_t)stream>>>(max_smem / 8, nullptr);
    return cudaGetLastError() == cudaSuccess ? PCE_OK : PCE_ECUDA;
}
