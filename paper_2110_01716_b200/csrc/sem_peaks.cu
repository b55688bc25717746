// sem_peaks.cu — register-resident arithmetic peaks of the device, measured in place ("~37 TFLOPS FP64
// peak ... measure it").  bench.py quotes the recomputed-G operator (a9, FP64-ALU bound) and the fast-diagonalisation
// local solve against these numbers, next to the HBM roofline.  Not part of the method: no input, no output but a rate.
//   SEM_PEAK_FMA_F64   dependent-chain-free DFMA stream, 16 accumulators per thread
//   SEM_PEAK_FMA_F32   same in FFMA
//   SEM_PEAK_DMMA_F64  mma.sync.m8n8k4.f64 (the tensor-core FP64 path; 256 FMA per warp instruction)
#include "sem_internal.h"

namespace {

template <typename T>
__global__ void __launch_bounds__(256) k_peak_fma(int iters, T seed, T* __restrict__ out) {
    T a[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) a[q] = seed + (T)(threadIdx.x + q);
    const T m = (T)0.999, c = (T)1e-3;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < 16; ++q) a[q] = a[q] * m + c;
    }
    T s = T(0);
#pragma unroll
    for (int q = 0; q < 16; ++q) s += a[q];
    if (s == (T)-1) out[0] = s;       // never true: keeps the chains alive
}

__global__ void __launch_bounds__(256) k_peak_dmma(int iters, double seed, double* __restrict__ out) {
    double c[4][2];
#pragma unroll
    for (int q = 0; q < 4; ++q) { c[q][0] = seed + threadIdx.x; c[q][1] = seed - q; }
    const double a = 0.5 + 1e-3 * (threadIdx.x & 3), b = 0.25 + 1e-3 * (threadIdx.x >> 2);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int q = 0; q < 4; ++q)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[q][0]), "+d"(c[q][1]) : "d"(a), "d"(b));
    }
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < 4; ++q) s += c[q][0] + c[q][1];
    if (s == -1.0) out[0] = s;
}

}  // namespace

extern "C" int sem_measure_peak(int kind, void* cuda_stream, double* tflops_out) {
    if (!tflops_out || kind < 0 || kind > 2) return SEM_EINVAL;
    *tflops_out = 0.0;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return SEM_ECUDA; }
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double* d_out = nullptr;
    if (cudaMalloc((void**)&d_out, 64) != cudaSuccess) { cudaGetLastError(); return SEM_ENOMEM; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int grid = sms * 8, threads = 256;
    const int iters = kind == SEM_PEAK_DMMA_F64 ? 4096 : 8192;
    // flops per launch: FMA = 2 flops; 16 chains per thread;  DMMA m8n8k4 = 256 FMA per warp, 4 per iteration
    const double flops = kind == SEM_PEAK_DMMA_F64 ? 2.0 * 256.0 * 4.0 * iters * (double)grid * (threads / 32)
                                                   : 2.0 * 16.0 * iters * (double)grid * threads;
    double best = 0.0;
    cudaError_t err = cudaSuccess;
    for (int rep = 0; rep < 6 && err == cudaSuccess; ++rep) {
        cudaEventRecord(e0, st);
        if (kind == SEM_PEAK_FMA_F64) k_peak_fma<double><<<grid, threads, 0, st>>>(iters, 1.0, d_out);
        else if (kind == SEM_PEAK_FMA_F32) k_peak_fma<float><<<grid, threads, 0, st>>>(iters, 1.0f, (float*)d_out);
        else k_peak_dmma<<<grid, threads, 0, st>>>(iters, 1.0, d_out);
        cudaEventRecord(e1, st);
        err = cudaEventSynchronize(e1);
        if (err == cudaSuccess) err = cudaGetLastError();
        float ms = 0.f;
        if (err == cudaSuccess) cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms > 0.f) {                     // the first launch is the warm-up
            const double tf = flops / (ms * 1e-3) / 1e12;
            if (tf > best) best = tf;
        }
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d_out);
    if (err != cudaSuccess) { cudaGetLastError(); return SEM_ECUDA; }
    *tflops_out = best;
    return SEM_OK;
}
