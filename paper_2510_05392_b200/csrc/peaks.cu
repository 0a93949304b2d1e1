// peaks.cu -- micro-benchmarks for the roofline denominators that MEASURED_PEAKS.json lacks (SURVEY.md §8d:
// "FP64 FMA, FP32 FMA, mma.sync f64, tcgen05 TF32 ... the builder must measure them on the box").
// Each probe runs dependent-chain-free FMA (or MMA) loops on every SM and reports achieved TFLOP/s.
#include <stdint.h>

#include "../../include/mg5_b200.h"
#include "color_sum.cuh"

namespace mg {

template <typename T>
__global__ void __launch_bounds__(256) fma_probe(T* out, int iters, T seed)
{
    T a[16];
#pragma unroll
    for (int i = 0; i < 16; i++) a[i] = seed + T(threadIdx.x + i);
    const T b = T(1.0000001), c = T(1e-9);
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 16; i++) a[i] = a[i] * b + c;
    }
    T s = T(0);
#pragma unroll
    for (int i = 0; i < 16; i++) s += a[i];
    if (s == T(-1)) out[0] = s;      // never true: keeps the loop alive
}

__global__ void __launch_bounds__(256) dmma_probe(double* out, int iters)
{
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; i++) { c[i][0] = threadIdx.x; c[i][1] = i; }
    const double a = 1.0000001, b = 0.5;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
    if (s == -1.0) out[0] = s;
}

cudaError_t tf32_probe(double* tflops);   // color_sum_tf32.cu

cudaError_t measure_peak(int kind, double* tflops)
{
    if (kind == 3) return tf32_probe(tflops);
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    void* buf = nullptr;
    cudaError_t e = cudaMalloc(&buf, 64);
    if (e != cudaSuccess) return e;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0); cudaEventCreate(&t1);
    const int blocks = sms * 8, threads = 256, iters = 4096;
    double best = 0.0;
    for (int rep = 0; rep < 4; rep++) {
        cudaEventRecord(t0);
        if (kind == 0) fma_probe<double><<<blocks, threads>>>((double*)buf, iters, 1.0);
        else if (kind == 1) fma_probe<float><<<blocks, threads>>>((float*)buf, iters * 4, 1.0f);
        else dmma_probe<<<blocks, threads>>>((double*)buf, iters);
        cudaEventRecord(t1);
        e = cudaEventSynchronize(t1);
        if (e != cudaSuccess) break;
        float ms = 0;
        cudaEventElapsedTime(&ms, t0, t1);
        double flop;
        if (kind == 0) flop = 2.0 * 16 * iters * (double)blocks * threads;
        else if (kind == 1) flop = 2.0 * 16 * iters * 4 * (double)blocks * threads;
        else flop = 2.0 * 8 * 8 * 4 * 8.0 * iters * (double)blocks * (threads / 32);
        const double tf = flop / (ms * 1e-3) * 1e-12;
        if (tf > best) best = tf;
    }
    cudaEventDestroy(t0); cudaEventDestroy(t1);
    cudaFree(buf);
    if (e == cudaSuccess) e = cudaGetLastError();
    *tflops = best;
    return e;
}

}  // namespace mg

extern "C" int mg_measure_peak(int device, int kind, double* tflops)
{
    if (!tflops || kind < 0 || kind > 3) return MG_EINVAL;
    if (cudaSetDevice(device) != cudaSuccess) return MG_ENODEV;
    cudaError_t e = mg::measure_peak(kind, tflops);
    return e == cudaSuccess ? MG_OK : MG_ECUDA;
}
