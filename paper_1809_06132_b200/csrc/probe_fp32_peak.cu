/*
 * probe_fp32_peak.cu -- bench-only measurement probe, built into its own shared object (libfsw_probe.so).
 * NOT part of the library's ABI (include/fsw.h) and not linked into libfsw.so: bench.py loads it to obtain the
 * denominator of the "alu" roofline, because MEASURED_PEAKS.json carries no FP32 figure.
 *
 * fsw_probe_fp32_peak runs 8 independent FFMA chains per thread (the plain FP32 FMA rate, 2 flop per FFMA) on
 * `cuda_stream` of `cuda_device`, times the best of three launches with CUDA events on that stream and returns the
 * rate in TFLOP/s and the kernel time in ms.  Returns 0 or the cudaError_t that failed.  Synchronizes the stream.
 */
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

__global__ void __launch_bounds__(256) ffma_peak_kernel(float* sink, int iters) {
    float x0 = threadIdx.x * 1e-3f, x1 = x0 + 1.f, x2 = x0 + 2.f, x3 = x0 + 3.f;
    float x4 = x0 + 4.f, x5 = x0 + 5.f, x6 = x0 + 6.f, x7 = x0 + 7.f;
    const float a = 0.999f, b = 1e-4f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
            x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
        }
    }
    float s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 123.456f) sink[0] = s; /* never true; keeps the chains alive */
}

}  // namespace

extern "C" int32_t fsw_probe_fp32_peak(int32_t cuda_device, void* cuda_stream, double* tflops, double* ms) {
    if (!tflops || !ms) return (int32_t)cudaErrorInvalidValue;
    int prev = -1;
    cudaError_t err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != cuda_device) err = cudaSetDevice(cuda_device);
    if (err != cudaSuccess) return (int32_t)err;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    cudaDeviceProp prop;
    float* sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    err = cudaGetDeviceProperties(&prop, cuda_device);
    if (err == cudaSuccess) err = cudaMalloc(&sink, 4);
    if (err == cudaSuccess) err = cudaEventCreate(&e0);
    if (err == cudaSuccess) err = cudaEventCreate(&e1);
    const int blocks = prop.multiProcessorCount * 8, iters = 4096;
    double best = 1e30;
    for (int rep = 0; rep < 4 && err == cudaSuccess; ++rep) { /* the first launch is a warm-up */
        cudaEventRecord(e0, stream);
        ffma_peak_kernel<<<blocks, 256, 0, stream>>>(sink, iters);
        err = cudaGetLastError();
        cudaEventRecord(e1, stream);
        if (err == cudaSuccess) err = cudaEventSynchronize(e1);
        float t = 0.f;
        if (err == cudaSuccess) err = cudaEventElapsedTime(&t, e0, e1);
        if (rep > 0 && t < best) best = t;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (sink) cudaFree(sink);
    if (prev >= 0 && prev != cuda_device) cudaSetDevice(prev);
    if (err != cudaSuccess) return (int32_t)err;
    const double flops = 2.0 * 8.0 * 16.0 * (double)iters * 256.0 * (double)blocks;
    *ms = best;
    *tflops = flops / (best * 1e-3) / 1e12;
    return 0;
}
