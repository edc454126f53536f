// pn_bench.cu -- libpn_bench.so (include/pn_bench.h): pipe-peak probes for bench.py.  Not part of the product path.
#include "../../include/pn_bench.h"

#include <cuda_runtime.h>

namespace {

// register-only DFMA chains, 8 independent accumulators per thread
__global__ void __launch_bounds__(128) fp64_peak_kernel(double* out, int iters)
{
    double a[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) a[q] = threadIdx.x * 1e-9 + q;
    const double m = 1.0000001, c = 1e-9;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u)
#pragma unroll
            for (int q = 0; q < 8; ++q) a[q] = fma(a[q], m, c);
    }
    double s = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) s += a[q];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// the same with scalar FFMA (16 accumulators) ...
__global__ void __launch_bounds__(256) fp32_peak_kernel(float* out, int iters)
{
    float a[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) a[q] = threadIdx.x * 1e-6f + q;
    const float m = 1.0000001f, c = 1e-6f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int q = 0; q < 16; ++q) a[q] = fmaf(a[q], m, c);
    }
    float s = 0;
#pragma unroll
    for (int q = 0; q < 16; ++q) s += a[q];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// ... and with the packed form (sm_100: fma.rn.f32x2 on 64-bit register pairs): 16 x 2 accumulators
__global__ void __launch_bounds__(256) fp32x2_peak_kernel(float* out, int iters)
{
    unsigned long long a[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        const float lo = threadIdx.x * 1e-6f + q, hi = lo + 0.5f;
        asm("mov.b64 %0, {%1, %2};" : "=l"(a[q]) : "f"(lo), "f"(hi));
    }
    unsigned long long m, c;
    asm("mov.b64 %0, {%1, %1};" : "=l"(m) : "f"(1.0000001f));
    asm("mov.b64 %0, {%1, %1};" : "=l"(c) : "f"(1e-6f));
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int q = 0; q < 16; ++q) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(a[q]) : "l"(m), "l"(c));
    }
    float s = 0;
#pragma unroll
    for (int q = 0; q < 16; ++q) {
        float lo, hi;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a[q]));
        s += lo + hi;
    }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <typename T, typename Launch>
int time_probe(cudaStream_t st, size_t n_out, double flops_per_launch, Launch launch, double* tflops)
{
    T* out = nullptr;
    cudaEvent_t a = nullptr, b = nullptr;
    int rc = -2;
    float best_ms = 0;
    if (cudaMalloc(reinterpret_cast<void**>(&out), n_out * sizeof(T)) != cudaSuccess) goto done;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) goto done;
    launch(out, true);  // warm-up
    for (int rep = 0; rep < 3; ++rep) {
        if (cudaEventRecord(a, st) != cudaSuccess) goto done;
        launch(out, false);
        if (cudaEventRecord(b, st) != cudaSuccess || cudaEventSynchronize(b) != cudaSuccess) goto done;
        float ms = 0;
        if (cudaEventElapsedTime(&ms, a, b) != cudaSuccess || !(ms > 0)) goto done;
        if (best_ms == 0 || ms < best_ms) best_ms = ms;
    }
    if (cudaGetLastError() != cudaSuccess) goto done;
    *tflops = flops_per_launch / (best_ms * 1e-3) / 1e12;
    rc = 0;
done:
    if (a) cudaEventDestroy(a);
    if (b) cudaEventDestroy(b);
    if (out) cudaFree(out);
    if (rc) cudaGetLastError();
    return rc;
}

int sm_count()
{
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        cudaGetLastError();
        return 0;
    }
    return n;
}

}  // namespace

extern "C" {

int pn_bench_fp64_peak(void* stream, double* tflops)
{
    const int sms = sm_count();
    if (!tflops || sms < 1) return -2;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int blocks = sms * 8, iters = 8192;
    return time_probe<double>(st, (size_t)blocks * 128, (double)blocks * 128 * iters * 64 * 2,
                              [&](double* out, bool warm) { fp64_peak_kernel<<<blocks, 128, 0, st>>>(out, warm ? 64 : iters); }, tflops);
}

int pn_bench_fp32_peak(void* stream, int packed, double* tflops)
{
    const int sms = sm_count();
    if (!tflops || sms < 1) return -2;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int blocks = sms * 8, iters = 16384;
    const double fmas = (double)blocks * 256 * iters * 64 * (packed ? 2 : 1);
    if (packed)
        return time_probe<float>(st, (size_t)blocks * 256, fmas * 2,
                                 [&](float* out, bool warm) { fp32x2_peak_kernel<<<blocks, 256, 0, st>>>(out, warm ? 64 : iters); }, tflops);
    return time_probe<float>(st, (size_t)blocks * 256, fmas * 2,
                             [&](float* out, bool warm) { fp32_peak_kernel<<<blocks, 256, 0, st>>>(out, warm ? 64 : iters); }, tflops);
}

}  // extern "C"
