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

// ---- operand-bandwidth probes behind the kernel design of DESIGN.md section 6.1 ---------------------------------------
// A stream of DFMAs (16 per loop trip, issue limit 2 cycles per warp instruction and sub-partition) in one-warp blocks, 12 per
// SM (the residency of the one-warp pair kernel).  The inline assembly is volatile, so ptxas keeps the order written here.
#define PROBE_FMA(d, a, b, c) asm volatile("fma.rn.f64 %0, %1, %2, %3;" : "=d"(d) : "d"(a), "d"(b), "d"(c))
#define PROBE_MUL(d, a, b) asm volatile("mul.rn.f64 %0, %1, %2;" : "=d"(d) : "d"(a), "d"(b))

// kind 0: FP64 operand patterns (mode), kind 1: a 2-register DFMA stream with nx other-pipe instructions per 16 DFMA (mode)
template <int KIND, int MODE, int NX>
__global__ void __launch_bounds__(32, 12) operand_probe_kernel(double* out, const double* in, int* iout, int iters)
{
    __shared__ double4 sm[64];
    double d[8], K[8], nK[8], a[8], b[8];
    int x[8], y[8], z[8];
    const unsigned lane = threadIdx.x, nxt = (lane + 1) & 31;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        d[q] = in[q + threadIdx.x], K[q] = in[64 + q + threadIdx.x], nK[q] = -K[q], a[q] = in[128 + q], b[q] = in[136 + q];
        x[q] = (int)in[144 + q] + q, y[q] = (int)in[152 + q] + 2 * q, z[q] = (int)in[160 + q] + 3 * q;
    }
    sm[lane] = make_double4(0, 0, 0, 0), sm[lane + 32] = make_double4(0, 0, 0, 0);
    __syncwarp();
#pragma unroll 1
    for (int it = 0; it < iters; ++it) {
        if (KIND == 0) {
            if (MODE == 0) {  // 2 distinct register operands
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    PROBE_FMA(a[q], d[q], d[q], a[q]);
                    PROBE_FMA(b[q], K[q], K[q], b[q]);
                }
            } else if (MODE == 1) {  // 3 distinct register operands, nothing shared by neighbours
#pragma unroll
                for (int q = 0; q < 8; ++q) PROBE_FMA(a[q], d[q], K[q], a[q]);
#pragma unroll
                for (int q = 0; q < 8; ++q) PROBE_FMA(b[q], K[q], d[(q + 1) & 7], b[q]);
            } else if (MODE == 2) {  // the accumulation pairs of the symmetric kernel: a += K d (3 reads), b -= K d (d, K reused)
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    PROBE_FMA(a[q], d[q], K[q], a[q]);
                    PROBE_FMA(b[q], d[q], nK[q], b[q]);
                }
            } else if (MODE == 3) {  // a 3-register DFMA next to a genuine 1-register instruction
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    PROBE_FMA(a[q], d[q], K[q], a[q]);
                    PROBE_MUL(b[q], b[q], b[q]);
                }
            } else {  // 1, 1, 3, 3
#pragma unroll
                for (int q = 0; q < 8; q += 2) {
                    PROBE_MUL(b[q], b[q], b[q]);
                    PROBE_MUL(b[q + 1], b[q + 1], b[q + 1]);
                    PROBE_FMA(a[q], d[q], K[q], a[q]);
                    PROBE_FMA(a[q + 1], d[q + 1], K[q + 1], a[q + 1]);
                }
            }
        } else {
#pragma unroll
            for (int q = 0; q < 8; ++q) {
                PROBE_FMA(a[q], d[q], d[q], a[q]);
                if (q < NX) {
                    if (MODE == 1) asm volatile("shfl.sync.idx.b32 %0, %1, %2, 0x1f, 0xffffffff;" : "=r"(x[q]) : "r"(x[q]), "r"(nxt));
                    if (MODE == 2) asm volatile("shfl.sync.bfly.b32 %0, %1, 1, 0x1f, 0xffffffff;" : "=r"(x[q]) : "r"(x[q]));
                    if (MODE == 3) asm volatile("mad.lo.s32 %0, %1, %2, %3;" : "=r"(x[q]) : "r"(y[q]), "r"(z[q]), "r"(x[q]));
                    if (MODE == 4) asm volatile("mov.b32 %0, 0;" : "=r"(x[q]));
                    if (MODE == 5) asm volatile("and.b32 %0, %1, 31;" : "=r"(x[q]) : "r"(x[q]));
                    if (MODE == 6) asm volatile("add.f32 %0, %1, %2;" : "=r"(x[q]) : "r"(x[q]), "r"(y[q]));
                    if (MODE == 7) {
                        const double4 v = sm[(lane + q) & 63];
                        asm volatile("" ::"d"(v.x), "d"(v.y), "d"(v.z), "d"(v.w));
                    }
                }
                PROBE_FMA(b[q], b[q], d[q], b[q]);
            }
        }
    }
    double s = 0;
    int si = 0;
#pragma unroll
    for (int q = 0; q < 8; ++q) s += a[q] + b[q], si += x[q];
    out[blockIdx.x * 32 + threadIdx.x] = s;
    iout[blockIdx.x * 32 + threadIdx.x] = si;
}

typedef void (*probe_fn)(double*, const double*, int*, int);

template <int KIND, int MODE, int NX>
probe_fn probe_ptr()
{
    return operand_probe_kernel<KIND, MODE, NX>;
}

probe_fn pick_probe(int kind, int mode, int nx)
{
    if (kind == 0) {
        switch (mode) {
            case 0: return probe_ptr<0, 0, 0>();
            case 1: return probe_ptr<0, 1, 0>();
            case 2: return probe_ptr<0, 2, 0>();
            case 3: return probe_ptr<0, 3, 0>();
            case 4: return probe_ptr<0, 4, 0>();
            default: return nullptr;
        }
    }
    if (nx != 0 && nx != 4 && nx != 8) return nullptr;
    if (nx == 0) return probe_ptr<1, 0, 0>();
#define PICK(M) \
    case M: return nx == 4 ? probe_ptr<1, M, 4>() : probe_ptr<1, M, 8>();
    switch (mode) {
        PICK(1) PICK(2) PICK(3) PICK(4) PICK(5) PICK(6) PICK(7)
        default: return nullptr;
    }
#undef PICK
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

int pn_bench_operand_probe(void* stream, int kind, int mode, int nx, double* cycles)
{
    const int sms = sm_count();
    probe_fn fn = pick_probe(kind, mode, nx);
    if (!cycles || sms < 1 || !fn) return -2;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int dev = 0, khz = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev) != cudaSuccess) return -2;
    const int blocks = sms * 12, iters = 1 << 16;
    double *out = nullptr, *in = nullptr;
    int* iout = nullptr;
    cudaEvent_t a = nullptr, b = nullptr;
    int rc = -2;
    float best = 0;
    if (cudaMalloc(reinterpret_cast<void**>(&out), (size_t)blocks * 32 * 8) != cudaSuccess) goto done;
    if (cudaMalloc(reinterpret_cast<void**>(&iout), (size_t)blocks * 32 * 4) != cudaSuccess) goto done;
    if (cudaMalloc(reinterpret_cast<void**>(&in), 256 * 8) != cudaSuccess || cudaMemsetAsync(in, 0, 256 * 8, st) != cudaSuccess) goto done;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) goto done;
    fn<<<blocks, 32, 0, st>>>(out, in, iout, 64);
    for (int rep = 0; rep < 3; ++rep) {
        if (cudaEventRecord(a, st) != cudaSuccess) goto done;
        fn<<<blocks, 32, 0, st>>>(out, in, iout, iters);
        if (cudaEventRecord(b, st) != cudaSuccess || cudaEventSynchronize(b) != cudaSuccess) goto done;
        float ms = 0;
        if (cudaEventElapsedTime(&ms, a, b) != cudaSuccess || !(ms > 0)) goto done;
        if (best == 0 || ms < best) best = ms;
    }
    if (cudaGetLastError() != cudaSuccess) goto done;
    // 16 DFMA per trip and warp, 3 warps per sub-partition: SM cycles per DFMA and sub-partition at the device's rated clock
    *cycles = best * 1e-3 * (khz * 1e3) / (16.0 * iters) / 3.0;
    rc = 0;
done:
    if (a) cudaEventDestroy(a);
    if (b) cudaEventDestroy(b);
    cudaFree(out), cudaFree(iout), cudaFree(in);
    if (rc) cudaGetLastError();
    return rc;
}

}  // extern "C"
