// pn_noalloc.cu -- pn_bh_accel_noalloc (include/pn.h): the acceleration of the massive object, a_1 of Eqs. 2.1 + 2.2
// (PAPER.md:43-49), for callers that must not allocate device memory.
//
// Who this is for.  Everything else in libpn.so works on a pn_ctx, and pn_create calls cudaMalloc for its work buffers.
// Two kinds of caller cannot live with that:
//   * a program whose own memory pool already holds (nearly) all of the GPU's memory -- a simulation that reserves the
//     device at start-up, or a process that runs under a fixed memory quota next to other jobs: there a further cudaMalloc
//     simply fails;
//   * a time-critical loop (an integrator that must not stall, a control or analysis step between two launches of the
//     caller's own kernels): cudaMalloc and cudaFree stop the whole device until they return, which such a loop cannot
//     afford.
// For them this one call needs no context and allocates nothing: not with cudaMalloc, not with cudaFree, not through any
// library routine that allocates.  The caller passes every input and the output; the only extra global memory the kernel
// needs -- one partial sum of a_1 per thread block and the counter that tells the last block to add them up -- lives in
// the fixed array g_scratch below, which is part of the library image.
//
// What that costs and what the caller must know:
//   * g_scratch is kMaxBlocks x 3 doubles + 256 B = 98 560 B.  Every GPU on which a process uses this library holds that much
//     from the moment the library's code is loaded on it until the process exits, whether or not this entry point is ever called.
//   * That size fixes the limit: at most PN_NOALLOC_MAX_STARS = 2^20 stars (N - 1).  Larger N is refused with PN_EINVAL
//     and a message; nothing is launched.
//   * In host code the name g_scratch is only a handle for the array, not its device address.  The first call on each device looks the address
//     up (cudaGetSymbolAddress, with that device current) and keeps it; that look-up may make the CUDA runtime load
//     the library's code onto the device.  Make that first call during start-up, before any stream capture.  Later calls
//     on the same device only clear a counter and launch one kernel.
//   * All calls on one device share g_scratch and the array keeps what the last call left in it.  The block partials are
//     rewritten in full before they are read; the counter has to start from zero, so each call clears it on its stream ahead of
//     the kernel.  Two calls that run on the GPU at the same time (two streams, two host threads, two contexts of one
//     process) use the same partials and the same counter and give wrong results: order them yourself, e.g. by
//     issuing all of them on one stream.
//
// The arithmetic per star is that of star_physics() in pn_epilogue.cuh (the "BH <- star" half); the reduction is the
// same scheme as epilogue_kernel's (warp shuffles, block sum, the last block adds the block partials in index order), so a
// result does not depend on how the blocks were scheduled and repeats bit for bit.  Block size and therefore summation
// order differ from pn_accel's, so the two agree to rounding (1e-12 of |a_1| in the tests), not bitwise.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <mutex>

#include "pn.h"

namespace {

constexpr int kThreads = 256;                                       // one star per thread
constexpr int kMaxBlocks = PN_NOALLOC_MAX_STARS / kThreads;         // 4096
constexpr int kTicketOffset = 3 * kMaxBlocks;                       // in doubles; 96 KB into the array, 256-B aligned
constexpr int kScratchDoubles = kTicketOffset + 256 / (int)sizeof(double);
static_assert(PN_NOALLOC_MAX_STARS % kThreads == 0, "the star limit is a whole number of blocks");
static_assert((kTicketOffset * sizeof(double)) % 256 == 0, "the counter sits on its own 256-byte line");

// The scratch memory of bh_accel_noalloc_kernel: [kMaxBlocks][3] block partials of a_1, then the block counter
// (an unsigned int at the start of the last 256 bytes).  Host code must not pass this name to a kernel: see scratch_address().
static __device__ __align__(256) double g_scratch[kScratchDoubles];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
double* g_scratch_addr[kMaxDevices] = {};  // device address of g_scratch on each device, looked up once

__device__ __forceinline__ void block_sum3(double& a, double& b, double& c, double* smem /* 3 * kThreads/32 */)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, o);
        b += __shfl_down_sync(0xffffffffu, b, o);
        c += __shfl_down_sync(0xffffffffu, c, o);
    }
    constexpr int NW = kThreads / 32;
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) smem[w] = a, smem[NW + w] = b, smem[2 * NW + w] = c;
    __syncthreads();
    if (threadIdx.x == 0) {
        double sa = 0, sb = 0, sc = 0;
        for (int q = 0; q < NW; ++q) sa += smem[q], sb += smem[NW + q], sc += smem[2 * NW + q];
        a = sa, b = sb, c = sc;
    }
    __syncthreads();  // smem is reused by the final pass
}

// a_1 = sum_j (G m_j / r^3) { x - (1/c^2)[ (5 G M / r - 2 v_j^2 + (3/2)(v_j.x)^2 / r^2) x + 3 (v_j.x) v_j ] },
// x = x_j - x_1 (= -x_1j), r = |x|.   Eqs. 2.1 + 2.2, PAPER.md:43-49 (readings R1, R2).
// scratch: device address of g_scratch; the counter at scratch + kTicketOffset must be 0 on entry.
__global__ void __launch_bounds__(kThreads) bh_accel_noalloc_kernel(const double* __restrict__ mass, const double* __restrict__ pos,
                                                                    const double* __restrict__ vel, int n_stars, double G,
                                                                    double inv_c2, double* __restrict__ scratch,
                                                                    double* __restrict__ a1_out)
{
    __shared__ double red[3 * (kThreads / 32)];
    __shared__ bool is_last;
    const int j = blockIdx.x * kThreads + threadIdx.x;  // star j is body j + 1
    double b0 = 0, b1 = 0, b2 = 0;
    if (j < n_stars) {
        const double GM = G * mass[0];
        const double gm = G * mass[j + 1];
        const double* p = pos + 3 * (size_t)(j + 1);
        const double* w = vel + 3 * (size_t)(j + 1);
        const double x[3] = {p[0] - pos[0], p[1] - pos[1], p[2] - pos[2]};
        const double v[3] = {w[0], w[1], w[2]};
        const double r2 = x[0] * x[0] + x[1] * x[1] + x[2] * x[2];
        const double r = sqrt(r2);
        const double inv_r = 1.0 / r;
        const double inv_r3 = inv_r * inv_r * inv_r;
        const double v2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
        const double vx = v[0] * x[0] + v[1] * x[1] + v[2] * x[2];
        const double cb = gm * inv_r3;
        const double gx = 1.0 - inv_c2 * (5.0 * GM * inv_r - 2.0 * v2 + 1.5 * vx * vx * inv_r * inv_r);
        const double gv = -inv_c2 * 3.0 * vx;
        b0 = cb * (gx * x[0] + gv * v[0]);
        b1 = cb * (gx * x[1] + gv * v[1]);
        b2 = cb * (gx * x[2] + gv * v[2]);
    }
    block_sum3(b0, b1, b2, red);
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + kTicketOffset);
    if (threadIdx.x == 0) {
        double* bp = scratch + 3 * (size_t)blockIdx.x;
        bp[0] = b0, bp[1] = b1, bp[2] = b2;
        __threadfence();
        is_last = (atomicAdd(ticket, 1u) == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    // the last block to arrive adds the block partials: fixed thread <- block assignment, fixed tree afterwards
    double c0 = 0, c1 = 0, c2 = 0;
    for (int q = threadIdx.x; q < (int)gridDim.x; q += kThreads) {
        const volatile double* bp = scratch + 3 * (size_t)q;
        c0 += bp[0], c1 += bp[1], c2 += bp[2];
    }
    block_sum3(c0, c1, c2, red);
    if (threadIdx.x == 0) {
        a1_out[0] = c0, a1_out[1] = c1, a1_out[2] = c2;
        *ticket = 0;  // leave the counter ready; the next call clears it again anyway
    }
}

int fail(int code, char* errbuf, size_t len, const char* fmt, const char* a = "", long long b = 0, long long c = 0)
{
    if (errbuf && len) std::snprintf(errbuf, len, fmt, a, b, c);
    return code;
}

// Device address of g_scratch on the CURRENT device.  In host code `g_scratch` names a host-side stand-in for the device
// array; handing that to a kernel would make it fault or, on systems where the GPU can reach host memory, quietly work on
// the wrong memory.  cudaGetSymbolAddress gives the real address; it is asked once per device, with that device current.
cudaError_t scratch_address(double** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_scratch_addr[dev] = static_cast<double*>(p);
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" int pn_bh_accel_noalloc(int64_t N, const double* masses_dev, const double* pos_dev, const double* vel_dev, double G,
                                   double c, double* a1_dev, void* cuda_stream, char* errbuf_host, size_t errbuf_len)
{
    if (errbuf_host && errbuf_len) errbuf_host[0] = '\0';
    if (N < 2) return fail(PN_EINVAL, errbuf_host, errbuf_len, "pn_bh_accel_noalloc: N = %s%lld, need N >= 2 (the massive object and one star)", "", (long long)N);
    if (N - 1 > (int64_t)PN_NOALLOC_MAX_STARS)
        return fail(PN_EINVAL, errbuf_host, errbuf_len,
                    "pn_bh_accel_noalloc: %s%lld stars exceed PN_NOALLOC_MAX_STARS = %lld, the size of the library's fixed scratch array "
                    "(use a pn_ctx and pn_accel for larger systems)",
                    "", (long long)(N - 1), (long long)PN_NOALLOC_MAX_STARS);
    if (!masses_dev || !pos_dev || !vel_dev || !a1_dev) return fail(PN_EINVAL, errbuf_host, errbuf_len, "pn_bh_accel_noalloc: null %s", "pointer");
    if (!(G > 0.0) || !std::isfinite(G)) return fail(PN_EINVAL, errbuf_host, errbuf_len, "pn_bh_accel_noalloc: %s", "G must be positive and finite");
    if (!(c > 0.0)) return fail(PN_EINVAL, errbuf_host, errbuf_len, "pn_bh_accel_noalloc: %s", "c must be positive (+inf: Newtonian)");

    double* scratch = nullptr;
    cudaError_t e = scratch_address(&scratch);
    if (e != cudaSuccess) return fail(PN_ECUDA, errbuf_host, errbuf_len, "pn_bh_accel_noalloc: address of the scratch array: %s", cudaGetErrorString(e));

    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    const int n_stars = (int)(N - 1);
    const int grid = (n_stars + kThreads - 1) / kThreads;
    // The counter is the one thing in the shared array that must start at zero (an earlier launch that was aborted, or a
    // kernel that faulted, may have left it part-way).  A memset on the stream is not an allocation.
    e = cudaMemsetAsync(scratch + kTicketOffset, 0, 256, stream);
    if (e != cudaSuccess) return fail(PN_ECUDA, errbuf_host, errbuf_len, "pn_bh_accel_noalloc: clearing the block counter: %s", cudaGetErrorString(e));
    const double inv_c2 = std::isinf(c) ? 0.0 : 1.0 / (c * c);
    bh_accel_noalloc_kernel<<<grid, kThreads, 0, stream>>>(masses_dev, pos_dev, vel_dev, n_stars, G, inv_c2, scratch, a1_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(PN_ECUDA, errbuf_host, errbuf_len, "pn_bh_accel_noalloc: kernel launch: %s", cudaGetErrorString(e));
    return PN_OK;
}
