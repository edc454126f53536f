// pn_common.cuh -- records, constants and small helpers shared by every kernel file.
// Part of the sm_100a kernels of the limited-1PN hot path (arXiv:1801.07986); pn_kernels.cuh includes every part.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

namespace pn {


struct __align__(16) JRec {
    double x, y, z;  // stage position of star j
    double gm;       // G m_j
    double g15;      // 1.5   G m_j
    double g1875;    // 1.875 G m_j
};
static_assert(sizeof(JRec) == 48, "JRec must be 48 bytes");

struct BhState {
    double xs[3], vs[3];  // stage state
    double x0[3], v0[3];  // state at step start
    double sx[3], sv[3];  // weighted k sums
};

struct StepParams {
    double dt;
};

constexpr double kPadPos = 1e100;  // pad stars sit far away with zero mass: they add exactly 0 to every sum

// rsqrt seed: MUFU.RSQ64H (operates on the upper 32 bits; ~2^-21 relative error, low word of the result zero)
__device__ __forceinline__ double rsqrt_seed(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    return y;
}

}  // namespace pn
