// pn_epilogue.cuh -- S2 - S4: per-star physics, partial-sum reduction, a_1 reduction, fused RK4 update; layout conversion.
// Part of the sm_100a kernels of the limited-1PN hot path (arXiv:1801.07986); pn_kernels.cuh includes every part.
#pragma once
#include "pn_common.cuh"
#include "pn_pair_cross.cuh"

namespace pn {

// ---------------------------------------------------------------------------------------------------------
// block-wide deterministic sum of three doubles (warp shuffle tree, then warp 0 sums the warp results in order)
// ---------------------------------------------------------------------------------------------------------
template <int NT>
__device__ __forceinline__ void block_sum3(double& a, double& b, double& c, double* smem /* 3 * NT/32 */)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, o);
        b += __shfl_down_sync(0xffffffffu, b, o);
        c += __shfl_down_sync(0xffffffffu, c, o);
    }
    constexpr int NW = NT / 32;
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) smem[w] = a, smem[NW + w] = b, smem[2 * NW + w] = c;
    __syncthreads();
    if (threadIdx.x == 0) {
        double sa = 0, sb = 0, sc = 0;
        for (int q = 0; q < NW; ++q) sa += smem[q], sb += smem[NW + q], sc += smem[2 * NW + q];
        a = sa, b = sb, c = sc;
    }
}

// ---------------------------------------------------------------------------------------------------------
// S2 + S3 + S4: per-star epilogue of one force evaluation.
//   a_i  = sum over j-chunk partials (fixed order) + BH -> star Newtonian + 1PN
//   a_1  = sum_i [star i -> BH, Newtonian + 1PN], block reduction + last-block fixed-order final sum
//   MODE_ACCEL: write acc[N][3] (acc[0] = a_1).
//   MODE_RK4 stage st: classical RK4 stage update fused onto the acceleration:
//       k_x = v_stage, k_v = a;  st 0: s = k;  st 1, 2: s += 2k;  next stage state = y0 + {dt/2, dt/2, dt} k;
//       st 3: y0 += dt/6 (s + k), next stage state = y0.
// ---------------------------------------------------------------------------------------------------------
// S2 + S3 (+ the O(N) parts of the Cross terms) for one star: x = x_i1 = x_i - x_1, vel = v_i, gm = G m_i, ss = the star's O(N^2)
// sums (a^SS; CROSS: + X (3), S, and U for CROSS = 2), csum = P (3), Q1, Q3, W (3).  Returns a_i in a and the star's share of
// a_1 in b.  Used by epilogue_kernel and by the small-system kernels.
template <int CROSS>
__device__ __forceinline__ void star_physics(double gm, const double (&x)[3], const double (&vel)[3], const double* ss,
                                             const double* __restrict__ csum, double GM, double inv_c2, double (&a)[3], double (&b)[3])
{
    const double r2 = x[0] * x[0] + x[1] * x[1] + x[2] * x[2];
    const double r = sqrt(r2);
    const double inv_r = 1.0 / r;
    const double inv_r3 = inv_r * inv_r * inv_r;
    const double v2 = vel[0] * vel[0] + vel[1] * vel[1] + vel[2] * vel[2];
    const double vx = vel[0] * x[0] + vel[1] * x[1] + vel[2] * x[2];
    const double GMr = GM * inv_r;
    // star <- BH: -GM x/r^3 + (1/c^2)(GM/r^3)[(4GM/r - v^2) x + 4 (v.x) v]
    const double cs = GM * inv_r3;
    const double fx = -1.0 + inv_c2 * (4.0 * GMr - v2);
    const double fv = inv_c2 * 4.0 * vx;
    // BH <- star (x_1j = -x): (G m/r^3){ x - (1/c^2)[(5GM/r - 2v^2 + 3/2 (v.x)^2/r^2) x + 3 (v.x) v] }
    const double cb = gm * inv_r3;
    const double gx = 1.0 - inv_c2 * (5.0 * GMr - 2.0 * v2 + 1.5 * vx * vx * inv_r * inv_r);
    const double gv = -inv_c2 * 3.0 * vx;
#pragma unroll
    for (int k = 0; k < 3; ++k) a[k] = ss[k] + cs * (fx * x[k] + fv * vel[k]);
#pragma unroll
    for (int k = 0; k < 3; ++k) b[k] = cb * (gx * x[k] + gv * vel[k]);
    if (CROSS) {
        // [a_i]_Cross = L0 + the O(N) parts of L1, L3, L4 (global sums minus this star's own term) + pair part
        const double P[3] = {csum[0] - gm * vel[0], csum[1] - gm * vel[1], csum[2] - gm * vel[2]};
        const double Q1 = csum[3] - gm * inv_r, Q3 = csum[4] - gm * inv_r3;
        const double W[3] = {csum[5] - gm * x[0] * inv_r3, csum[6] - gm * x[1] * inv_r3, csum[7] - gm * x[2] * inv_r3};
        const double vP = vel[0] * P[0] + vel[1] * P[1] + vel[2] * P[2];
        const double xP = x[0] * P[0] + x[1] * P[1] + x[2] * P[2];
        // coefficient of x_i1: L0 (5 G m_i GM / r^4 - 4 G m_i v^2 / r^3) + L1 (GM/r^3)(5/4 Q1 + r^2/4 Q3) - L4 4 (v.P)/r^3
        // + the pair part of L1, S / r^3 (S = sum_j G m_j (4 GM / rho_ij - GM rho_ij^2 / (4 r_j1^3)), 7th component)
        const double kx = inv_r3 * (5.0 * gm * GMr - 4.0 * gm * v2 + GM * (1.25 * Q1 + 0.25 * r2 * Q3) - 4.0 * vP + ss[6]);
        // coefficient of v_i: L0 7 G m_i (v.x)/r^3 + L4 3 (P.x)/r^3
        const double kv = inv_r3 * (7.0 * gm * vx + 3.0 * xP);
        const double kp = 4.0 * vx * inv_r3;  // L4: + 4 (v_i.x_i1) P / r^3
        const double kw = 3.5 * GM * inv_r;   // L3: + (7/2) GM W / r_i1
#pragma unroll
        for (int k = 0; k < 3; ++k) a[k] += inv_c2 * (ss[3 + k] + kx * x[k] + kv * vel[k] + kp * P[k] + kw * W[k]);
        if (CROSS == 2) {
            // this star's share of [a_1]_Cross (x_1j = -x): T0 + T1 along x, T2 along a_j^SS, T3 with the FULL sum P
            const double Pf[3] = {csum[0], csum[1], csum[2]};
            const double vPf = vel[0] * Pf[0] + vel[1] * Pf[1] + vel[2] * Pf[2];
            const double xPf = x[0] * Pf[0] + x[1] * Pf[1] + x[2] * Pf[2];
            const double gr3 = gm * inv_r3, g_M = gr3 / GM;
            const double tx = -(4.0 * gm * gr3 * inv_r + gr3 * (4.0 * Q1 + ss[CROSS == 2 ? 7 : 0])) + 4.0 * g_M * vPf;  // times x
            const double tP = -3.0 * g_M * vx;       // times P
            const double tv = -4.0 * g_M * xPf;      // times v_j
            const double ta = 3.5 * gm * inv_r;      // times a_j^SS
#pragma unroll
            for (int k = 0; k < 3; ++k) b[k] += inv_c2 * (tx * x[k] + tP * Pf[k] + tv * vel[k] + ta * ss[k]);
        }
    }
}

struct EpiArgs {
    JRec* jrec;           // stage positions (x, y, z updated in RK4 mode)
    double* v;            // [3][NP] stage velocity
    const double* part;   // [S][3][NP]
    double* x0;           // [3][NP]
    double* v0;           // [3][NP]
    double* sx;           // [3][NP]
    double* sv;           // [3][NP]
    BhState* bh;          // stage/step state of the massive object
    double* bh_part;      // [gridDim.x][3] per-block partial of a_1
    unsigned int* ticket; // last-block detection
    double* acc_out;      // MODE_ACCEL: [N][3]
    const StepParams* prm;
    int n_stars, np, n_split;
    double GM, inv_c2;
    const double* csum;   // CROSS: P (3), Q1, Q3, W (3) of cross_sum_kernel
};

enum { MODE_ACCEL = 0, MODE_RK4 = 1 };

constexpr int kEpiStars = 32;  // stars per epilogue block: lane = star, warp w sums the partial-sum slots w, w + NW, ...

// CROSS: the partial sums carry 7 components (a^SS, the pair part X of [a_i]_Cross, Eq. 2.6, and the scalar S of its line
// L1); the O(N) parts of the Cross term are added here (see the pair_cross kernels).
// CROSS = 2: additionally the star's share of [a_1]_Cross (Eq. 2.3), 8th component U.
template <int MODE, int NT, int CROSS>
__global__ void __launch_bounds__(NT) epilogue_kernel(EpiArgs A, int stage)
{
    constexpr int NW = NT / 32;
    constexpr int NC = CROSS == 2 ? 8 : (CROSS ? 7 : 3);
    __shared__ double red[3 * NW];
    __shared__ double wsum[NW][NC][kEpiStars];
    __shared__ bool is_last;
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int i = blockIdx.x * kEpiStars + lane;
    const int np = A.np;

    // fixed-order reduction of the partial-sum slots.  Every load is a coalesced 256 B row of one (slot, component);
    // 4 slots x 3 components are in flight per thread, so the O(S N) read runs at L2/HBM bandwidth, not latency.
    double ss[NC];
#pragma unroll
    for (int k = 0; k < NC; ++k) ss[k] = 0.0;
    if (i < A.n_stars) {
        constexpr int UN = CROSS ? 2 : 4;  // slots in flight per thread (12 - 16 loads)
        const size_t stride = (size_t)NW * NC * np;
        const double* p = A.part + (size_t)w * NC * np + i;
        int s = w;
        for (; s + (UN - 1) * NW < A.n_split; s += UN * NW, p += UN * stride) {
            double q[UN][NC];
#pragma unroll
            for (int u = 0; u < UN; ++u)
#pragma unroll
                for (int k = 0; k < NC; ++k) q[u][k] = __ldcg(p + u * stride + (size_t)k * np);
#pragma unroll
            for (int u = 0; u < UN; ++u)
#pragma unroll
                for (int k = 0; k < NC; ++k) ss[k] += q[u][k];
        }
        for (; s < A.n_split; s += NW, p += stride)
#pragma unroll
            for (int k = 0; k < NC; ++k) ss[k] += __ldcg(p + (size_t)k * np);
    }
#pragma unroll
    for (int k = 0; k < NC; ++k) wsum[w][k][lane] = ss[k];
    __syncthreads();
    if (w == 0) {
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            double t = wsum[0][k][lane];
#pragma unroll
            for (int q = 1; q < NW; ++q) t += wsum[q][k][lane];  // fixed order: warp 0, 1, ...
            ss[k] = t;
        }
    }
    const bool live = (w == 0) && (i < A.n_stars);

    double b0 = 0, b1 = 0, b2 = 0;  // this star's contribution to a_1
    double a[3] = {0, 0, 0}, vel[3] = {0, 0, 0};
    if (live) {
        const JRec rec = A.jrec[i];
        const double x[3] = {rec.x - A.bh->xs[0], rec.y - A.bh->xs[1], rec.z - A.bh->xs[2]};  // x_i1 = x_i - x_1
        vel[0] = A.v[i], vel[1] = A.v[np + i], vel[2] = A.v[2 * np + i];
        double bb[3];
        star_physics<CROSS>(rec.gm, x, vel, ss, A.csum, A.GM, A.inv_c2, a, bb);
        b0 = bb[0], b1 = bb[1], b2 = bb[2];
    }

    double hh = 0, dt = 0;
    if (MODE == MODE_RK4) {
        dt = A.prm->dt;
        hh = (stage == 2) ? dt : 0.5 * dt;
    }
    if (live) {
        if (MODE == MODE_ACCEL) {
            double* o = A.acc_out + 3 * (size_t)(i + 1);
            o[0] = a[0], o[1] = a[1], o[2] = a[2];
        } else {
            JRec* rec = A.jrec + i;
            double xn[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const size_t q = (size_t)k * np + i;
                const double kx = vel[k], kv = a[k];
                if (stage == 3) {
                    const double xnew = A.x0[q] + dt / 6.0 * (A.sx[q] + kx);
                    const double vnew = A.v0[q] + dt / 6.0 * (A.sv[q] + kv);
                    A.x0[q] = xnew, A.v0[q] = vnew;
                    xn[k] = xnew, A.v[q] = vnew;
                } else {
                    if (stage == 0) {
                        A.sx[q] = kx, A.sv[q] = kv;
                    } else {
                        A.sx[q] += 2.0 * kx, A.sv[q] += 2.0 * kv;
                    }
                    xn[k] = A.x0[q] + hh * kx;
                    A.v[q] = A.v0[q] + hh * kv;
                }
            }
            rec->x = xn[0], rec->y = xn[1], rec->z = xn[2];
        }
    }

    // ---- a_1: block partial, then the last block to finish adds the block partials in index order
    block_sum3<NT>(b0, b1, b2, red);
    if (threadIdx.x == 0) {
        double* bp = A.bh_part + 3 * (size_t)blockIdx.x;
        bp[0] = b0, bp[1] = b1, bp[2] = b2;
        __threadfence();
        const unsigned int t = atomicAdd(A.ticket, 1u);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (!is_last) return;
    __threadfence();
    double c0 = 0, c1 = 0, c2 = 0;
    // fixed assignment of block partials to threads, fixed tree afterwards: deterministic
    for (int q = threadIdx.x; q < (int)gridDim.x; q += NT) {
        const volatile double* bp = A.bh_part + 3 * (size_t)q;
        c0 += bp[0], c1 += bp[1], c2 += bp[2];
    }
    __syncthreads();
    block_sum3<NT>(c0, c1, c2, red);
    if (threadIdx.x == 0) {
        *A.ticket = 0;
        const double a1[3] = {c0, c1, c2};
        BhState* bh = A.bh;
        if (MODE == MODE_ACCEL) {
            A.acc_out[0] = a1[0], A.acc_out[1] = a1[1], A.acc_out[2] = a1[2];
        } else {
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const double kx = bh->vs[k], kv = a1[k];
                if (stage == 3) {
                    bh->x0[k] += dt / 6.0 * (bh->sx[k] + kx);
                    bh->v0[k] += dt / 6.0 * (bh->sv[k] + kv);
                    bh->xs[k] = bh->x0[k], bh->vs[k] = bh->v0[k];
                } else {
                    if (stage == 0) {
                        bh->sx[k] = kx, bh->sv[k] = kv;
                    } else {
                        bh->sx[k] += 2.0 * kx, bh->sv[k] += 2.0 * kv;
                    }
                    bh->xs[k] = bh->x0[k] + hh * kx;
                    bh->vs[k] = bh->v0[k] + hh * kv;
                }
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// Layout conversion: user AoS [N][3] <-> internal records.  to_state: also initialise x0, v0 and the BH state.
// ---------------------------------------------------------------------------------------------------------
__global__ void pack_kernel(const double* __restrict__ pos, const double* __restrict__ vel, JRec* jrec, double* v,
                            double* x0, double* v0, BhState* bh, int n_stars, int np, int to_state)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_stars) {
        const double* p = pos + 3 * (size_t)(i + 1);
        const double* w = vel + 3 * (size_t)(i + 1);
        JRec* r = jrec + i;
        r->x = p[0], r->y = p[1], r->z = p[2];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            v[(size_t)k * np + i] = w[k];
            if (to_state) x0[(size_t)k * np + i] = p[k], v0[(size_t)k * np + i] = w[k];
        }
    }
    if (i == 0) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            bh->xs[k] = pos[k], bh->vs[k] = vel[k];
            if (to_state) bh->x0[k] = pos[k], bh->v0[k] = vel[k], bh->sx[k] = 0, bh->sv[k] = 0;
        }
    }
}

__global__ void unpack_kernel(const double* __restrict__ x0, const double* __restrict__ v0, const BhState* bh,
                              double* __restrict__ pos, double* __restrict__ vel, int n_stars, int np)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n_stars) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            pos[3 * (size_t)(i + 1) + k] = x0[(size_t)k * np + i];
            vel[3 * (size_t)(i + 1) + k] = v0[(size_t)k * np + i];
        }
    }
    if (i == 0) {
#pragma unroll
        for (int k = 0; k < 3; ++k) pos[k] = bh->x0[k], vel[k] = bh->v0[k];
    }
}

}  // namespace pn
