// pn_small.cuh -- S1 - S4 for small systems: a whole pn_step / pn_accel call in one cooperative launch (hot path, Cross terms).
// Part of the sm_100a kernels of the limited-1PN hot path (arXiv:1801.07986); pn_kernels.cuh includes every part.
#pragma once
#include "pn_common.cuh"
#include "pn_pair_fp64.cuh"
#include "pn_pair_cross.cuh"
#include "pn_epilogue.cuh"

namespace pn {

// ---------------------------------------------------------------------------------------------------------
// S1 - S4 for small systems (N_s < 3072, where a force evaluation is a few microseconds of arithmetic and the multi-kernel
// path is bound by launch latency): ONE cooperative launch runs a whole pn_step call (every stage of every RK4 step) or
// one pn_accel.  Each warp of the grid owns IW consecutive i-stars for the whole launch; its lanes share out the j-stars
// (lane l takes j = l, l + 32, ...: every ordered pair, the 15-instruction form of pair_fp64_kernel), a butterfly
// reduction gives every lane the complete sums, and lane k < IW then does the per-star physics of star k (S2, S3) and its
// RK4 stage update (S4) with that star's step state held in registers.  What the other blocks need of an evaluation --
// the new stage positions and one a_1 partial per warp -- goes through global memory, followed by one grid-wide barrier
// per evaluation (an atomic arrival counter; the launch is cooperative, so every block is resident).  After the barrier
// every block copies the stage records into its shared memory and forms a_1 from the per-warp partials in the same fixed
// order (so every block integrates the massive object identically); block 0 writes its state back at the end.
// Every sum has a fixed order: results are bit-reproducible.
// ---------------------------------------------------------------------------------------------------------
struct SmallArgs {
    JRec* jrec[2];       // stage records: evaluation e reads set e & 1 and writes the next stage positions into the other
    double* v;           // [3][np] stage velocity
    double *x0, *v0, *sx, *sv;
    BhState* bh;
    double* bh_part;     // [2][warps of the grid][3]: evaluation e writes set e & 1
    unsigned int* bar;   // [2]: arrival counter of the grid barrier (monotonic; bar_base = its value at launch), give-up flag
    unsigned int* host_flag;  // mapped host word, set together with the give-up flag: the host sees it without a copy
    double* acc_out;     // MODE_ACCEL: [N][3]
    int n_stars, np;
    double GM, inv_c2, eps2, dt;
    long long nsteps;
    unsigned int bar_base;
};

// TMA bulk copy (cp.async.bulk, global -> shared, completion on an mbarrier): one thread moves a whole contiguous array
// into shared memory without staging it through registers; the data comes from L2, never from a stale L1 line
__device__ __forceinline__ unsigned int smem_u32(const void* p) { return (unsigned int)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void bulk_copy_g2s(void* dst_smem, const void* src_gmem, unsigned int bytes, unsigned long long* bar)
{
    asm volatile("fence.proxy.async;" ::: "memory");  // earlier generic-proxy accesses are ordered before the async-proxy copy
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned int parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\tMBAR_WAIT:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@!p bra MBAR_WAIT;\n\t}" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}

constexpr int kSmallNT = 128;  // threads per block of small_path_kernel (one warp per SM sub-partition)

// ctr[0]: arrivals (monotonic); ctr[1]: set if a wait ever gave up.  The wait is bounded (about half a minute of polling) so
// that a broken invariant -- blocks not all resident, a counter out of step with the host's copy -- ends in an error the host
// reports (pn_api.cu: small_check) instead of a hung device.  The bound holds for the whole LAUNCH, not per barrier: a waiting
// block also looks at the give-up flag (every 1024 polls), and the barrier returns false to every thread of a block that gave
// up or saw the flag; the kernels then return at once, without another barrier and without writing any state back.
__device__ __forceinline__ bool small_grid_barrier(unsigned int* ctr, unsigned int target, unsigned int* s_abort /* shared */,
                                                   unsigned int* host_flag /* mapped host memory */)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();  // this block's global writes are visible before its arrival is
        atomicAdd(ctr, 1u);
        unsigned int seen, polls = 0, abort = 0;
        for (;;) {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(ctr) : "memory");
            if ((int)(seen - target) >= 0) break;
            ++polls;
            if ((polls & 1023u) == 0) {
                asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(abort) : "l"(ctr + 1) : "memory");
                if (abort) break;  // another block gave up: it will never arrive
            }
            if (polls == (1u << 26)) {
                atomicExch(ctr + 1, 1u);
                *reinterpret_cast<volatile unsigned int*>(host_flag) = 1u;  // the next API call on the context reports it
                __threadfence_system();
                abort = 1;
                break;
            }
        }
        *s_abort = abort;
    }
    __syncthreads();
    return *s_abort == 0;
}

template <int MODE, int IW, int JU, bool MASK>
__global__ void __launch_bounds__(kSmallNT, 1) small_path_kernel(SmallArgs A)
{
    extern __shared__ double2 small_smem[];              // JRec[np]: this block's copy of the stage records
    JRec* sj = reinterpret_cast<JRec*>(small_smem);
    __shared__ double red[3 * (kSmallNT / 32)];
    __shared__ BhState sbh;
    __shared__ __align__(8) unsigned long long fill_bar;  // completion of the bulk copy of the stage records
    __shared__ unsigned int bar_abort;                    // small_grid_barrier: this block gave up / saw the give-up flag
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int np = A.np;
    const int gw = blockIdx.x * (kSmallNT / 32) + w;     // warp of the grid
    const int i0 = gw * IW;                              // its first i-star
    const int my = i0 + lane;                            // lane k < IW owns star i0 + k
    const bool own = (lane < IW) && (my < A.n_stars);
    unsigned int target = A.bar_base;

    double x0[3] = {0, 0, 0}, v0[3] = {0, 0, 0}, vs[3] = {0, 0, 0}, sx[3] = {0, 0, 0}, sv[3] = {0, 0, 0}, gm_me = 0;
    if (own) {
        gm_me = A.jrec[0][my].gm;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const size_t q = (size_t)k * np + my;
            vs[k] = A.v[q];
            if (MODE == MODE_RK4) x0[k] = A.x0[q], v0[k] = A.v0[q], sx[k] = A.sx[q], sv[k] = A.sv[q];
        }
    }
    if (tid == 0) {
        sbh = *A.bh;
        mbar_init(&fill_bar, 1);
    }
    __syncthreads();

    // a_1 of an evaluation from the per-warp partials (fixed order), then the massive object's RK4 stage update
    const int n_part = (int)gridDim.x * (kSmallNT / 32);
    auto finish_bh = [&](long long e) {  // e: the evaluation whose a_1 is formed
        const int stage = (int)(e & 3);
        const double* part = A.bh_part + (size_t)(e & 1) * 3 * n_part;
        double c0 = 0, c1 = 0, c2 = 0;
        for (int q = tid; q < n_part; q += kSmallNT) {
            c0 += __ldcg(part + 3 * q), c1 += __ldcg(part + 3 * q + 1), c2 += __ldcg(part + 3 * q + 2);
        }
        __syncthreads();  // red is free again
        block_sum3<kSmallNT>(c0, c1, c2, red);
        if (tid == 0) {
            const double a1[3] = {c0, c1, c2};
            if (MODE == MODE_ACCEL) {
                if (blockIdx.x == 0) A.acc_out[0] = a1[0], A.acc_out[1] = a1[1], A.acc_out[2] = a1[2];
            } else {
                const double dt = A.dt, hh = (stage == 2) ? dt : 0.5 * dt;
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    const double kx = sbh.vs[k], kv = a1[k];
                    if (stage == 3) {
                        sbh.x0[k] += dt / 6.0 * (sbh.sx[k] + kx);
                        sbh.v0[k] += dt / 6.0 * (sbh.sv[k] + kv);
                        sbh.xs[k] = sbh.x0[k], sbh.vs[k] = sbh.v0[k];
                    } else {
                        if (stage == 0) {
                            sbh.sx[k] = kx, sbh.sv[k] = kv;
                        } else {
                            sbh.sx[k] += 2.0 * kx, sbh.sv[k] += 2.0 * kv;
                        }
                        sbh.xs[k] = sbh.x0[k] + hh * kx;
                        sbh.vs[k] = sbh.v0[k] + hh * kv;
                    }
                }
            }
        }
    };

    const long long n_eval = (MODE == MODE_RK4) ? 4 * A.nsteps : 1;
    for (long long ev = 0; ev < n_eval; ++ev) {
        const int stage = (int)(ev & 3);
        // (A) the stage records of all stars -> shared memory: one TMA bulk copy (other blocks wrote them before the barrier)
        if (tid == 0) bulk_copy_g2s(small_smem, A.jrec[ev & 1], (unsigned int)(np * sizeof(JRec)), &fill_bar);
        // (B) meanwhile, the massive object's stage state: a_1 of the previous evaluation
        if (ev > 0) finish_bh(ev - 1);
        mbar_wait(&fill_bar, (unsigned int)(ev & 1));
        __syncthreads();

        // (C) every ordered pair (i, j) of this warp's IW i-stars: lane l takes j = l + 32 q
        double xi[IW], yi[IW], zi[IW], ax[IW], ay[IW], az[IW];
        int ii[IW];
#pragma unroll
        for (int k = 0; k < IW; ++k) {
            ii[k] = i0 + k;
            const JRec* pi = sj + min(ii[k], np - 1);  // beyond the padded range: a pad star, result unused
            xi[k] = pi->x, yi[k] = pi->y, zi[k] = pi->z;
            ax[k] = ay[k] = az[k] = 0.0;
        }
#pragma unroll 1
        for (int jq = lane; jq < np; jq += 32 * JU) pairs_fp64<IW, JU, MASK, 32>(sj, jq, jq, xi, yi, zi, ii, ax, ay, az, A.eps2);
        double s0 = 0, s1 = 0, s2 = 0;
#pragma unroll
        for (int k = 0; k < IW; ++k) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                ax[k] += __shfl_xor_sync(0xffffffffu, ax[k], o);
                ay[k] += __shfl_xor_sync(0xffffffffu, ay[k], o);
                az[k] += __shfl_xor_sync(0xffffffffu, az[k], o);
            }
            if (lane == k) s0 = ax[k], s1 = ay[k], s2 = az[k];
        }

        // S2 + S3 + S4 for the lane's own star (same formulas as epilogue_kernel)
        double b0 = 0, b1 = 0, b2 = 0;
        if (own) {
            const JRec rec = sj[my];
            const double x[3] = {rec.x - sbh.xs[0], rec.y - sbh.xs[1], rec.z - sbh.xs[2]};  // x_i1 = x_i - x_1
            const double ss[3] = {s0, s1, s2};
            double a[3], bb[3];
            star_physics<0>(gm_me, x, vs, ss, nullptr, A.GM, A.inv_c2, a, bb);
            b0 = bb[0], b1 = bb[1], b2 = bb[2];
            if (MODE == MODE_ACCEL) {
                double* o = A.acc_out + 3 * (size_t)(my + 1);
                o[0] = a[0], o[1] = a[1], o[2] = a[2];
            } else {
                const double dt = A.dt, hh = (stage == 2) ? dt : 0.5 * dt;
                double xn[3];
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    const double kx = vs[k], kv = a[k];
                    if (stage == 3) {
                        x0[k] = x0[k] + dt / 6.0 * (sx[k] + kx);
                        v0[k] = v0[k] + dt / 6.0 * (sv[k] + kv);
                        xn[k] = x0[k], vs[k] = v0[k];
                    } else {
                        if (stage == 0) {
                            sx[k] = kx, sv[k] = kv;
                        } else {
                            sx[k] += 2.0 * kx, sv[k] += 2.0 * kv;
                        }
                        xn[k] = x0[k] + hh * kx;
                        vs[k] = v0[k] + hh * kv;
                    }
                }
                JRec* g = A.jrec[(ev + 1) & 1] + my;  // the next evaluation's stage position, for every block
                g->x = xn[0], g->y = xn[1], g->z = xn[2];
            }
        }
        // this warp's a_1 partial: its stars in index order
        {
            double p0 = 0, p1 = 0, p2 = 0;
#pragma unroll
            for (int k = 0; k < IW; ++k) {
                p0 += __shfl_sync(0xffffffffu, b0, k);
                p1 += __shfl_sync(0xffffffffu, b1, k);
                p2 += __shfl_sync(0xffffffffu, b2, k);
            }
            if (lane == 0) {
                double* bp = A.bh_part + (size_t)(ev & 1) * 3 * n_part + 3 * (size_t)gw;
                bp[0] = p0, bp[1] = p1, bp[2] = p2;
            }
        }
        // (D) everything of this evaluation is in global memory before anyone starts the next one
        target += gridDim.x;
        if (!small_grid_barrier(A.bar, target, &bar_abort, A.host_flag)) return;  // timed out: the host reports it (small_check)
    }
    finish_bh(n_eval - 1);
    __syncthreads();
    if (MODE == MODE_RK4) {
        if (blockIdx.x == 0 && tid == 0) *A.bh = sbh;
        if (own) {
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const size_t q = (size_t)k * np + my;
                A.v[q] = vs[k], A.x0[q] = x0[k], A.v0[q] = v0[k], A.sx[q] = sx[k], A.sv[q] = sv[k];
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------
// The small-system path with the Cross terms (Eqs. 2.6 and 2.3; N_s <= kSmallCrossMaxStars): the same one-launch scheme as
// small_path_kernel.  What the blocks exchange per evaluation is the stage position AND velocity of every star (48 B, two
// buffers by evaluation parity); from them every block builds, for itself and in the same order, the per-star records of the
// Cross kernels (CRec) and the eight global sums P, Q1, Q3, W in shared memory -- redundant O(N) work instead of a second grid
// barrier.  Every ordered pair (cross_pair, j != i by index), lanes share out the j-stars, 7 or 8 sums per i-star.
// ---------------------------------------------------------------------------------------------------------
struct __align__(16) XVRec {
    double x, y, z, vx, vy, vz;  // stage position and velocity of a star
};
static_assert(sizeof(XVRec) == 48, "XVRec must be 48 bytes");

struct SmallCrossArgs {
    const JRec* jrec_in;  // positions of the state the launch starts from (and G m of every star)
    JRec* jrec_out;       // MODE_RK4: the integrator's stage records, positions written back at the end
    double* v;            // [3][np] stage velocity (read at the start, MODE_RK4: written at the end)
    double *x0, *v0, *sx, *sv;
    BhState* bh;
    XVRec* xv;            // [2][np]: evaluation e >= 1 reads set e & 1, evaluation e writes set (e + 1) & 1
    double* bh_part;      // [2][warps of the grid][3]
    unsigned int* bar;
    unsigned int* host_flag;  // as in SmallArgs
    double* acc_out;
    int n_stars, np;
    double GM, inv_c2, eps2, dt;
    long long nsteps;
    unsigned int bar_base;
};

constexpr int kSmallCrossMaxStars = 1279;                                   // np <= 1280
constexpr int kSmallCrossBytesPerStar = (int)(sizeof(XVRec) + sizeof(CRec) + 8);  // staged exchange record + CRec + G m

template <int MODE, int IW, bool BHX>
__global__ void __launch_bounds__(kSmallNT, 1) small_cross_kernel(SmallCrossArgs A)
{
    constexpr int CROSS = BHX ? 2 : 1;
    constexpr int NW = kSmallNT / 32;
    extern __shared__ double2 small_smem[];
    const int np = A.np;
    XVRec* sxv = reinterpret_cast<XVRec*>(small_smem);                    // [np] this evaluation's stage state of every star
    CRec* scr = reinterpret_cast<CRec*>(small_smem + 3 * (size_t)np);     // [np] Cross records
    double* sgm = reinterpret_cast<double*>(small_smem + 10 * (size_t)np); // [np] G m
    __shared__ double red[kCrossSums][NW];
    __shared__ double red3[3 * NW];
    __shared__ double scsum[kCrossSums];
    __shared__ BhState sbh;
    __shared__ __align__(8) unsigned long long fill_bar;
    __shared__ unsigned int bar_abort;
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    const int gw = blockIdx.x * NW + w;
    const int i0 = gw * IW;
    const int my = i0 + lane;
    const bool own = (lane < IW) && (my < A.n_stars);
    const double GM4 = 4.0 * A.GM;
    unsigned int target = A.bar_base;

    double x0[3] = {0, 0, 0}, v0[3] = {0, 0, 0}, sx[3] = {0, 0, 0}, sv[3] = {0, 0, 0};
    if (own && MODE == MODE_RK4) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const size_t q = (size_t)k * np + my;
            x0[k] = A.x0[q], v0[k] = A.v0[q], sx[k] = A.sx[q], sv[k] = A.sv[q];
        }
    }
    for (int q = tid; q < np; q += kSmallNT) {  // G m of every star; evaluation 0's stage state straight from the caller's arrays
        const JRec r = A.jrec_in[q];
        sgm[q] = r.gm;
        XVRec o;
        o.x = r.x, o.y = r.y, o.z = r.z;
        o.vx = A.v[q], o.vy = A.v[np + q], o.vz = A.v[2 * (size_t)np + q];
        sxv[q] = o;
    }
    if (tid == 0) {
        sbh = *A.bh;
        mbar_init(&fill_bar, 1);
    }
    __syncthreads();

    const int n_part = (int)gridDim.x * NW;
    auto finish_bh = [&](long long e) {
        const int stage = (int)(e & 3);
        const double* part = A.bh_part + (size_t)(e & 1) * 3 * n_part;
        double c0 = 0, c1 = 0, c2 = 0;
        for (int q = tid; q < n_part; q += kSmallNT) {
            c0 += __ldcg(part + 3 * q), c1 += __ldcg(part + 3 * q + 1), c2 += __ldcg(part + 3 * q + 2);
        }
        __syncthreads();
        block_sum3<kSmallNT>(c0, c1, c2, red3);
        if (tid == 0) {
            const double a1[3] = {c0, c1, c2};
            if (MODE == MODE_ACCEL) {
                if (blockIdx.x == 0) A.acc_out[0] = a1[0], A.acc_out[1] = a1[1], A.acc_out[2] = a1[2];
            } else {
                const double dt = A.dt, hh = (stage == 2) ? dt : 0.5 * dt;
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    const double kx = sbh.vs[k], kv = a1[k];
                    if (stage == 3) {
                        sbh.x0[k] += dt / 6.0 * (sbh.sx[k] + kx);
                        sbh.v0[k] += dt / 6.0 * (sbh.sv[k] + kv);
                        sbh.xs[k] = sbh.x0[k], sbh.vs[k] = sbh.v0[k];
                    } else {
                        if (stage == 0) {
                            sbh.sx[k] = kx, sbh.sv[k] = kv;
                        } else {
                            sbh.sx[k] += 2.0 * kx, sbh.sv[k] += 2.0 * kv;
                        }
                        sbh.xs[k] = sbh.x0[k] + hh * kx;
                        sbh.vs[k] = sbh.v0[k] + hh * kv;
                    }
                }
            }
        }
    };

    const long long n_eval = (MODE == MODE_RK4) ? 4 * A.nsteps : 1;
    double xs_my[3] = {0, 0, 0}, vs_my[3] = {0, 0, 0};  // the own star's stage state after the last update
    for (long long ev = 0; ev < n_eval; ++ev) {
        const int stage = (int)(ev & 3);
        if (ev > 0) {
            if (tid == 0) bulk_copy_g2s(sxv, A.xv + (size_t)(ev & 1) * np, (unsigned int)(np * sizeof(XVRec)), &fill_bar);
            finish_bh(ev - 1);
            mbar_wait(&fill_bar, (unsigned int)((ev - 1) & 1));
        }
        __syncthreads();

        // per-star records of the Cross kernels and the eight global sums, every block for itself in the same order
        {
            double sums[kCrossSums] = {0, 0, 0, 0, 0, 0, 0, 0};
            for (int q = tid; q < np; q += kSmallNT) {
                const XVRec s = sxv[q];
                const double gm = sgm[q];
                CRec o;
                o.x = s.x, o.y = s.y, o.z = s.z, o.gm = gm;
                o.vx = o.vy = o.vz = o.a5 = o.b = o.wx = o.wy = o.wz = o.rj2 = o.kap = 0.0;
                if (q < A.n_stars) {
                    const double d[3] = {s.x - sbh.xs[0], s.y - sbh.xs[1], s.z - sbh.xs[2]};  // x_j1
                    const double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
                    const double inv_r = 1.0 / sqrt(r2);
                    const double inv_r3 = inv_r * inv_r * inv_r;
                    o.vx = s.vx, o.vy = s.vy, o.vz = s.vz;
                    o.a5 = A.GM * 1.25 * inv_r, o.b = A.GM * 0.25 * inv_r3, o.rj2 = r2;
                    o.kap = 4.0 * A.GM * inv_r + (s.vx * s.vx + s.vy * s.vy + s.vz * s.vz);
                    const double wv[3] = {gm * d[0] * inv_r3, gm * d[1] * inv_r3, gm * d[2] * inv_r3};
                    o.wx = -3.5 * A.GM * wv[0], o.wy = -3.5 * A.GM * wv[1], o.wz = -3.5 * A.GM * wv[2];
                    sums[0] += gm * s.vx, sums[1] += gm * s.vy, sums[2] += gm * s.vz;
                    sums[3] += gm * inv_r, sums[4] += gm * inv_r3;
                    sums[5] += wv[0], sums[6] += wv[1], sums[7] += wv[2];
                }
                scr[q] = o;
            }
#pragma unroll
            for (int q = 0; q < kCrossSums; ++q) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) sums[q] += __shfl_down_sync(0xffffffffu, sums[q], o);
                if (lane == 0) red[q][w] = sums[q];
            }
            __syncthreads();
            if (tid < kCrossSums) {
                double t = 0;
                for (int q = 0; q < NW; ++q) t += red[tid][q];
                scsum[tid] = t;
            }
            __syncthreads();
        }

        // every ordered pair (i, j != i) of this warp's IW i-stars: lane l takes j = l, l + 32, ...
        double xi[IW][3], vi[IW][3], ri2[IW], kapi[IW];
        CrossAcc acc[IW];
#pragma unroll
        for (int k = 0; k < IW; ++k) {
            const CRec c = scr[min(i0 + k, np - 1)];
            xi[k][0] = c.x, xi[k][1] = c.y, xi[k][2] = c.z, vi[k][0] = c.vx, vi[k][1] = c.vy, vi[k][2] = c.vz;
            ri2[k] = c.rj2, kapi[k] = c.kap;
            cross_acc_zero(acc[k]);
        }
        {
            CrossAcc dummy;
            cross_acc_zero(dummy);
            const double zero3[3] = {0, 0, 0};
#pragma unroll 2
            for (int jq = lane; jq < np; jq += 32) {
                const CRec r = scr[jq];
#pragma unroll
                for (int k = 0; k < IW; ++k)
                    cross_pair<false, BHX, false>(r, xi[k], vi[k], ri2[k], kapi[k], 0.0, 0.0, 0.0, zero3, acc[k], dummy, A.eps2, GM4, jq == i0 + k);
            }
        }
        double ss[8] = {0, 0, 0, 0, 0, 0, 0, 0};
#pragma unroll
        for (int k = 0; k < IW; ++k) {
            double t[8] = {acc[k].n[0], acc[k].n[1], acc[k].n[2], acc[k].X[0], acc[k].X[1], acc[k].X[2], acc[k].S, BHX ? acc[k].U : 0.0};
#pragma unroll
            for (int c = 0; c < (BHX ? 8 : 7); ++c) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) t[c] += __shfl_xor_sync(0xffffffffu, t[c], o);
                if (lane == k) ss[c] = t[c];
            }
        }

        double b[3] = {0, 0, 0};
        if (own) {
            const XVRec me = sxv[my];
            const double x[3] = {me.x - sbh.xs[0], me.y - sbh.xs[1], me.z - sbh.xs[2]};  // x_i1
            const double vel[3] = {me.vx, me.vy, me.vz};
            double a[3];
            star_physics<CROSS>(sgm[my], x, vel, ss, scsum, A.GM, A.inv_c2, a, b);
            if (MODE == MODE_ACCEL) {
                double* o = A.acc_out + 3 * (size_t)(my + 1);
                o[0] = a[0], o[1] = a[1], o[2] = a[2];
            } else {
                const double dt = A.dt, hh = (stage == 2) ? dt : 0.5 * dt;
#pragma unroll
                for (int k = 0; k < 3; ++k) {
                    const double kx = vel[k], kv = a[k];
                    if (stage == 3) {
                        x0[k] = x0[k] + dt / 6.0 * (sx[k] + kx);
                        v0[k] = v0[k] + dt / 6.0 * (sv[k] + kv);
                        xs_my[k] = x0[k], vs_my[k] = v0[k];
                    } else {
                        if (stage == 0) {
                            sx[k] = kx, sv[k] = kv;
                        } else {
                            sx[k] += 2.0 * kx, sv[k] += 2.0 * kv;
                        }
                        xs_my[k] = x0[k] + hh * kx;
                        vs_my[k] = v0[k] + hh * kv;
                    }
                }
                XVRec o;
                o.x = xs_my[0], o.y = xs_my[1], o.z = xs_my[2], o.vx = vs_my[0], o.vy = vs_my[1], o.vz = vs_my[2];
                A.xv[(size_t)((ev + 1) & 1) * np + my] = o;  // the next evaluation's stage state, for every block
            }
        }
        {
            double p0 = 0, p1 = 0, p2 = 0;
#pragma unroll
            for (int k = 0; k < IW; ++k) {
                p0 += __shfl_sync(0xffffffffu, b[0], k);
                p1 += __shfl_sync(0xffffffffu, b[1], k);
                p2 += __shfl_sync(0xffffffffu, b[2], k);
            }
            if (lane == 0) {
                double* bp = A.bh_part + (size_t)(ev & 1) * 3 * n_part + 3 * (size_t)gw;
                bp[0] = p0, bp[1] = p1, bp[2] = p2;
            }
        }
        target += gridDim.x;
        if (!small_grid_barrier(A.bar, target, &bar_abort, A.host_flag)) return;  // timed out: the host reports it (small_check)
    }
    finish_bh(n_eval - 1);
    __syncthreads();
    if (MODE == MODE_RK4) {
        if (blockIdx.x == 0 && tid == 0) *A.bh = sbh;
        if (own) {
            JRec* g = A.jrec_out + my;
            g->x = xs_my[0], g->y = xs_my[1], g->z = xs_my[2];
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const size_t q = (size_t)k * np + my;
                A.v[q] = vs_my[k], A.x0[q] = x0[k], A.v0[q] = v0[k], A.sx[q] = sx[k], A.sv[q] = sv[k];
            }
        }
    }
}

}  // namespace pn
