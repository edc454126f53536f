// pn_kernels.cuh -- sm_100a kernels of the limited-1PN hot path (arXiv:1801.07986).
// Product code: shares nothing with oracle/.  Citations: /root/reference/PAPER.md:<line>.
//
// Kernels, in the order of this file (DESIGN.md section 6 has the roofline of each):
//   S1  pair_fp64_kernel          star-star Newtonian, every ordered pair, tiled (PN_PAIR_TILED)
//       pair_sym_fp64_kernel      the same, every unordered pair once (Newton's third law), general / equal-mass form; the
//                                 j-side sums travel through the lanes of a warp in Gray-code order (N_s >= 3072)
//       pair_cross_fp64_kernel, pair_cross_sym_kernel   NEXT-1/2: S1 + the O(N^2) sums of the Cross terms, Eqs. 2.6 and 2.3, on
//                                 ordered / unordered pairs (cross_prep/sum: O(N))
//       pair_fp32_kernel, pair_sym_fp32_kernel   fp32-pair / fp64-accumulate variant (packed f32x2 arithmetic; split kernels:
//                                 two-float records)
//   S2-S4  epilogue_kernel        partial-sum reduction, BH <-> star Newtonian + 1PN, a_1 reduction, fused RK4 stage update
//   S1-S4  small_path_kernel      N_s < 3072: a whole pn_step call (or one pn_accel) in ONE cooperative launch
//   S5  energy_prep / energy_pair / energy_final   Eq. 2.7, compensated
//   NEXT-3  momentum_prep / momentum_pair / momentum_final   Eq. 2.8, compensated
//   pack / unpack (AoS <-> internal layout)
//
// Internal data layout (all fp64, star index s = body index - 1, padded to NP):
//   JRec  jrec[NP]      : stage position + mass constants of star s, 48 B, 16 B aligned.  This is the record the
//                         O(N^2) pair kernels read; pad records have gm = 0, x = 1e100.
//   double v[3][NP]     : stage velocity, SoA
//   double x0/v0[3][NP] : state at the beginning of the RK4 step;  double sx/sv[3][NP] : weighted sum of k's
//   double part[S][3][NP]: partial star-star accelerations, one slot per j-chunk (tiled) or j-group (symmetric), each entry
//                         written by exactly one block; summed in fixed order by the epilogue (7 or 8 components per slot
//                         in Cross mode)
//   BhState             : the massive object's stage state, step state, k-sums (a handful of doubles)
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

// ---------------------------------------------------------------------------------------------------------
// S1: star-star Newtonian all-pairs, fp64.   a_i^SS = sum_{j != i} G m_j (x_j - x_i) / rho_ij^3
// PAPER.md:63 (Eq. 2.4, second term; exponent 3: reading R4) with rho_ij^2 = r_ij^2 + eps^2.
//
// Per ordered pair: 15 FP64-pipe instructions + 1 MUFU:
//   d = x_j - x_i (3 DADD); r2 = d.d + eps^2 (3 DFMA); y0 = MUFU.RSQ64H(r2);
//   t = y0*y0 (DMUL, exact: y0 has 21 significant bits); e = 1 - r2*t (DFMA)              [e = O(2^-20)]
//   rho^-3 = y0^3 (1-e)^(-3/2) = y0^3 (1 + 3/2 e + 15/8 e^2 + O(e^3 ~ 2^-60))
//   q = G m_j (1 + 3/2 e + 15/8 e^2) = fma(e, fma(e, g1875, g15), gm) (2 DFMA, constants precomputed per j)
//   u = t*y0 (DMUL); s = u*q (DMUL); a += s*d (3 DFMA)
// Each thread keeps I i-particles (position + accumulator) in registers; j records are broadcast from shared
// memory with 3 LDS.128 per j, amortised over I pairs.  grid = (i-tiles, j-splits); block (it, sp) writes the
// partial sums of its i-tile over j-tiles [sp*tiles_per_split, (sp+1)*tiles_per_split).
// MASK (eps == 0 only): the self pair j == i is skipped by index (it would be 0 * inf).
// ---------------------------------------------------------------------------------------------------------
// The I x JU pairs of one inner-loop trip are evaluated stage by stage (all subtractions, then all r2, ...), so
// that dependent FP64 instructions of one pair are separated by the same stage of the other pairs: DFMA latency
// is hidden inside the warp and consecutive instructions share operands (x_j, g15, g1875, gm, s) in the same
// slot, which the operand-reuse cache needs (a DFMA with three distinct register operands costs 3 issue cycles
// on sm_100a instead of 2 -- measured).
template <int I, int JU, bool MASK, int JSTR = 1>
__device__ __forceinline__ void pairs_fp64(const JRec* __restrict__ tile, int jj, int jglob, const double (&xi)[I],
                                           const double (&yi)[I], const double (&zi)[I], const int (&ii)[I],
                                           double (&ax)[I], double (&ay)[I], double (&az)[I], double eps2)
{
    JRec r[JU];
#pragma unroll
    for (int u = 0; u < JU; ++u) r[u] = tile[jj + u * JSTR];  // JSTR = 32: the lanes of a warp share out the j-stars
    double dx[JU][I], dy[JU][I], dz[JU][I], r2[JU][I], y0[JU][I], t[JU][I], e[JU][I], s[JU][I];
#pragma unroll
    for (int u = 0; u < JU; ++u)
#pragma unroll
        for (int k = 0; k < I; ++k) {
            dx[u][k] = r[u].x - xi[k];
            dy[u][k] = r[u].y - yi[k];
            dz[u][k] = r[u].z - zi[k];
        }
#pragma unroll
    for (int u = 0; u < JU; ++u)
#pragma unroll
        for (int k = 0; k < I; ++k) r2[u][k] = fma(dz[u][k], dz[u][k], eps2);
#pragma unroll
    for (int u = 0; u < JU; ++u)
#pragma unroll
        for (int k = 0; k < I; ++k) r2[u][k] = fma(dy[u][k], dy[u][k], r2[u][k]);
#pragma unroll
    for (int u = 0; u < JU; ++u)
#pragma unroll
        for (int k = 0; k < I; ++k) r2[u][k] = fma(dx[u][k], dx[u][k], r2[u][k]);
#pragma unroll
    for (int u = 0; u < JU; ++u)
#pragma unroll
        for (int k = 0; k < I; ++k) y0[u][k] = rsqrt_seed(r2[u][k]);
#pragma unroll
    for (int u = 0; u < JU; ++u)
#pragma unroll
        for (int k = 0; k < I; ++k) t[u][k] = y0[u][k] * y0[u][k];
#pragma unroll
    for (int u = 0; u < JU; ++u)
#pragma unroll
        for (int k = 0; k < I; ++k) e[u][k] = fma(-r2[u][k], t[u][k], 1.0);
#pragma unroll
    for (int u = 0; u < JU; ++u)
#pragma unroll
        for (int k = 0; k < I; ++k) {
            t[u][k] = t[u][k] * y0[u][k];                        // y0^3
            s[u][k] = fma(e[u][k], r[u].g1875, r[u].g15);        // G m_j (3/2 + 15/8 e)
        }
#pragma unroll
    for (int u = 0; u < JU; ++u)
#pragma unroll
        for (int k = 0; k < I; ++k) s[u][k] = fma(e[u][k], s[u][k], r[u].gm);  // G m_j (1 + 3/2 e + 15/8 e^2)
#pragma unroll
    for (int u = 0; u < JU; ++u)
#pragma unroll
        for (int k = 0; k < I; ++k) {
            s[u][k] = s[u][k] * t[u][k];  // G m_j / rho^3
            if (MASK) s[u][k] = (jglob + u * JSTR == ii[k]) ? 0.0 : s[u][k];
        }
#pragma unroll
    for (int u = 0; u < JU; ++u)
#pragma unroll
        for (int k = 0; k < I; ++k) {
            ax[k] = fma(s[u][k], dx[u][k], ax[k]);
            ay[k] = fma(s[u][k], dy[u][k], ay[k]);
            az[k] = fma(s[u][k], dz[u][k], az[k]);
        }
}

template <int I, int JU, int MINB, int NT, int TJ, bool MASK>
__global__ void __launch_bounds__(NT, MINB) pair_fp64_kernel(const JRec* __restrict__ jrec, double* __restrict__ part,
                                                             int np, int tiles_per_split, double eps2)
{
    static_assert(TJ % JU == 0, "tile must be a multiple of the j unroll");
    __shared__ JRec sj[2][TJ];
    const int tid = threadIdx.x;
    const int i_base = blockIdx.x * (I * NT) + tid;

    double xi[I], yi[I], zi[I], ax[I], ay[I], az[I];
    int ii[I];
#pragma unroll
    for (int k = 0; k < I; ++k) {
        ii[k] = i_base + k * NT;
        const JRec* p = jrec + ii[k];
        xi[k] = p->x, yi[k] = p->y, zi[k] = p->z;
        ax[k] = ay[k] = az[k] = 0.0;
    }

    const int n_tiles = np / TJ;
    const int t_begin = blockIdx.y * tiles_per_split;
    const int t_end = min(n_tiles, t_begin + tiles_per_split);

    constexpr int kVecPerTile = TJ * 3;  // double2 per tile
    auto fill = [&](int buf, int t) {
        const double2* src = reinterpret_cast<const double2*>(jrec + (size_t)t * TJ);
        double2* dst = reinterpret_cast<double2*>(sj[buf]);
        for (int q = tid; q < kVecPerTile; q += NT) dst[q] = src[q];
    };

    if (t_begin < t_end) fill(0, t_begin);
    __syncthreads();
    for (int t = t_begin; t < t_end; ++t) {
        const int buf = (t - t_begin) & 1;
        if (t + 1 < t_end) fill(buf ^ 1, t + 1);  // next tile into the other buffer while this one is consumed
        const JRec* tile = sj[buf];
        const int j0 = t * TJ;
#pragma unroll 1
        for (int jj = 0; jj < TJ; jj += JU) pairs_fp64<I, JU, MASK>(tile, jj, j0 + jj, xi, yi, zi, ii, ax, ay, az, eps2);
        __syncthreads();
    }

    double* out = part + (size_t)blockIdx.y * 3 * np;
#pragma unroll
    for (int k = 0; k < I; ++k) {
        out[ii[k]] = ax[k];
        out[np + ii[k]] = ay[k];
        out[2 * np + ii[k]] = az[k];
    }
}

// ---------------------------------------------------------------------------------------------------------
// S1, symmetric form: every unordered star pair {i, j} is evaluated once and applied to both stars (Newton's
// third law holds exactly for the softened Newtonian star-star term of Eq. 2.4):
//     a_i += G m_j K d,   a_j -= G m_i K d,   d = x_j - x_i,   K = rho_ij^-3.
// Per unordered pair: 20 FP64-pipe instructions + 1 MUFU (= 10 per ordered pair instead of 15):
//   d (3 DADD); r2 = d.d + eps^2 (3 DFMA); y0 = MUFU.RSQ64H(r2); t = y0^2; e = 1 - r2 t;
//   p = 1 + 3/2 e + 15/8 e^2 (2 DFMA); u = t y0; K = u p; s_j = K Gm_j; s_i = -K Gm_i; 6 DFMA accumulate.
//
// Work decomposition.  Stars are cut into unit tiles of U = 32 W I stars and the tiles into G groups of m tiles.
// Block (A <= B) owns the group pair: it walks the unit-tile pairs (ta in A, tb in B; tb >= ta when A == B).
// Inside a unit-tile pair each warp keeps I i-stars per lane in registers (position, accumulator, -G m_i) and
// sweeps the tile's j-stars in sub-groups of 32: lane l starts with j-star l of the sub-group and in 32 rotation
// steps meets all 32 (positions come from shared memory at a rotating index; the three j-side accumulators
// travel from lane to lane with SHFL), so after 32 steps the j-side sums are complete and back in their home
// lane without any reduction across lanes.  The diagonal unit tile (ta == tb) is evaluated as ordered pairs,
// i-side only.
//
// Output: slot P of part[P][3][np] receives, for every star, the sum over the j-stars of group P -- written by
// exactly one block in a fixed order (row sums of block (A,B) go to slot B, column sums to slot A), so the
// epilogue's fixed-order sum over the G slots is bit-reproducible and nothing has to be zeroed between launches.
// ---------------------------------------------------------------------------------------------------------
template <int I, bool SYM, bool MASK, bool EQM>
__device__ __forceinline__ void sym_step(const double2 xy, const double2 zm, const double (&xi)[I],
                                         const double (&yi)[I], const double (&zi)[I], const double (&ngi)[I],
                                         double (&ax)[I], double (&ay)[I], double (&az)[I], double& bx, double& by,
                                         double& bz, double eps2, int self_k)
{
    double dx[I], dy[I], dz[I], r2[I], y0[I], t[I], e[I], p[I], sj[I];
#pragma unroll
    for (int k = 0; k < I; ++k) {
        dx[k] = xy.x - xi[k];
        dy[k] = xy.y - yi[k];
        dz[k] = zm.x - zi[k];
    }
#pragma unroll
    for (int k = 0; k < I; ++k) r2[k] = fma(dz[k], dz[k], eps2);
#pragma unroll
    for (int k = 0; k < I; ++k) r2[k] = fma(dy[k], dy[k], r2[k]);
#pragma unroll
    for (int k = 0; k < I; ++k) r2[k] = fma(dx[k], dx[k], r2[k]);
#pragma unroll
    for (int k = 0; k < I; ++k) y0[k] = rsqrt_seed(r2[k]);
#pragma unroll
    for (int k = 0; k < I; ++k) t[k] = y0[k] * y0[k];
#pragma unroll
    for (int k = 0; k < I; ++k) e[k] = fma(-r2[k], t[k], 1.0);
#pragma unroll
    for (int k = 0; k < I; ++k) {
        t[k] = t[k] * y0[k];             // y0^3
        p[k] = fma(e[k], 1.875, 1.5);
    }
#pragma unroll
    for (int k = 0; k < I; ++k) p[k] = fma(e[k], p[k], 1.0);  // (1 - e)^(-3/2) to O(e^3)
#pragma unroll
    for (int k = 0; k < I; ++k) {
        t[k] = t[k] * p[k];              // K = rho^-3
        if (MASK) t[k] = (k == self_k) ? 0.0 : t[k];
    }

    if (EQM) {  // all stars have the same mass: accumulate K d on both sides, the common G m is applied at the flush
#pragma unroll
        for (int k = 0; k < I; ++k) {
            ax[k] = fma(t[k], dx[k], ax[k]);
            ay[k] = fma(t[k], dy[k], ay[k]);
            az[k] = fma(t[k], dz[k], az[k]);
        }
        if (SYM) {
#pragma unroll
            for (int k = 0; k < I; ++k) {
                bx = fma(-t[k], dx[k], bx);
                by = fma(-t[k], dy[k], by);
                bz = fma(-t[k], dz[k], bz);
            }
        }
    } else {
#pragma unroll
        for (int k = 0; k < I; ++k) sj[k] = t[k] * zm.y;  // G m_j K
#pragma unroll
        for (int k = 0; k < I; ++k) {
            ax[k] = fma(sj[k], dx[k], ax[k]);
            ay[k] = fma(sj[k], dy[k], ay[k]);
            az[k] = fma(sj[k], dz[k], az[k]);
        }
        if (SYM) {
#pragma unroll
            for (int k = 0; k < I; ++k) t[k] = t[k] * ngi[k];  // -G m_i K
#pragma unroll
            for (int k = 0; k < I; ++k) {
                bx = fma(t[k], dx[k], bx);
                by = fma(t[k], dy[k], by);
                bz = fma(t[k], dz[k], bz);
            }
        }
    }
}

template <int I, int U, bool SYM, bool MASK, bool EQM, int UNR = 32 / I>
__device__ __forceinline__ void sym_unit_tile(const double2* __restrict__ sxy, const double2* __restrict__ szm,
                                              double* __restrict__ cw /* [3][U] column sums this warp writes into */,
                                              const double (&xi)[I], const double (&yi)[I], const double (&zi)[I],
                                              const double (&ngi)[I], double (&ax)[I], double (&ay)[I],
                                              double (&az)[I], double eps2, int lane, int i_local0, int jb0, int jb1)
{
#pragma unroll 1
    for (int jb = jb0; jb < jb1; jb += 32) {
        double bx = 0.0, by = 0.0, bz = 0.0;
        constexpr int kUnr = UNR;  // rotation steps unrolled: 32 independent pairs per trip (16: -1 %, 8: -4 %, 128: -9 %, measured)
#pragma unroll kUnr
        for (int r = 0; r < 32; ++r) {
            const int jj = jb + ((lane + r) & 31);
            int self_k = -1;
            if (MASK) {  // diagonal unit tile with eps == 0: the self pair would be 0 * inf
                const int q = jj - i_local0;
                self_k = (q >= 0 && (q & 31) == 0) ? (q >> 5) : -1;
            }
            sym_step<I, SYM, MASK, EQM>(sxy[jj], szm[jj], xi, yi, zi, ngi, ax, ay, az, bx, by, bz, eps2, self_k);
            if (SYM) {  // the j-star moves on to the next lane together with its partial sums
                const int src = (lane + 1) & 31;
                bx = __shfl_sync(0xffffffffu, bx, src);
                by = __shfl_sync(0xffffffffu, by, src);
                bz = __shfl_sync(0xffffffffu, bz, src);
            }
        }
        if (SYM) {  // after 32 rotations lane l holds the complete sums of j-star jb + l again
            cw[jb + lane] = bx;
            cw[U + jb + lane] = by;
            cw[2 * U + jb + lane] = bz;
        }
    }
}

// Gray-code traversal of a rotation group (the default of the symmetric kernels): lane l meets j-star l ^ g(r) at step r,
// g(r) = r ^ (r >> 1), so consecutive steps differ in ONE bit and the j-side sums move on with a butterfly shuffle whose
// lane mask is an immediate (SHFL.BFLY: one register read, measured free next to the FP64 stream), where the rotation
// (lane + r) mod 32 needs SHFL.IDX with the source lane in a register (two register reads: measured 1.9 FP64-pipe
// cycles each on sm_100a, profiles/r2_ncu_summary.md section 2) and four integer instructions per step for the index.
// The 32 steps are two identical halves of 16 (g(16 + q) = 24 ^ g(q); masks 1 2 1 4 1 2 1 8 1 2 1 4 1 2 1 16, the last
// one brings the sums to the next half's first lane or, after step 31, home), so the unrolled body is 16 steps long and
// every mask and every index offset in it is a compile-time constant.
template <int I, int U, bool EQM, int STEPS>
__device__ __forceinline__ void sym_unit_tile_gray(const double2* __restrict__ sxy, const double2* __restrict__ szm,
                                                   double* __restrict__ cw, const double (&xi)[I], const double (&yi)[I],
                                                   const double (&zi)[I], const double (&ngi)[I], double (&ax)[I],
                                                   double (&ay)[I], double (&az)[I], double eps2, int lane, int jb0, int jb1)
{
    static_assert(STEPS == 8 || STEPS == 16, "unrolled steps of the Gray-code walk");
#pragma unroll 1
    for (int jb = jb0; jb < jb1; jb += 32) {
        double bx = 0.0, by = 0.0, bz = 0.0;
#pragma unroll 1
        for (int c = 0; c < 32 / STEPS; ++c) {
            // first j index of chunk c: l ^ g(STEPS c); g(8) = 12, g(16) = 24, g(24) = 20
            const int off = (STEPS == 16) ? (c ? 24 : 0) : ((c & 1 ? 12 : 0) ^ (c & 2 ? 24 : 0));
            const int base = jb + (lane ^ off);
            // mask of the chunk's last move: g(STEPS c + STEPS - 1) ^ g(STEPS (c + 1)); 16 for both halves, 8 / 16 for quarters
            const int last_mask = (STEPS == 16) ? 16 : ((c & 1) ? 16 : 8);
#pragma unroll
            for (int q = 0; q < STEPS; ++q) {
                const int jj = base ^ (q ^ (q >> 1));
                sym_step<I, true, false, EQM>(sxy[jj], szm[jj], xi, yi, zi, ngi, ax, ay, az, bx, by, bz, eps2, -1);
                if (q + 1 < STEPS) {
                    const int mask = (q + 1) & -(q + 1);  // lowest set bit of q + 1: the bit in which g(q) and g(q + 1) differ
                    bx = __shfl_xor_sync(0xffffffffu, bx, mask);
                    by = __shfl_xor_sync(0xffffffffu, by, mask);
                    bz = __shfl_xor_sync(0xffffffffu, bz, mask);
                } else {
                    bx = __shfl_xor_sync(0xffffffffu, bx, last_mask);
                    by = __shfl_xor_sync(0xffffffffu, by, last_mask);
                    bz = __shfl_xor_sync(0xffffffffu, bz, last_mask);
                }
            }
        }
        cw[jb + lane] = bx;  // after 32 steps lane l holds the complete sums of j-star jb + l again
        cw[U + jb + lane] = by;
        cw[2 * U + jb + lane] = bz;
    }
}

// triangular decode of a work-item index: (A <= B), id = B (B + 1) / 2 + A
__device__ __forceinline__ void sym_decode_block(int id, int& A, int& B)
{
    B = (int)((sqrtf(8.0f * (float)id + 1.0f) - 1.0f) * 0.5f);
    while ((B + 1) * (B + 2) / 2 <= id) ++B;
    while (B * (B + 1) / 2 > id) --B;
    A = id - B * (B + 1) / 2;
}

// a one-warp block needs warp-level barriers only
template <int W>
__device__ __forceinline__ void sym_sync()
{
    if (W == 1)
        __syncwarp();
    else
        __syncthreads();
}

// adds n_src block-owned [3][U] tiles (consecutive in shared memory) into one (slot, tile) of part.  Every element of part
// has one writer in the whole launch, the same thread of the same block on every call: the first contribution is a plain
// store, later ones are reductions to the same address by the same thread (RED.ADD.F64, applied in program order, no
// read-modify-write latency), so the order of the sum stays fixed
template <int U, int NT>
__device__ __forceinline__ void sym_flush(const double* __restrict__ cacc, double* __restrict__ dst, int np, bool first,
                                          int n_src, int tid, double scale = 1.0)
{
    for (int q = tid; q < 3 * U; q += NT) {
        const int c = q / U, el = q - c * U;
        double v = cacc[q];
        for (int s = 1; s < n_src; ++s) v += cacc[s * 3 * U + q];
        v *= scale;
        double* d = dst + (size_t)c * np + el;
        if (first)
            *d = v;
        else
            atomicAdd(d, v);
    }
}

// unit tile of the symmetric kernels: W warps of I i-stars per lane each (JS = false), or -- j-split form, JS = true,
// W == I -- I i-stars per lane held by EVERY warp, warp w sweeping rotation group w of the j tile
template <int I, int W, bool JS>
constexpr int kSymU = JS ? 32 * I : W * 32 * I;

template <int I, int W, bool JS = false>
constexpr int kSymSmemBytes = kSymU<I, W, JS> * (2 * 16 + W * 3 * 8);

// EQM: every star has the same mass (true of every BASELINE.json config and of the paper's own model):
// both sides accumulate K d and the common G m = gm_eq multiplies the sums once, at the flush: 18 instead of 20 FP64
// instructions per unordered pair.
// JS (j-split form, W == I warps, U = 32 I): all warps of the block hold the SAME I i-stars per lane and each sweeps one
// rotation group (32 j-stars) of the j tile, so a unit-tile pair costs a quarter (1 / W) of the time it costs a one-warp
// block of the same U while the partial-sum slots stay those of U = 32 I: W times more, W times shorter work items for
// the same slot layout -- this is what shortens the launch tail at N_s ~ 10^4.  The column sums
// of a warp are complete for its 32 j-stars; the row sums of the W warps are added in fixed warp order at the flush.
template <int I, int W, int MINB, bool MASK, bool EQM, bool JS = false, int UNR = 32 / I, int TRAV = 16>
__global__ void __launch_bounds__(W * 32, MINB) pair_sym_fp64_kernel(const JRec* __restrict__ jrec,
                                                                     double* __restrict__ part, int np, int n_tiles,
                                                                     int m, double eps2, double gm_eq, int item0)
{
    static_assert(!JS || W == I, "j-split form: one rotation group of the j tile per warp");
    constexpr int U = kSymU<I, W, JS>;
    constexpr int NT = W * 32;
    extern __shared__ double2 sym_smem[];  // kSymSmemBytes<I, W, JS>: dynamic, U = 512 needs more than 48 KB
    const int item = item0 + blockIdx.x;
    double2* sxy = sym_smem;                                                   // [U] x, y of the j tile
    double2* szm = sym_smem + U;                                               // [U] z, G m
    double(*cacc)[3][U] = reinterpret_cast<double(*)[3][U]>(sym_smem + 2 * U);  // [W][3][U] per-warp sums
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    int A, B;
    sym_decode_block(item, A, B);

    const int ta0 = A * m, ta1 = min(ta0 + m, n_tiles);
    const int tb0 = B * m, tb1 = min(tb0 + m, n_tiles);
    const int i_local0 = JS ? lane : w * 32 * I + lane;  // this lane's k-th i-star is i_local0 + 32 k inside the unit tile
    const int jb0 = JS ? 32 * w : 0, jb1 = JS ? 32 * w + 32 : U;  // rotation groups of the j tile this warp sweeps
    double* cw = JS ? &cacc[0][0][0] : &cacc[w][0][0];            // where this warp's column sums go

    auto flush = [&](int slot, int tile, bool first, int n_src) {
        sym_flush<U, NT>(&cacc[0][0][0], part + (size_t)slot * 3 * np + (size_t)tile * U, np, first, n_src, tid, EQM ? gm_eq : 1.0);
    };

    for (int ta = ta0; ta < ta1; ++ta) {
        double xi[I], yi[I], zi[I], ngi[I], ax[I], ay[I], az[I];
#pragma unroll
        for (int k = 0; k < I; ++k) {
            const JRec* p = jrec + (size_t)ta * U + i_local0 + 32 * k;
            xi[k] = p->x, yi[k] = p->y, zi[k] = p->z, ngi[k] = -p->gm;
            ax[k] = ay[k] = az[k] = 0.0;
        }
        for (int tb = (A == B) ? ta : tb0; tb < tb1; ++tb) {
            sym_sync<W>();  // everyone is done with the previous tile's shared memory
            for (int q = tid; q < U; q += NT) {
                const double2* src = reinterpret_cast<const double2*>(jrec + (size_t)tb * U + q);
                sxy[q] = src[0];  // x, y
                szm[q] = src[1];  // z, G m
            }
            sym_sync<W>();
            if (ta == tb) {
                sym_unit_tile<I, U, false, MASK, EQM, UNR>(sxy, szm, cw, xi, yi, zi, ngi, ax, ay, az, eps2, lane, i_local0, jb0, jb1);
            } else {
                if (TRAV)
                    sym_unit_tile_gray<I, U, EQM, (TRAV == 8) ? 8 : 16>(sxy, szm, cw, xi, yi, zi, ngi, ax, ay, az, eps2, lane, jb0, jb1);
                else
                    sym_unit_tile<I, U, true, false, EQM, UNR>(sxy, szm, cw, xi, yi, zi, ngi, ax, ay, az, eps2, lane, i_local0, jb0, jb1);
                sym_sync<W>();
                flush(A, tb, ta == ta0, JS ? 1 : W);  // column sums: the i-stars of tile ta acting on the j-stars of tile tb
            }
        }
        sym_sync<W>();
        {
            double(*rw)[U] = JS ? cacc[w] : cacc[0];  // JS: every warp holds partial row sums of all U i-stars
#pragma unroll
            for (int k = 0; k < I; ++k) {
                rw[0][i_local0 + 32 * k] = ax[k];
                rw[1][i_local0 + 32 * k] = ay[k];
                rw[2][i_local0 + 32 * k] = az[k];
            }
        }
        sym_sync<W>();
        flush(B, ta, (A < B) || (ta == ta0), JS ? W : 1);  // row sums: the j-stars of group B acting on the i-stars of tile ta
    }
}

// ---------------------------------------------------------------------------------------------------------
// NEXT-1 of the scope table: [a_i]_Cross, Eq. 2.6, fused into the star-star pair loop
// (PN_OPT_CROSS_TERMS).  With x_ab = x_a - x_b, v_ij = v_i - v_j, every star-star r_ij -> rho_ij (reading R9):
//   L0  5 G^2 m_i M x_i1 / r_i1^4 - (G m_i / r_i1^3) [ 4 v_i^2 x_i1 - 7 (v_i.x_i1) v_i ]
//   L1  sum_j G^2 m_j M x_i1 / r_i1^3 ( 4/rho_ij + 5/(4 r_j1) + r_i1^2/(4 r_j1^3) - rho_ij^2/(4 r_j1^3) )
//   L2  sum_j G^2 m_j M x_ij / rho_ij^3 ( 4/r_i1 + 5/(4 r_j1) - r_i1^2/(4 r_j1^3) + rho_ij^2/(4 r_j1^3) )
//   L3  -(7/2) sum_j G^2 m_j M x_j1 / r_j1^3 ( 1/rho_ij - 1/r_i1 )
//   L4  - sum_j (G m_j / r_i1^3) [ 4 (v_i.v_j) x_i1 - 3 (v_j.x_i1) v_i - 4 (v_i.x_i1) v_j ]
//   L5  + sum_j (G m_j x_ij / rho_ij^3) [ v_i^2 - 2 |v_ij|^2 + (3/2)(v_j.x_ij)^2 / rho_ij^2 ]
//   L6  + sum_j (G m_j / rho_ij^3) [ x_ij.(4 v_i - 3 v_j) ] v_ij
// Regrouping (the oracle evaluates the lines as printed).  Everything in which the pair distance does not appear is a
// sum over all j != i of a per-j quantity, i.e. a global sum minus star i's own term: with
//   P = sum_j G m_j v_j,  Q1 = sum_j G m_j / r_j1,  Q3 = sum_j G m_j / r_j1^3,  W = sum_j G m_j x_j1 / r_j1^3
// (cross_prep_kernel + cross_sum_kernel, O(N)) L4 and parts of L1 and L3 are O(N) work in the epilogue.  What is left for
// the O(N^2) loop, per ordered pair (i <- j) with d = x_ij, u = v_ij, y = 1/rho_ij, s = G m_j y^3 and the per-star constants
// of the record below (a5_j = GM 5/(4 r_j1), b_j = GM/(4 r_j1^3), w_j = -(7/2) GM G m_j x_j1/r_j1^3, kap_i = 4GM/r_i1 + v_i^2):
//   n  -= s d                                                           (the Newtonian term of Eq. 2.4)
//   X  += s g d + h u + y w_j                                            (pair parts of L2 + L5, L6, L3)
//         g = (rho^2 - r_i1^2) b_j + a5_j + kap_i - 2 |u|^2 + (3/2)(v_j.d)^2 y^2,    h = s (4 v_i.d - 3 v_j.d)
//   S  += G m_j (4 GM y - rho^2 b_j)                                     (L1: coefficient of x_i1 / r_i1^3, applied by the epilogue)
//   U  += G m_j y (5/4 + (r_i1^2 - r_j1^2) y^2 / 4)                      (BHX: [a_1]_Cross, below)
// Output part[S][7 or 8][np]: n (3), X (3), S, U per partial-sum slot, reduced in fixed order by the epilogue.
//
// Two kernels.  pair_cross_fp64_kernel walks every ORDERED pair (tiled: j tiles through double-buffered shared memory,
// I i-stars per thread; used below kCrossSymMinStars).  pair_cross_sym_kernel evaluates every UNORDERED pair once, for
// both stars: d, rho^-1, |u|^2, v_i.d and v_j.d are shared, the reversed pair (j <- i) has d -> -d, u -> -u,
//   n_j += s_i d,   X_j += -s_i g' d - h' u + y w_i,   g' = (rho^2 - r_j1^2) b_i + a5_i + kap_j - 2|u|^2 + (3/2)(v_i.d)^2 y^2,
//   h' = s_i (3 v_i.d - 4 v_j.d),   S_j += G m_i (4 GM y - rho^2 b_i),   U_j += G m_i y (5/4 - (r_i1^2 - r_j1^2) y^2 / 4),
// and the eight j-side sums travel through the lanes of the warp with the j-star (Gray-code walk, butterfly shuffles) as
// in pair_sym_fp64_kernel: 76 FP64-pipe instructions + 1 MUFU.RSQ64H per unordered pair (84 with U) = 38 (42) per ordered
// pair instead of 54 (59).
// ---------------------------------------------------------------------------------------------------------
struct __align__(16) CRec {
    double x, y, z, gm;      // position, G m_j
    double vx, vy, vz, a5;   // velocity, GM 5 / (4 r_j1)
    double b, wx, wy, wz;    // GM / (4 r_j1^3),  -(7/2) GM G m_j x_j1 / r_j1^3
    double rj2, kap;         // r_j1^2,  4 GM / r_j1 + v_j^2
};
static_assert(sizeof(CRec) == 112, "CRec must be 112 bytes");

constexpr int kCrossSums = 8;  // P (3), Q1, Q3, W (3)

template <int NT>
__global__ void __launch_bounds__(NT) cross_prep_kernel(const JRec* __restrict__ jrec, const double* __restrict__ v,
                                                        const BhState* __restrict__ bh, CRec* __restrict__ crec,
                                                        double* __restrict__ blk /* [grid][8] */, int n_stars, int np, double GM,
                                                        double w_scale /* 1, or 1 / (G m) for the equal-mass form of the symmetric kernel */)
{
    __shared__ double red[kCrossSums][NT / 32];
    const int i = blockIdx.x * NT + threadIdx.x;
    double sums[kCrossSums] = {0, 0, 0, 0, 0, 0, 0, 0};
    if (i < np) {
        const JRec r = jrec[i];
        CRec o;
        o.x = r.x, o.y = r.y, o.z = r.z, o.gm = r.gm;
        o.vx = o.vy = o.vz = o.a5 = o.b = o.wx = o.wy = o.wz = o.rj2 = o.kap = 0.0;
        if (i < n_stars) {
            const double d[3] = {r.x - bh->xs[0], r.y - bh->xs[1], r.z - bh->xs[2]};  // x_j1
            const double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
            const double inv_r = 1.0 / sqrt(r2);
            const double inv_r3 = inv_r * inv_r * inv_r;
            o.vx = v[i], o.vy = v[np + i], o.vz = v[2 * np + i];
            o.a5 = GM * 1.25 * inv_r, o.b = GM * 0.25 * inv_r3, o.rj2 = r2;
            o.kap = 4.0 * GM * inv_r + (o.vx * o.vx + o.vy * o.vy + o.vz * o.vz);
            const double w[3] = {r.gm * d[0] * inv_r3, r.gm * d[1] * inv_r3, r.gm * d[2] * inv_r3};
            o.wx = -3.5 * GM * w_scale * w[0], o.wy = -3.5 * GM * w_scale * w[1], o.wz = -3.5 * GM * w_scale * w[2];
            sums[0] = r.gm * o.vx, sums[1] = r.gm * o.vy, sums[2] = r.gm * o.vz;
            sums[3] = r.gm * inv_r, sums[4] = r.gm * inv_r3;
            sums[5] = w[0], sums[6] = w[1], sums[7] = w[2];
        }
        crec[i] = o;
    }
#pragma unroll
    for (int q = 0; q < kCrossSums; ++q) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) sums[q] += __shfl_down_sync(0xffffffffu, sums[q], o);
        if ((threadIdx.x & 31) == 0) red[q][threadIdx.x >> 5] = sums[q];
    }
    __syncthreads();
    if (threadIdx.x < kCrossSums) {
        double s = 0;
        for (int w = 0; w < NT / 32; ++w) s += red[threadIdx.x][w];
        blk[(size_t)blockIdx.x * kCrossSums + threadIdx.x] = s;
    }
}

// fixed-order sum of the block partials: one warp per quantity
__global__ void __launch_bounds__(256) cross_sum_kernel(const double* __restrict__ blk, int n_blk, double* __restrict__ out)
{
    const int q = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double s = 0;
    for (int b = lane; b < n_blk; b += 32) s += blk[(size_t)b * kCrossSums + q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if (lane == 0) out[q] = s;
}

// BHX (NEXT-2, [a_1]_Cross, Eq. 2.3): with x_1j = x_1 - x_j and i, j both running over the stars,
//   4 sum_j G^2 m_j^2 x_1j / r_1j^4
//   + sum_{j != k} G^2 m_j m_k x_1j / r_1j^3 ( 4/r_1k + 5/(4 rho_jk) + (r_1j^2 - r_1k^2)/(4 rho_jk^3) )
//   - (7/2) sum_{j != k} G^2 m_j m_k x_jk / (rho_jk^3 r_1j)                  [= + (7/2) sum_j (G m_j / r_1j) a_j^SS]
//   - sum_{j, k} (G m_j m_k / (M r_1j^3)) [ 4 (v_j.v_k) x_1j - 3 (v_j.x_1j) v_k - 4 (v_k.x_1j) v_j ]   [O(N) with P]
// needs one more O(N^2) sum per star, U_i = sum_{j != i} G m_j ( 5/(4 rho) + (r_i1^2 - r_j1^2)/(4 rho^3) ) (last output
// component); everything else is O(N) work in the epilogue, summed over the stars by the reduction that already builds a_1.
template <bool BHX>
constexpr int kCrossNC = BHX ? 8 : 7;

template <int I, int MINB, int NT, int TJ, bool BHX>
__global__ void __launch_bounds__(NT, MINB) pair_cross_fp64_kernel(const CRec* __restrict__ crec, double* __restrict__ part /* [S][NC][np] */,
                                                                   int np, int tiles_per_split, double eps2, double GM4)
{
    constexpr int NC = kCrossNC<BHX>;
    __shared__ CRec sj[2][TJ];
    const int tid = threadIdx.x;
    double xi[I], yi[I], zi[I], vxi[I], vyi[I], vzi[I], ri2[I], kapi[I];
    double nx[I], ny[I], nz[I], ax[I], ay[I], az[I], S[I], Yx[I], Yy[I], Yz[I], H[I], Vx[I], Vy[I], Vz[I], U[I];
    int ii[I];
#pragma unroll
    for (int k = 0; k < I; ++k) {
        ii[k] = blockIdx.x * (I * NT) + tid + k * NT;
        const CRec c = crec[ii[k]];
        xi[k] = c.x, yi[k] = c.y, zi[k] = c.z, vxi[k] = c.vx, vyi[k] = c.vy, vzi[k] = c.vz;
        ri2[k] = c.rj2, kapi[k] = c.kap;
        nx[k] = ny[k] = nz[k] = ax[k] = ay[k] = az[k] = S[k] = Yx[k] = Yy[k] = Yz[k] = H[k] = Vx[k] = Vy[k] = Vz[k] = U[k] = 0.0;
    }
    const int n_tiles = np / TJ;
    const int t_begin = blockIdx.y * tiles_per_split;
    const int t_end = min(n_tiles, t_begin + tiles_per_split);
    constexpr int kVec = TJ * 7;  // double2 per tile
    auto fill = [&](int buf, int t) {
        const double2* src = reinterpret_cast<const double2*>(crec + (size_t)t * TJ);
        double2* dst = reinterpret_cast<double2*>(sj[buf]);
        for (int q = tid; q < kVec; q += NT) dst[q] = src[q];
    };
    if (t_begin < t_end) fill(0, t_begin);
    __syncthreads();
    for (int t = t_begin; t < t_end; ++t) {
        const int buf = (t - t_begin) & 1;
        if (t + 1 < t_end) fill(buf ^ 1, t + 1);
        const CRec* tile = sj[buf];
        const int j0 = t * TJ;
        // j != i by index (with eps > 0 the self term does not cancel in these sums): only a tile that overlaps the block's own
        // i range can hold a self pair, so all other tiles run a body without the compare and the two selects per pair
        auto walk_tile = [&](auto masked) {
#pragma unroll 2
            for (int jj = 0; jj < TJ; ++jj) {
                const CRec r = tile[jj];
#pragma unroll
                for (int k = 0; k < I; ++k) {
                    const double dx = xi[k] - r.x, dy = yi[k] - r.y, dz = zi[k] - r.z;  // x_ij
                    const double r2 = fma(dx, dx, fma(dy, dy, fma(dz, dz, eps2)));
                    const double y0 = rsqrt_seed(r2);
                    const double e = fma(-r2, y0 * y0, 1.0);
                    double y = fma(y0 * e, fma(e, 0.375, 0.5), y0);  // 1 / rho to full fp64 accuracy
                    double gm = r.gm;
                    if (decltype(masked)::value) {
                        const bool self = (j0 + jj == ii[k]);
                        y = self ? 0.0 : y;
                        gm = self ? 0.0 : gm;
                    }
                    const double y2 = y * y;
                    const double s = gm * (y2 * y);  // G m_j / rho^3
                    nx[k] = fma(-s, dx, nx[k]), ny[k] = fma(-s, dy, ny[k]), nz[k] = fma(-s, dz, nz[k]);
                    const double ux = vxi[k] - r.vx, uy = vyi[k] - r.vy, uz = vzi[k] - r.vz;  // v_ij
                    const double uu = fma(ux, ux, fma(uy, uy, uz * uz));
                    const double vjx = fma(r.vx, dx, fma(r.vy, dy, r.vz * dz));
                    const double vix = fma(vxi[k], dx, fma(vyi[k], dy, vzi[k] * dz));
                    double g = fma(r2 - ri2[k], r.b, r.a5) + kapi[k];
                    g = fma(-2.0, uu, g);
                    g = fma(1.5, (vjx * vjx) * y2, g);
                    const double sg = s * g;
                    ax[k] = fma(sg, dx, ax[k]), ay[k] = fma(sg, dy, ay[k]), az[k] = fma(sg, dz, az[k]);
                    S[k] = fma(gm, fma(-r2, r.b, GM4 * y), S[k]);
                    Yx[k] = fma(y, r.wx, Yx[k]), Yy[k] = fma(y, r.wy, Yy[k]), Yz[k] = fma(y, r.wz, Yz[k]);
                    const double h = s * fma(4.0, vix, -3.0 * vjx);
                    H[k] += h;
                    Vx[k] = fma(h, r.vx, Vx[k]), Vy[k] = fma(h, r.vy, Vy[k]), Vz[k] = fma(h, r.vz, Vz[k]);
                    if (BHX) U[k] = fma(gm * y, fma((ri2[k] - r.rj2) * y2, 0.25, 1.25), U[k]);
                }
            }
        };
        const int i_lo = blockIdx.x * (I * NT);
        if (j0 + TJ > i_lo && j0 < i_lo + I * NT)
            walk_tile(std::true_type{});
        else
            walk_tile(std::false_type{});
        __syncthreads();
    }
    double* out = part + (size_t)blockIdx.y * NC * np;
#pragma unroll
    for (int k = 0; k < I; ++k) {
        out[ii[k]] = nx[k], out[np + ii[k]] = ny[k], out[2 * np + ii[k]] = nz[k];
        out[3 * np + ii[k]] = ax[k] + Yx[k] + fma(H[k], vxi[k], -Vx[k]);
        out[4 * np + ii[k]] = ay[k] + Yy[k] + fma(H[k], vyi[k], -Vy[k]);
        out[5 * np + ii[k]] = az[k] + Yz[k] + fma(H[k], vzi[k], -Vz[k]);
        out[6 * np + ii[k]] = S[k];
        if (BHX) out[7 * np + ii[k]] = U[k];
    }
}

// ---- the symmetric form: every unordered pair once.  One-warp blocks, I = 2 i-stars per lane, unit tiles of U = 64 stars,
// the work-item / slot scheme of pair_sym_fp64_kernel (block (A <= B) of a triangular grid over G groups of m tiles: row
// sums to slot B, column sums to slot A, one writer per (slot, star), nothing zeroed, no atomics).
#ifndef PN_CROSS_STEPS
#define PN_CROSS_STEPS 8
#endif
constexpr int kCrossSymI = 2;
constexpr int kCrossSymU = 32 * kCrossSymI;
template <bool BHX>
constexpr int kCrossSymSmemBytes = kCrossSymU * (2 * (int)sizeof(CRec) + kCrossNC<BHX> * 8);

struct CrossAcc {  // the sums of one star: n (3), X (3), S, U
    double n[3], X[3], S, U;
};

// one ordered or unordered pair: i-star (register state) against the j record r.  SYM: also the reversed pair into b.
// EQM (every star has the same mass; the record's w is per unit G m): every sum is proportional to the common G m, which is
// applied once, at the flush: s = y^3 for both directions and the mass factors of S and U go (72 instead of 76 FP64
// instructions per unordered pair, 80 instead of 84 with U).
template <bool SYM, bool BHX, bool EQM>
__device__ __forceinline__ void cross_pair(const CRec& r, const double (&xi)[3], const double (&vi)[3], double ri2, double kapi,
                                           double gmi, double a5i, double bi, const double (&wi)[3], CrossAcc& a, CrossAcc& b,
                                           double eps2, double GM4, bool self)
{
    const double d[3] = {xi[0] - r.x, xi[1] - r.y, xi[2] - r.z};  // x_ij
    const double r2 = fma(d[0], d[0], fma(d[1], d[1], fma(d[2], d[2], eps2)));
    const double y0 = rsqrt_seed(r2);
    const double e = fma(-r2, y0 * y0, 1.0);
    double y = fma(y0 * e, fma(e, 0.375, 0.5), y0);  // 1 / rho to full fp64 accuracy
    double gmj = r.gm;
    if (!SYM) {  // diagonal unit tile, ordered pairs: j != i in every sum of Eq. 2.6 (eps > 0 does not cancel the self term here)
        y = self ? 0.0 : y;
        gmj = self ? 0.0 : gmj;
    }
    const double y2 = y * y, y3 = y2 * y;
    const double u[3] = {vi[0] - r.vx, vi[1] - r.vy, vi[2] - r.vz};  // v_ij
    const double uu = fma(u[0], u[0], fma(u[1], u[1], u[2] * u[2]));
    const double vjx = fma(r.vx, d[0], fma(r.vy, d[1], r.vz * d[2]));
    const double vix = fma(vi[0], d[0], fma(vi[1], d[1], vi[2] * d[2]));
    const double da = vix - vjx;                 // u.d
    const double y4 = GM4 * y;
    const double yq = 1.2247448713915890 * y;    // sqrt(3/2) / rho
    double dy2 = 0.0;
    if (BHX) dy2 = (ri2 - r.rj2) * y2;
    {   // i <- j
        const double s = EQM ? y3 : gmj * y3;
        const double pj = vjx * yq;
        const double g = fma(pj, pj, fma(r2 - ri2, r.b, r.a5) + fma(-2.0, uu, kapi));
        const double sg = s * g;
        const double h = s * fma(3.0, da, vix);  // s (4 v_i.d - 3 v_j.d)
#pragma unroll
        for (int c = 0; c < 3; ++c) a.n[c] = fma(-s, d[c], a.n[c]);
        a.X[0] = fma(y, r.wx, fma(h, u[0], fma(sg, d[0], a.X[0])));
        a.X[1] = fma(y, r.wy, fma(h, u[1], fma(sg, d[1], a.X[1])));
        a.X[2] = fma(y, r.wz, fma(h, u[2], fma(sg, d[2], a.X[2])));
        if (EQM) {
            const double ts = fma(-r2, r.b, y4);
            a.S += (!SYM && self) ? 0.0 : ts;
            if (BHX) a.U = fma(y, fma(dy2, 0.25, 1.25), a.U);
        } else {
            a.S = fma(gmj, fma(-r2, r.b, y4), a.S);
            if (BHX) a.U = fma(gmj * y, fma(dy2, 0.25, 1.25), a.U);
        }
    }
    if (SYM) {  // j <- i: d -> -d, u -> -u
        const double s = EQM ? y3 : gmi * y3;
        const double pi = vix * yq;
        const double g = fma(pi, pi, fma(r2 - r.rj2, bi, a5i) + fma(-2.0, uu, r.kap));
        const double sg = s * g;
        const double h = s * fma(3.0, da, -vjx);  // s (3 v_i.d - 4 v_j.d)
#pragma unroll
        for (int c = 0; c < 3; ++c) b.n[c] = fma(s, d[c], b.n[c]);
#pragma unroll
        for (int c = 0; c < 3; ++c) b.X[c] = fma(y, wi[c], fma(-h, u[c], fma(-sg, d[c], b.X[c])));
        if (EQM) {
            b.S += fma(-r2, bi, y4);
            if (BHX) b.U = fma(y, fma(dy2, -0.25, 1.25), b.U);
        } else {
            b.S = fma(gmi, fma(-r2, bi, y4), b.S);
            if (BHX) b.U = fma(gmi * y, fma(dy2, -0.25, 1.25), b.U);
        }
    }
}

__device__ __forceinline__ void cross_acc_zero(CrossAcc& a)
{
    a.n[0] = a.n[1] = a.n[2] = a.X[0] = a.X[1] = a.X[2] = a.S = a.U = 0.0;
}

template <bool BHX>
__device__ __forceinline__ void cross_acc_shfl(CrossAcc& a, int mask)
{
#pragma unroll
    for (int c = 0; c < 3; ++c) a.n[c] = __shfl_xor_sync(0xffffffffu, a.n[c], mask), a.X[c] = __shfl_xor_sync(0xffffffffu, a.X[c], mask);
    a.S = __shfl_xor_sync(0xffffffffu, a.S, mask);
    if (BHX) a.U = __shfl_xor_sync(0xffffffffu, a.U, mask);
}

__device__ __forceinline__ void cp_async16(void* dst_smem, const void* src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((unsigned int)__cvta_generic_to_shared(dst_smem)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

template <int MINB, bool BHX, bool EQM, int CSTEPS = PN_CROSS_STEPS>
__global__ void __launch_bounds__(32, MINB) pair_cross_sym_kernel(const CRec* __restrict__ crec, double* __restrict__ part /* [G][NC][np] */,
                                                                  int np, int n_tiles, int m, double eps2, double GM4, double gm_eq)
{
    constexpr int I = kCrossSymI, U = kCrossSymU, NC = kCrossNC<BHX>;
    extern __shared__ double2 sym_smem[];
    // two j tiles (the next one is on its way, cp.async, while the current one is evaluated), then [NC][U] column / row sums
    double(*cacc)[U] = reinterpret_cast<double(*)[U]>(sym_smem + 2 * U * 7);
    const int lane = threadIdx.x;
    int A, B;
    sym_decode_block(blockIdx.x, A, B);
    const int ta0 = A * m, ta1 = min(ta0 + m, n_tiles);
    const int tb0 = B * m, tb1 = min(tb0 + m, n_tiles);

    auto fetch_tile = [&](int buf, int tile) {
        const double2* src = reinterpret_cast<const double2*>(crec + (size_t)tile * U);
        double2* dst = sym_smem + buf * (U * 7);
#pragma unroll
        for (int q = lane; q < U * 7; q += 32) cp_async16(dst + q, src + q);
        cp_async_commit();
    };
    auto store_acc = [&](const CrossAcc& a, int el) {
        cacc[0][el] = a.n[0], cacc[1][el] = a.n[1], cacc[2][el] = a.n[2];
        cacc[3][el] = a.X[0], cacc[4][el] = a.X[1], cacc[5][el] = a.X[2];
        cacc[6][el] = a.S;
        if (BHX) cacc[7][el] = a.U;
    };
    // cacc -> part[slot][NC][tile].  Every element of part has ONE writer in the whole launch -- the same lane of the same block every
    // time -- so its first contribution is a plain store and the later ones are reductions to the same address by the same thread
    // (RED.ADD.F64: applied in program order, nothing to wait for), which keeps the sum's order fixed without a read-modify-write
    auto flush = [&](int slot, int tile, bool first) {
        double* dst = part + (size_t)slot * NC * np + (size_t)tile * U;
#pragma unroll
        for (int c = 0; c < NC; ++c)
#pragma unroll
            for (int q = lane; q < U; q += 32) {
                double* p = dst + (size_t)c * np + q;
                const double v = EQM ? cacc[c][q] * gm_eq : cacc[c][q];
                if (first)
                    *p = v;
                else
                    atomicAdd(p, v);
            }
    };

    int buf = 0;
    fetch_tile(0, (A == B) ? ta0 : tb0);
    for (int ta = ta0; ta < ta1; ++ta) {
        double xi[I][3], vi[I][3], ri2[I], kapi[I], gmi[I], a5i[I], bi[I], wi[I][3];
        CrossAcc acc[I];
#pragma unroll
        for (int k = 0; k < I; ++k) {
            const CRec c = crec[(size_t)ta * U + lane + 32 * k];
            xi[k][0] = c.x, xi[k][1] = c.y, xi[k][2] = c.z, vi[k][0] = c.vx, vi[k][1] = c.vy, vi[k][2] = c.vz;
            ri2[k] = c.rj2, kapi[k] = c.kap, gmi[k] = c.gm, a5i[k] = c.a5, bi[k] = c.b;
            wi[k][0] = c.wx, wi[k][1] = c.wy, wi[k][2] = c.wz;
            cross_acc_zero(acc[k]);
        }
        for (int tb = (A == B) ? ta : tb0; tb < tb1; ++tb) {
            cp_async_wait_all();
            __syncwarp();  // the tile is there, and everyone is done with the other buffer
            {   // the next tile of this item's walk, if any
                int nt = tb + 1;
                if (nt >= tb1) nt = (ta + 1 < ta1) ? ((A == B) ? ta + 1 : tb0) : -1;
                if (nt >= 0) fetch_tile(buf ^ 1, nt);
            }
            const CRec* sj = reinterpret_cast<const CRec*>(sym_smem + buf * (U * 7));
            if (ta == tb) {  // diagonal unit tile: ordered pairs, i-side only, j != i by index
                CrossAcc dummy;
                cross_acc_zero(dummy);
#pragma unroll 1
                for (int jj = 0; jj < U; ++jj) {
                    const CRec r = sj[jj];
#pragma unroll
                    for (int k = 0; k < I; ++k)
                        cross_pair<false, BHX, EQM>(r, xi[k], vi[k], ri2[k], kapi[k], gmi[k], a5i[k], bi[k], wi[k], acc[k], dummy, eps2, GM4,
                                               jj == lane + 32 * k);
                }
            } else {
#pragma unroll 1
                for (int jb = 0; jb < U; jb += 32) {
                    CrossAcc b;
                    cross_acc_zero(b);
#pragma unroll 1
                    for (int c = 0; c < 32 / CSTEPS; ++c) {  // Gray-code walk in chunks of CSTEPS steps (see sym_unit_tile_gray)
                        const int r0 = CSTEPS * c, r1 = r0 + CSTEPS - 1, r2 = (r0 + CSTEPS) & 31;  // g(r) = r ^ (r >> 1)
                        const int base = jb + (lane ^ (r0 ^ (r0 >> 1)));
                        const int last_mask = (r1 ^ (r1 >> 1)) ^ (r2 ^ (r2 >> 1));  // into the next chunk or, after step 31, home
#pragma unroll
                        for (int q = 0; q < CSTEPS; ++q) {
                            const CRec r = sj[base ^ (q ^ (q >> 1))];
#pragma unroll
                            for (int k = 0; k < I; ++k)
                                cross_pair<true, BHX, EQM>(r, xi[k], vi[k], ri2[k], kapi[k], gmi[k], a5i[k], bi[k], wi[k], acc[k], b, eps2, GM4, false);
                            cross_acc_shfl<BHX>(b, (q + 1 < CSTEPS) ? ((q + 1) & -(q + 1)) : last_mask);
                        }
                    }
                    store_acc(b, jb + lane);
                }
                __syncwarp();
                flush(A, tb, ta == ta0);  // column sums: the i-stars of tile ta acting on the j-stars of tile tb
                __syncwarp();
            }
            buf ^= 1;
        }
#pragma unroll
        for (int k = 0; k < I; ++k) store_acc(acc[k], lane + 32 * k);
        __syncwarp();
        flush(B, ta, (A < B) || (ta == ta0));  // row sums: the j-stars of group B acting on the i-stars of tile ta
        __syncwarp();
    }
}

// ---------------------------------------------------------------------------------------------------------
// S1 variant: fp32 pair arithmetic, fp64 accumulation (PN_FP32_PAIR, parity 1e-5).
// Positions are split into two floats, hi = fl32(x), lo = fl32(x - hi), so that the pair separation
//   d = (hi_j - hi_i) + (lo_j - lo_i)
// keeps a relative accuracy of ~1e-7 of |d| even for close pairs (a position ~1 has fp32 spacing 6e-8 while the
// softening is 1e-3...1e-4).  Per ordered pair: 9 FADD + 6 FFMA + 3 FMUL = 18 FP32-pipe instructions + 1 MUFU.RSQ.
// fp32 partial sums run over FL consecutive j only and are then flushed into fp64 accumulators.
// ---------------------------------------------------------------------------------------------------------
__device__ __forceinline__ float rsqrt_seed_f32(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));  // MUFU.RSQ
    return y;
}

struct __align__(16) FRec {
    float xh, yh, zh, gm;  // high parts, G m_j
    float xl, yl, zl, pad; // low parts
};
static_assert(sizeof(FRec) == 32, "FRec must be 32 bytes");

constexpr float kPadPosF = 1e15f;  // pad stars for the fp32 kernel: finite r^2, zero mass

__global__ void split_kernel(const JRec* __restrict__ jrec, FRec* __restrict__ frec, int n_stars, int np)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= np) return;
    FRec f;
    if (i < n_stars) {
        const JRec r = jrec[i];
        f.xh = (float)r.x, f.yh = (float)r.y, f.zh = (float)r.z;
        f.xl = (float)(r.x - (double)f.xh), f.yl = (float)(r.y - (double)f.yh), f.zl = (float)(r.z - (double)f.zh);
        f.gm = (float)r.gm;
    } else {
        f.xh = f.yh = f.zh = kPadPosF;
        f.xl = f.yl = f.zl = 0.f, f.gm = 0.f;
    }
    f.pad = 0.f;
    frec[i] = f;
}

// two-float records of a PAIR of consecutive stars (2 q, 2 q + 1), component by component: every 8-byte word is one packed
// operand of the f32x2 kernels (loaded as such: a 64-bit value that was never two 32-bit registers keeps its register pair)
struct __align__(16) FPair {
    float xh[2], yh[2], zh[2], gm[2];
    float xl[2], yl[2], zl[2], pad[2];
};
static_assert(sizeof(FPair) == 64, "FPair must be 64 bytes");

__global__ void split_pair_kernel(const JRec* __restrict__ jrec, FPair* __restrict__ fpair, int n_stars, int np)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= np) return;
    float xh = kPadPosF, yh = kPadPosF, zh = kPadPosF, xl = 0.f, yl = 0.f, zl = 0.f, gm = 0.f;
    if (i < n_stars) {
        const JRec r = jrec[i];
        xh = (float)r.x, yh = (float)r.y, zh = (float)r.z;
        xl = (float)(r.x - (double)xh), yl = (float)(r.y - (double)yh), zl = (float)(r.z - (double)zh);
        gm = (float)r.gm;
    }
    FPair* p = fpair + (i >> 1);
    const int h = i & 1;
    p->xh[h] = xh, p->yh[h] = yh, p->zh[h] = zh, p->gm[h] = gm;
    p->xl[h] = xl, p->yl[h] = yl, p->zl[h] = zl, p->pad[h] = 0.f;
}

template <int I, int NT, int TJ, int FL, bool MASK>
__global__ void __launch_bounds__(NT) pair_fp32_kernel(const FRec* __restrict__ frec, double* __restrict__ part, int np,
                                                       int tiles_per_split, float eps2)
{
    static_assert(TJ % FL == 0, "tile must be a multiple of the flush interval");
    __shared__ FRec sj[2][TJ];
    const int tid = threadIdx.x;
    const int i_base = blockIdx.x * (I * NT) + tid;

    float xh[I], yh[I], zh[I], xl[I], yl[I], zl[I];
    double ax[I], ay[I], az[I];
    int ii[I];
#pragma unroll
    for (int k = 0; k < I; ++k) {
        ii[k] = i_base + k * NT;
        const FRec f = frec[ii[k]];
        xh[k] = f.xh, yh[k] = f.yh, zh[k] = f.zh, xl[k] = f.xl, yl[k] = f.yl, zl[k] = f.zl;
        ax[k] = ay[k] = az[k] = 0.0;
    }
    const int n_tiles = np / TJ;
    const int t_begin = blockIdx.y * tiles_per_split;
    const int t_end = min(n_tiles, t_begin + tiles_per_split);
    auto fill = [&](int buf, int t) {
        const float4* src = reinterpret_cast<const float4*>(frec + (size_t)t * TJ);
        float4* dst = reinterpret_cast<float4*>(sj[buf]);
        for (int q = tid; q < TJ * 2; q += NT) dst[q] = src[q];
    };
    if (t_begin < t_end) fill(0, t_begin);
    __syncthreads();
    for (int t = t_begin; t < t_end; ++t) {
        const int buf = (t - t_begin) & 1;
        if (t + 1 < t_end) fill(buf ^ 1, t + 1);
        const FRec* tile = sj[buf];
        const int j0 = t * TJ;
#pragma unroll 1
        for (int jb = 0; jb < TJ; jb += FL) {
            float fx[I], fy[I], fz[I];
#pragma unroll
            for (int k = 0; k < I; ++k) fx[k] = fy[k] = fz[k] = 0.f;
#pragma unroll 4
            for (int jj = jb; jj < jb + FL; ++jj) {
                const FRec r = tile[jj];
#pragma unroll
                for (int k = 0; k < I; ++k) {
                    const float dx = (r.xh - xh[k]) + (r.xl - xl[k]);
                    const float dy = (r.yh - yh[k]) + (r.yl - yl[k]);
                    const float dz = (r.zh - zh[k]) + (r.zl - zl[k]);
                    const float r2 = fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps2)));
                    const float y = rsqrt_seed_f32(r2);
                    float s = (y * y) * (y * r.gm);
                    if (MASK) s = (j0 + jj == ii[k]) ? 0.f : s;
                    fx[k] = fmaf(s, dx, fx[k]);
                    fy[k] = fmaf(s, dy, fy[k]);
                    fz[k] = fmaf(s, dz, fz[k]);
                }
            }
#pragma unroll
            for (int k = 0; k < I; ++k) ax[k] += (double)fx[k], ay[k] += (double)fy[k], az[k] += (double)fz[k];
        }
        __syncthreads();
    }
    double* out = part + (size_t)blockIdx.y * 3 * np;
#pragma unroll
    for (int k = 0; k < I; ++k) {
        out[ii[k]] = ax[k];
        out[np + ii[k]] = ay[k];
        out[2 * np + ii[k]] = az[k];
    }
}

// ---------------------------------------------------------------------------------------------------------
// S1 variant, symmetric form: fp32 pair arithmetic on two-float positions, every unordered pair once (same
// decomposition, rotation and slot scheme as pair_sym_fp64_kernel), on the PACKED fp32 instructions of sm_100
// (add / mul / fma.rn.f32x2 -> FADD2 / FMUL2 / FFMA2: one instruction, two lanes of a 64-bit register pair).
// A lane's I = 4 i-stars form two packed pairs (k, k + 1); the j-star's components are stored twice in shared memory
// ({x, x}, {y, y}, ...), so one LDS.128 delivers two ready-made packed operands.  Per TWO unordered pairs:
//   d = (h_j - h_i) + (l_j - l_i)   9 FADD2      r2 = d.d + eps^2   3 FFMA2      y = MUFU.RSQ (scalar, one per pair)
//   K = y y y                       2 FMUL2      f_i += K d         3 FFMA2      b_j += K d   3 FFMA2
// = 20 packed instructions for two pairs (general masses: + 2 FMUL2), i.e. half the issue slots of the scalar form
// (the scalar kernel was bound by the one issue port of a sub-partition, not by the FMA pipe: profiles/r1_ncu_summary.md
// section 11).  Counted per ordered pair in fp32 operations as before: 10 (equal masses) or 11.
// The j-side sums of the two packed lanes travel together (a 64-bit SHFL per component and step) and are added at the
// end of the rotation; the i-side fp32 sums run over the 32 steps of one rotation, the j-side sums over its 64 terms per
// packed lane; both are then added in fp64.
// ---------------------------------------------------------------------------------------------------------
typedef unsigned long long f32x2;  // {lo, hi}: two floats in a 64-bit register pair

__device__ __forceinline__ f32x2 pack2(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

// shared-memory image of a j tile for the packed kernels: every component twice, so that a 16-byte load is two packed
// operands; one array per 16-byte group keeps consecutive lanes on consecutive banks
struct Sym32Tile {
    ulonglong2* a;  // [U] {xh, xh}, {yh, yh}
    ulonglong2* b;  // [U] {zh, zh}, {xl, xl}
    ulonglong2* c;  // [U] {yl, yl}, {zl, zl}
    f32x2* g;       // [U] {G m_j, G m_j}
};

template <int U, bool SYM, bool MASK, bool EQM>
__device__ __forceinline__ void sym32_unit_tile(const Sym32Tile& tj, float* __restrict__ cw /* this warp's [3][U] column sums */,
                                                const f32x2 (&xh)[2], const f32x2 (&yh)[2], const f32x2 (&zh)[2],
                                                const f32x2 (&xl)[2], const f32x2 (&yl)[2], const f32x2 (&zl)[2],
                                                const f32x2 (&ngi)[2], double (&ax)[4], double (&ay)[4], double (&az)[4],
                                                f32x2 eps2, int lane, int i_local0, int jb0, int jb1)
{
#pragma unroll 1
    for (int jb = jb0; jb < jb1; jb += 32) {
        f32x2 fx[2], fy[2], fz[2];
#pragma unroll
        for (int g = 0; g < 2; ++g) fx[g] = fy[g] = fz[g] = 0ull;
        f32x2 bx = 0ull, by = 0ull, bz = 0ull;
#pragma unroll 4
        for (int r = 0; r < 32; ++r) {
            const int jj = jb + ((lane + r) & 31);
            const ulonglong2 ja = tj.a[jj], jbv = tj.b[jj], jc = tj.c[jj];
            f32x2 gmj = 0ull;
            if (!EQM) gmj = tj.g[jj];
#pragma unroll
            for (int g = 0; g < 2; ++g) {
                const f32x2 dx = add2(sub2(ja.x, xh[g]), sub2(jbv.y, xl[g]));
                const f32x2 dy = add2(sub2(ja.y, yh[g]), sub2(jc.x, yl[g]));
                const f32x2 dz = add2(sub2(jbv.x, zh[g]), sub2(jc.y, zl[g]));
                const f32x2 r2 = fma2(dx, dx, fma2(dy, dy, fma2(dz, dz, eps2)));
                float r2a, r2b;
                unpack2(r2, r2a, r2b);
                float ya = rsqrt_seed_f32(r2a), yb = rsqrt_seed_f32(r2b);
                if (MASK) {  // diagonal unit tile with eps == 0: the self pair would be 0 * inf
                    ya = (jj == i_local0 + 64 * g) ? 0.f : ya;
                    yb = (jj == i_local0 + 64 * g + 1) ? 0.f : yb;
                }
                const f32x2 y = pack2(ya, yb);
                const f32x2 K = mul2(mul2(y, y), y);
                const f32x2 sj = EQM ? K : mul2(K, gmj);  // EQM: the common G m is applied at the flush
                fx[g] = fma2(sj, dx, fx[g]);
                fy[g] = fma2(sj, dy, fy[g]);
                fz[g] = fma2(sj, dz, fz[g]);
                if (SYM) {  // EQM: + K d is accumulated and the sign is turned at the end of the rotation
                    const f32x2 si = EQM ? K : mul2(K, ngi[g]);
                    bx = fma2(si, dx, bx);
                    by = fma2(si, dy, by);
                    bz = fma2(si, dz, bz);
                }
            }
            if (SYM) {
                const int src = (lane + 1) & 31;
                bx = __shfl_sync(0xffffffffu, bx, src);
                by = __shfl_sync(0xffffffffu, by, src);
                bz = __shfl_sync(0xffffffffu, bz, src);
            }
        }
#pragma unroll
        for (int g = 0; g < 2; ++g) {
            float lo, hi;
            unpack2(fx[g], lo, hi), ax[2 * g] += (double)lo, ax[2 * g + 1] += (double)hi;
            unpack2(fy[g], lo, hi), ay[2 * g] += (double)lo, ay[2 * g + 1] += (double)hi;
            unpack2(fz[g], lo, hi), az[2 * g] += (double)lo, az[2 * g + 1] += (double)hi;
        }
        if (SYM) {
            float lo, hi;
            unpack2(bx, lo, hi), cw[jb + lane] = EQM ? -(lo + hi) : (lo + hi);
            unpack2(by, lo, hi), cw[U + jb + lane] = EQM ? -(lo + hi) : (lo + hi);
            unpack2(bz, lo, hi), cw[2 * U + jb + lane] = EQM ? -(lo + hi) : (lo + hi);
        }
    }
}

// the same unit tile walked in Gray-code order (see sym_unit_tile_gray): butterfly shuffles with immediate masks
template <int U, bool EQM>
__device__ __forceinline__ void sym32_unit_tile_gray(const Sym32Tile& tj, float* __restrict__ cw, const f32x2 (&xh)[2],
                                                     const f32x2 (&yh)[2], const f32x2 (&zh)[2], const f32x2 (&xl)[2],
                                                     const f32x2 (&yl)[2], const f32x2 (&zl)[2], const f32x2 (&ngi)[2],
                                                     double (&ax)[4], double (&ay)[4], double (&az)[4], f32x2 eps2, int lane,
                                                     int jb0, int jb1)
{
#pragma unroll 1
    for (int jb = jb0; jb < jb1; jb += 32) {
        f32x2 fx[2], fy[2], fz[2];
#pragma unroll
        for (int g = 0; g < 2; ++g) fx[g] = fy[g] = fz[g] = 0ull;
        f32x2 bx = 0ull, by = 0ull, bz = 0ull;
#pragma unroll 1
        for (int c = 0; c < 2; ++c) {
            const int base = jb + (lane ^ (c ? 24 : 0));
#pragma unroll
            for (int q = 0; q < 16; ++q) {
                const int jj = base ^ (q ^ (q >> 1));
                const ulonglong2 ja = tj.a[jj], jbv = tj.b[jj], jc = tj.c[jj];
                f32x2 gmj = 0ull;
                if (!EQM) gmj = tj.g[jj];
#pragma unroll
                for (int g = 0; g < 2; ++g) {
                    const f32x2 dx = add2(sub2(ja.x, xh[g]), sub2(jbv.y, xl[g]));
                    const f32x2 dy = add2(sub2(ja.y, yh[g]), sub2(jc.x, yl[g]));
                    const f32x2 dz = add2(sub2(jbv.x, zh[g]), sub2(jc.y, zl[g]));
                    const f32x2 r2 = fma2(dx, dx, fma2(dy, dy, fma2(dz, dz, eps2)));
                    float r2a, r2b;
                    unpack2(r2, r2a, r2b);
                    const f32x2 y = pack2(rsqrt_seed_f32(r2a), rsqrt_seed_f32(r2b));
                    const f32x2 K = mul2(mul2(y, y), y);
                    const f32x2 sj = EQM ? K : mul2(K, gmj);
                    fx[g] = fma2(sj, dx, fx[g]);
                    fy[g] = fma2(sj, dy, fy[g]);
                    fz[g] = fma2(sj, dz, fz[g]);
                    const f32x2 si = EQM ? K : mul2(K, ngi[g]);
                    bx = fma2(si, dx, bx);
                    by = fma2(si, dy, by);
                    bz = fma2(si, dz, bz);
                }
                const int mask = (q + 1 < 16) ? ((q + 1) & -(q + 1)) : 16;
                bx = __shfl_xor_sync(0xffffffffu, bx, mask);
                by = __shfl_xor_sync(0xffffffffu, by, mask);
                bz = __shfl_xor_sync(0xffffffffu, bz, mask);
            }
        }
#pragma unroll
        for (int g = 0; g < 2; ++g) {
            float lo, hi;
            unpack2(fx[g], lo, hi), ax[2 * g] += (double)lo, ax[2 * g + 1] += (double)hi;
            unpack2(fy[g], lo, hi), ay[2 * g] += (double)lo, ay[2 * g + 1] += (double)hi;
            unpack2(fz[g], lo, hi), az[2 * g] += (double)lo, az[2 * g + 1] += (double)hi;
        }
        float lo, hi;
        unpack2(bx, lo, hi), cw[jb + lane] = EQM ? -(lo + hi) : (lo + hi);
        unpack2(by, lo, hi), cw[U + jb + lane] = EQM ? -(lo + hi) : (lo + hi);
        unpack2(bz, lo, hi), cw[2 * U + jb + lane] = EQM ? -(lo + hi) : (lo + hi);
    }
}

// column sums of the packed kernels: n_src per-warp [3][U] float tiles, added in fp64 in fixed warp order
template <int U, int NT>
__device__ __forceinline__ void sym32_flush_cols(const float* __restrict__ cw, double* __restrict__ dst, int np, bool first, int n_src,
                                                 int tid, double scale)
{
    for (int q = tid; q < 3 * U; q += NT) {
        const int c = q / U, el = q - c * U;
        double v = (double)cw[q];
        for (int s = 1; s < n_src; ++s) v += (double)cw[s * 3 * U + q];
        v *= scale;
        double* d = dst + (size_t)c * np + el;
        if (first)
            *d = v;
        else
            atomicAdd(d, v);
    }
}

// shared memory: the doubled j tile (56 B per star), W per-warp float column-sum tiles, one double row-sum tile
template <int W>
constexpr int kSym32SmemBytes = (W * 128) * (56 + 12 * W + 24);

template <int W, int MINB, bool MASK, bool EQM, bool GRAY = true>
__global__ void __launch_bounds__(W * 32, MINB) pair_sym_fp32_kernel(const FPair* __restrict__ fpair,
                                                                     double* __restrict__ part, int np, int n_tiles,
                                                                     int m, float eps2, double gm_eq)
{
    constexpr int I = 4;
    constexpr int U = W * 32 * I;
    constexpr int NT = W * 32;
    extern __shared__ double2 sym_smem[];  // kSym32SmemBytes<W>
    Sym32Tile tj;
    tj.a = reinterpret_cast<ulonglong2*>(sym_smem);
    tj.b = tj.a + U;
    tj.c = tj.b + U;
    tj.g = reinterpret_cast<f32x2*>(tj.c + U);
    double* rowd = reinterpret_cast<double*>(tj.g + U);         // [3][U] row sums (fp64)
    float* cwf = reinterpret_cast<float*>(rowd + 3 * U);        // [W][3][U] per-warp column sums
    const int item = blockIdx.x;
    const int tid = threadIdx.x, w = tid >> 5, lane = tid & 31;
    int A, B;
    sym_decode_block(item, A, B);
    const int ta0 = A * m, ta1 = min(ta0 + m, n_tiles);
    const int tb0 = B * m, tb1 = min(tb0 + m, n_tiles);
    // this lane's i-stars: packed pair g holds the consecutive stars i_local0 + 64 g and i_local0 + 64 g + 1 of the unit tile
    const int i_local0 = w * 32 * I + 2 * lane;
    const f32x2 eps2p = pack2(eps2, eps2);
    const f32x2 minus1 = pack2(-1.f, -1.f);
    const double scale = EQM ? gm_eq : 1.0;

    for (int ta = ta0; ta < ta1; ++ta) {
        f32x2 xh[2], yh[2], zh[2], xl[2], yl[2], zl[2], ngi[2];
        double ax[I], ay[I], az[I];
#pragma unroll
        for (int g = 0; g < 2; ++g) {
            const ulonglong2* p = reinterpret_cast<const ulonglong2*>(fpair + (((size_t)ta * U + i_local0 + 64 * g) >> 1));
            const ulonglong2 q0 = p[0], q1 = p[1], q2 = p[2], q3 = p[3];
            xh[g] = q0.x, yh[g] = q0.y, zh[g] = q1.x, ngi[g] = mul2(q1.y, minus1);
            xl[g] = q2.x, yl[g] = q2.y, zl[g] = q3.x;
        }
#pragma unroll
        for (int k = 0; k < I; ++k) ax[k] = ay[k] = az[k] = 0.0;
        for (int tb = (A == B) ? ta : tb0; tb < tb1; ++tb) {
            sym_sync<W>();
            for (int q = tid; q < U; q += NT) {
                const FPair* f = fpair + (((size_t)tb * U + q) >> 1);
                const int h = q & 1;
                tj.a[q] = make_ulonglong2(pack2(f->xh[h], f->xh[h]), pack2(f->yh[h], f->yh[h]));
                tj.b[q] = make_ulonglong2(pack2(f->zh[h], f->zh[h]), pack2(f->xl[h], f->xl[h]));
                tj.c[q] = make_ulonglong2(pack2(f->yl[h], f->yl[h]), pack2(f->zl[h], f->zl[h]));
                tj.g[q] = pack2(f->gm[h], f->gm[h]);
            }
            sym_sync<W>();
            if (ta == tb) {
                sym32_unit_tile<U, false, MASK, EQM>(tj, cwf + w * 3 * U, xh, yh, zh, xl, yl, zl, ngi, ax, ay, az, eps2p, lane, i_local0, 0, U);
            } else {
                if (GRAY)
                    sym32_unit_tile_gray<U, EQM>(tj, cwf + w * 3 * U, xh, yh, zh, xl, yl, zl, ngi, ax, ay, az, eps2p, lane, 0, U);
                else
                    sym32_unit_tile<U, true, false, EQM>(tj, cwf + w * 3 * U, xh, yh, zh, xl, yl, zl, ngi, ax, ay, az, eps2p, lane, i_local0, 0, U);
                sym_sync<W>();
                sym32_flush_cols<U, NT>(cwf, part + (size_t)A * 3 * np + (size_t)tb * U, np, ta == ta0, W, tid, scale);
            }
        }
        sym_sync<W>();
#pragma unroll
        for (int k = 0; k < I; ++k) {  // star k of this lane: pair k / 2, half k % 2
            const int el = i_local0 + 64 * (k >> 1) + (k & 1);
            rowd[el] = ax[k];
            rowd[U + el] = ay[k];
            rowd[2 * U + el] = az[k];
        }
        sym_sync<W>();
        sym_flush<U, NT>(rowd, part + (size_t)B * 3 * np + (size_t)ta * U, np, (A < B) || (ta == ta0), 1, tid, scale);
    }
}

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
    static_assert(NW == 4, "the fixed-order cross-warp sum below is written for 4 warps");
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
        for (int k = 0; k < NC; ++k) ss[k] = ((wsum[0][k][lane] + wsum[1][k][lane]) + wsum[2][k][lane]) + wsum[3][k][lane];
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
// reports (pn_api.cu: small_check) instead of a hung device.
__device__ __forceinline__ void small_grid_barrier(unsigned int* ctr, unsigned int target)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();  // this block's global writes are visible before its arrival is
        atomicAdd(ctr, 1u);
        unsigned int seen, polls = 0;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(ctr) : "memory");
            if (++polls == (1u << 26)) {
                atomicExch(ctr + 1, 1u);
                break;
            }
        } while ((int)(seen - target) < 0);
    }
    __syncthreads();
}

template <int MODE, int IW, int JU, bool MASK>
__global__ void __launch_bounds__(kSmallNT, 1) small_path_kernel(SmallArgs A)
{
    extern __shared__ double2 small_smem[];              // JRec[np]: this block's copy of the stage records
    JRec* sj = reinterpret_cast<JRec*>(small_smem);
    __shared__ double red[3 * (kSmallNT / 32)];
    __shared__ BhState sbh;
    __shared__ __align__(8) unsigned long long fill_bar;  // completion of the bulk copy of the stage records
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
        small_grid_barrier(A.bar, target);
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
        small_grid_barrier(A.bar, target);
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

// ---------------------------------------------------------------------------------------------------------
// S5: total 1PN energy, Eq. 2.7, regrouped:
//   E = 1/2 M v_1^2 + sum_i e_i + (1/c^2) 1/2 G^2 M (sum_i m_i/r_1i)^2 + sum_{i < j} Epair(i, j)
//   e_i = 1/2 m v^2 - GMm/r + (1/c^2){3/8 m v^4 + 3/2 (GMm/r) v^2 + 1/2 G^2M^2 m/r^2
//                                    + 1/2 (GMm/r)[3 v_1^2 - 7 v_1.v_i - (n_1i.v_1)(n_1i.v_i)]}
//   Epair(i,j) = (G m_i m_j / rho){-1 + (1/c^2)[w_i + w_j - 7/2 v_i.v_j - 1/2 (x_ij.v_i)(x_ij.v_j)/rho^2]},
//   w_i = 3/2 v_i^2 + G M / r_1i (the record stores w_i / c^2).
// All sums are compensated (TwoSum): a (hi, lo) pair per thread, per block and in the final reduction.
// ---------------------------------------------------------------------------------------------------------
struct __align__(16) ERec {
    double x, y, z, gm;     // position, G m_j
    double vx, vy, vz, w;   // velocity, w_j / c^2
};
static_assert(sizeof(ERec) == 64, "ERec must be 64 bytes");

__device__ __forceinline__ void two_sum_acc(double& hi, double& lo, double t)
{
    const double s = hi + t;
    const double bb = s - hi;
    lo += (hi - (s - bb)) + (t - bb);
    hi = s;
}

template <int NT>
__device__ __forceinline__ void block_sum_dd(double& hi, double& lo, double* smem /* 2*NT/32 */)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double oh = __shfl_down_sync(0xffffffffu, hi, o);
        const double ol = __shfl_down_sync(0xffffffffu, lo, o);
        two_sum_acc(hi, lo, oh);
        lo += ol;
    }
    constexpr int NW = NT / 32;
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) smem[w] = hi, smem[NW + w] = lo;
    __syncthreads();
    if (threadIdx.x == 0) {
        double h = 0, lw = 0;
        for (int q = 0; q < NW; ++q) {
            two_sum_acc(h, lw, smem[q]);
            lw += smem[NW + q];
        }
        hi = h, lo = lw;
    }
    __syncthreads();
}

// O(N) part: builds the ERec stream for the pair kernel and the per-block partials of sum e_i and sum m_i/r_1i.
template <int NT>
__global__ void __launch_bounds__(NT) energy_prep_kernel(const JRec* __restrict__ jrec, const double* __restrict__ v,
                                                         const BhState* __restrict__ bh, ERec* __restrict__ erec,
                                                         double* __restrict__ blk /* [grid][4]: e hi, lo; mr hi, lo */,
                                                         int n_stars, int np, double GM, double G, double inv_c2)
{
    __shared__ double red[2 * (NT / 32)];
    const int i = blockIdx.x * NT + threadIdx.x;
    double e_hi = 0, e_lo = 0, mr = 0;
    if (i < np) {
        ERec o;
        const JRec r = jrec[i];
        o.x = r.x, o.y = r.y, o.z = r.z, o.gm = r.gm;
        o.vx = o.vy = o.vz = o.w = 0.0;
        if (i < n_stars) {
            const double vv[3] = {v[i], v[np + i], v[2 * np + i]};
            const double v1[3] = {bh->vs[0], bh->vs[1], bh->vs[2]};
            const double d[3] = {bh->xs[0] - r.x, bh->xs[1] - r.y, bh->xs[2] - r.z};  // x_1i
            const double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
            const double inv_r = 1.0 / sqrt(r2);
            const double m = r.gm / G;
            const double v2 = vv[0] * vv[0] + vv[1] * vv[1] + vv[2] * vv[2];
            const double v12 = v1[0] * v1[0] + v1[1] * v1[1] + v1[2] * v1[2];
            const double v1v = v1[0] * vv[0] + v1[1] * vv[1] + v1[2] * vv[2];
            const double nv1 = (d[0] * v1[0] + d[1] * v1[1] + d[2] * v1[2]) * inv_r;
            const double nvi = (d[0] * vv[0] + d[1] * vv[1] + d[2] * vv[2]) * inv_r;
            const double U = GM * m * inv_r;  // G M m / r
            o.vx = vv[0], o.vy = vv[1], o.vz = vv[2];
            o.w = inv_c2 * (1.5 * v2 + GM * inv_r);
            two_sum_acc(e_hi, e_lo, 0.5 * m * v2);
            two_sum_acc(e_hi, e_lo, -U);
            const double pn = 0.375 * m * v2 * v2 + 1.5 * U * v2 + 0.5 * U * GM * inv_r +
                              0.5 * U * (3.0 * v12 - 7.0 * v1v - nv1 * nvi);
            two_sum_acc(e_hi, e_lo, inv_c2 * pn);
            mr = m * inv_r;
        }
        erec[i] = o;
    }
    double m_hi = mr, m_lo = 0;
    block_sum_dd<NT>(e_hi, e_lo, red);
    block_sum_dd<NT>(m_hi, m_lo, red);
    if (threadIdx.x == 0) {
        double* b = blk + 4 * (size_t)blockIdx.x;
        b[0] = e_hi, b[1] = e_lo, b[2] = m_hi, b[3] = m_lo;
    }
}

// The upper-triangular list of tile pairs (it <= jt), row by row: row it holds the n_tiles - it pairs (it, it), ..., (it, n_tiles - 1).
// Every block of the energy / momentum pair kernels takes the same number of consecutive entries of that list, so all blocks
// carry the same work to within one tile pair (the mirrored i-tile scheme of round 1 left a 12 % spread between blocks).
__device__ __forceinline__ void tri_decode(long long p, int n_tiles, int& it, int& jt)
{
    // offset(it) = it n_tiles - it (it - 1) / 2 <= p
    const double b = 2.0 * n_tiles + 1.0;
    int r = (int)((b - sqrt(b * b - 8.0 * (double)p)) * 0.5);
    r = max(0, min(r, n_tiles - 1));
    auto off = [&](int q) { return (long long)q * n_tiles - (long long)q * (q - 1) / 2; };
    while (r > 0 && off(r) > p) --r;
    while (r + 1 < n_tiles && off(r + 1) <= p) ++r;
    it = r, jt = r + (int)(p - off(r));
}

// O(N^2) part: Epair is symmetric in (i, j), so only the unordered pairs i < j are visited: tile pairs (it <= jt), thread = i-star
// of tile it, j records of tile jt broadcast from shared memory; inside the diagonal tile j <= i is masked.
template <int NT, int TJ>
__global__ void __launch_bounds__(NT) energy_pair_kernel(const ERec* __restrict__ erec, double* __restrict__ blk /* [grid][2] */,
                                                         int n_stars, int np, long long per_block, double eps2, double G, double inv_c2)
{
    __shared__ ERec sj[TJ];
    __shared__ double red[2 * (NT / 32)];
    const int tid = threadIdx.x;
    constexpr int kEGroup = 8;
    static_assert(TJ % kEGroup == 0, "tile must be a multiple of the summation group");
    static_assert(NT == TJ, "i-tiles and j-tiles share one index space");
    const double c35 = 3.5 * inv_c2, c05 = 0.5 * inv_c2;
    const int n_tiles = np / TJ;
    const long long n_pairs = (long long)n_tiles * (n_tiles + 1) / 2;
    const long long p0 = (long long)blockIdx.x * per_block, p1 = min(n_pairs, p0 + per_block);
    double hi = 0, lo = 0;      // this thread's total: sum over its i-stars of m_i * (their pair sums)
    double h_hi = 0, h_lo = 0;  // pair sum of the current i-star
    int it = 0, jt = 0;
    if (p0 < p1) tri_decode(p0, n_tiles, it, jt);
    int i = it * NT + tid;
    ERec me = erec[i];
    double wi1 = me.w - 1.0;
    auto close_row = [&]() {  // the factor m_i is common to all of star i's pairs
        if (i < n_stars) {
            const double mi = me.gm / G;
            two_sum_acc(hi, lo, h_hi * mi);
            lo += h_lo * mi;
        }
        h_hi = h_lo = 0;
    };
    for (long long p = p0; p < p1; ++p) {
        __syncthreads();
        {
            const double2* src = reinterpret_cast<const double2*>(erec + (size_t)jt * TJ);
            double2* dst = reinterpret_cast<double2*>(sj);
            for (int q = tid; q < TJ * 4; q += NT) dst[q] = src[q];
        }
        __syncthreads();
        const int j0 = jt * TJ;
        // the i < j mask is needed inside the diagonal tile only: two loop bodies, so that the 127 of 128 tile pairs off the
        // diagonal carry no compare / select per pair (two-register non-FP64 instructions cost FP64 operand bandwidth)
        auto walk_tile = [&](auto diag) {
#pragma unroll 1
            for (int jb = 0; jb < TJ; jb += kEGroup) {
                // kEGroup terms are added plainly (their sum is tiny next to the running total), then the group sum
                // goes into the compensated accumulator: one TwoSum per kEGroup pairs instead of one per pair
                double g = 0.0;
#pragma unroll
                for (int u = 0; u < kEGroup; ++u) {
                    const int jj = jb + u;
                    const ERec r = sj[jj];
                    const double dx = me.x - r.x, dy = me.y - r.y, dz = me.z - r.z;  // x_ij
                    const double r2 = fma(dx, dx, fma(dy, dy, fma(dz, dz, eps2)));
                    const double y0 = rsqrt_seed(r2);
                    const double t2 = y0 * y0;
                    const double e = fma(-r2, t2, 1.0);
                    const double y = fma(y0 * e, fma(e, 0.375, 0.5), y0);  // 1/rho to full fp64 accuracy
                    const double vv = fma(me.vx, r.vx, fma(me.vy, r.vy, me.vz * r.vz));
                    const double xvi = fma(dx, me.vx, fma(dy, me.vy, dz * me.vz));
                    const double xvj = fma(dx, r.vx, fma(dy, r.vy, dz * r.vz));
                    // q = -1 + (1/c^2)[w_i + w_j - 7/2 v_i.v_j - 1/2 (x_ij.v_i)(x_ij.v_j)/rho^2]; me.w, r.w carry the 1/c^2
                    double q = wi1 + r.w;
                    q = fma(-c35, vv, q);
                    q = fma(-c05, (xvi * xvj) * (y * y), q);
                    double term = (r.gm * y) * q;
                    if (decltype(diag)::value) term = (j0 + jj <= i) ? 0.0 : term;  // i < j only
                    g += term;
                }
                two_sum_acc(h_hi, h_lo, g);
            }
        };
        if (it == jt)
            walk_tile(std::true_type{});
        else
            walk_tile(std::false_type{});
        if (++jt == n_tiles) {  // next row of the list: the next i-tile, starting at its diagonal pair
            close_row();
            ++it, jt = it;
            if (p + 1 < p1) {
                i = it * NT + tid;
                me = erec[i];
                wi1 = me.w - 1.0;
            }
        }
    }
    close_row();
    block_sum_dd<NT>(hi, lo, red);
    if (tid == 0) {
        double* b = blk + 2 * (size_t)blockIdx.x;
        b[0] = hi, b[1] = lo;
    }
}

// Final fixed-order reduction: one block.  out[0] = E.
template <int NT>
__global__ void __launch_bounds__(NT) energy_final_kernel(const double* __restrict__ blk_prep, int n_prep,
                                                          const double* __restrict__ blk_pair, int n_pair,
                                                          const BhState* __restrict__ bh, double M, double GM, double G,
                                                          double inv_c2, double* __restrict__ out)
{
    __shared__ double red[2 * (NT / 32)];
    double e_hi = 0, e_lo = 0, m_hi = 0, m_lo = 0, p_hi = 0, p_lo = 0;
    for (int q = threadIdx.x; q < n_prep; q += NT) {
        two_sum_acc(e_hi, e_lo, blk_prep[4 * q]);
        e_lo += blk_prep[4 * q + 1];
        two_sum_acc(m_hi, m_lo, blk_prep[4 * q + 2]);
        m_lo += blk_prep[4 * q + 3];
    }
    for (int q = threadIdx.x; q < n_pair; q += NT) {
        two_sum_acc(p_hi, p_lo, blk_pair[2 * q]);
        p_lo += blk_pair[2 * q + 1];
    }
    block_sum_dd<NT>(e_hi, e_lo, red);
    block_sum_dd<NT>(m_hi, m_lo, red);
    block_sum_dd<NT>(p_hi, p_lo, red);
    if (threadIdx.x == 0) {
        const double v12 = bh->vs[0] * bh->vs[0] + bh->vs[1] * bh->vs[1] + bh->vs[2] * bh->vs[2];
        const double smr = m_hi + m_lo;  // sum_i m_i / r_1i
        double hi = 0, lo = 0;
        two_sum_acc(hi, lo, e_hi);
        lo += e_lo;
        two_sum_acc(hi, lo, p_hi);  // unordered pairs i < j
        lo += p_lo;
        two_sum_acc(hi, lo, 0.5 * M * v12);
        two_sum_acc(hi, lo, inv_c2 * 0.5 * G * GM * smr * smr);
        out[0] = hi + lo;
    }
}

// ---------------------------------------------------------------------------------------------------------
// NEXT-3 of the scope table: total 1PN momentum, Eq. 2.8 in the reading R16 of DESIGN.md:
//   P = M v_1 + sum_i m_i v_i (1 + v_i^2/2c^2)
//       - (1/2c^2) { sum_i (GM m_i / r_1i)[v_i + (v_i.n_1i) n_1i + v_1 + (v_1.n_1i) n_1i]
//                  + sum_{i != j} (G m_i m_j / rho_ij)[v_i + (v_i.x_ij) x_ij / rho_ij^2] }.
// The pair sum is symmetrised, sum_{i<j} (G m_i m_j / rho)[u + (u.d) d / rho^2] with u = v_i + v_j, d = x_ij, and walks
// the unordered pairs exactly like energy_pair_kernel (same ERec stream, same grouped compensated summation).
// ---------------------------------------------------------------------------------------------------------
template <int NT>
__global__ void __launch_bounds__(NT) momentum_prep_kernel(const JRec* __restrict__ jrec, const double* __restrict__ v,
                                                           const BhState* __restrict__ bh, double* __restrict__ blk /* [grid][6] */,
                                                           int n_stars, int np, double GM, double G, double inv_c2)
{
    __shared__ double red[2 * (NT / 32)];
    const int i = blockIdx.x * NT + threadIdx.x;
    double t[3] = {0, 0, 0};
    if (i < n_stars) {
        const JRec r = jrec[i];
        const double vv[3] = {v[i], v[np + i], v[2 * np + i]};
        const double v1[3] = {bh->vs[0], bh->vs[1], bh->vs[2]};
        const double d[3] = {bh->xs[0] - r.x, bh->xs[1] - r.y, bh->xs[2] - r.z};  // x_1i
        const double inv_r = 1.0 / sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        const double m = r.gm / G;
        const double v2 = vv[0] * vv[0] + vv[1] * vv[1] + vv[2] * vv[2];
        const double w[3] = {vv[0] + v1[0], vv[1] + v1[1], vv[2] + v1[2]};
        const double wn = (w[0] * d[0] + w[1] * d[1] + w[2] * d[2]) * inv_r * inv_r;  // (w.n) / r
        const double U = GM * m * inv_r;
#pragma unroll
        for (int k = 0; k < 3; ++k) t[k] = m * vv[k] * (1.0 + 0.5 * inv_c2 * v2) - 0.5 * inv_c2 * U * (w[k] + wn * d[k]);
    }
    double* b = blk + 6 * (size_t)blockIdx.x;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        double hi = t[k], lo = 0;
        block_sum_dd<NT>(hi, lo, red);
        if (threadIdx.x == 0) b[2 * k] = hi, b[2 * k + 1] = lo;
    }
}

template <int NT, int TJ>
__global__ void __launch_bounds__(NT) momentum_pair_kernel(const ERec* __restrict__ erec, double* __restrict__ blk /* [grid][6] */,
                                                           int n_stars, int np, long long per_block, double eps2, double G)
{
    static_assert(NT == TJ, "i-tiles and j-tiles share one index space");
    constexpr int kGroup = 8;
    __shared__ ERec sj[TJ];
    __shared__ double red[2 * (NT / 32)];
    const int tid = threadIdx.x;
    const int n_tiles = np / TJ;
    const long long n_pairs = (long long)n_tiles * (n_tiles + 1) / 2;
    const long long p0 = (long long)blockIdx.x * per_block, p1 = min(n_pairs, p0 + per_block);
    double tot_hi[3] = {0, 0, 0}, tot_lo[3] = {0, 0, 0};  // this thread's total over its i-stars, m_i applied
    double hi[3] = {0, 0, 0}, lo[3] = {0, 0, 0};          // the current i-star's pair sums
    int it = 0, jt = 0;
    if (p0 < p1) tri_decode(p0, n_tiles, it, jt);
    int i = it * NT + tid;
    ERec me = erec[i];
    auto close_row = [&]() {
        if (i < n_stars) {  // pad stars (coincident, massless) may hold NaN with eps = 0
            const double mi = me.gm / G;
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                two_sum_acc(tot_hi[k], tot_lo[k], hi[k] * mi);
                tot_lo[k] += lo[k] * mi;
            }
        }
#pragma unroll
        for (int k = 0; k < 3; ++k) hi[k] = lo[k] = 0;
    };
    for (long long p = p0; p < p1; ++p) {
        __syncthreads();
        {
            const double2* src = reinterpret_cast<const double2*>(erec + (size_t)jt * TJ);
            double2* dst = reinterpret_cast<double2*>(sj);
            for (int q = tid; q < TJ * 4; q += NT) dst[q] = src[q];
        }
        __syncthreads();
        const int j0 = jt * TJ;
        auto walk_tile = [&](auto diag) {  // the i < j mask inside the diagonal tile only (see energy_pair_kernel)
#pragma unroll 1
            for (int jb = 0; jb < TJ; jb += kGroup) {
                double g[3] = {0, 0, 0};
#pragma unroll
                for (int u = 0; u < kGroup; ++u) {
                    const int jj = jb + u;
                    const ERec r = sj[jj];
                    const double dx = me.x - r.x, dy = me.y - r.y, dz = me.z - r.z;  // x_ij
                    const double r2 = fma(dx, dx, fma(dy, dy, fma(dz, dz, eps2)));
                    const double y0 = rsqrt_seed(r2);
                    const double e = fma(-r2, y0 * y0, 1.0);
                    double y = fma(y0 * e, fma(e, 0.375, 0.5), y0);  // 1 / rho
                    if (decltype(diag)::value) y = (j0 + jj <= i) ? 0.0 : y;  // i < j only (also keeps the self pair's 1/0 out when eps = 0)
                    const double ux = me.vx + r.vx, uy = me.vy + r.vy, uz = me.vz + r.vz;
                    const double ud = fma(ux, dx, fma(uy, dy, uz * dz)) * (y * y);
                    const double c = r.gm * y;
                    g[0] = fma(c, fma(ud, dx, ux), g[0]);
                    g[1] = fma(c, fma(ud, dy, uy), g[1]);
                    g[2] = fma(c, fma(ud, dz, uz), g[2]);
                }
#pragma unroll
                for (int k = 0; k < 3; ++k) two_sum_acc(hi[k], lo[k], g[k]);
            }
        };
        if (it == jt)
            walk_tile(std::true_type{});
        else
            walk_tile(std::false_type{});
        if (++jt == n_tiles) {
            close_row();
            ++it, jt = it;
            if (p + 1 < p1) {
                i = it * NT + tid;
                me = erec[i];
            }
        }
    }
    close_row();
    double* b = blk + 6 * (size_t)blockIdx.x;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        double h = tot_hi[k], l = tot_lo[k];
        block_sum_dd<NT>(h, l, red);
        if (tid == 0) b[2 * k] = h, b[2 * k + 1] = l;
    }
}

// out[0..2] = P.  One block; fixed order.
template <int NT>
__global__ void __launch_bounds__(NT) momentum_final_kernel(const double* __restrict__ blk_prep, int n_prep,
                                                            const double* __restrict__ blk_pair, int n_pair,
                                                            const BhState* __restrict__ bh, double M, double inv_c2,
                                                            double* __restrict__ out)
{
    __shared__ double red[2 * (NT / 32)];
    for (int k = 0; k < 3; ++k) {
        double a_hi = 0, a_lo = 0, p_hi = 0, p_lo = 0;
        for (int q = threadIdx.x; q < n_prep; q += NT) {
            two_sum_acc(a_hi, a_lo, blk_prep[6 * q + 2 * k]);
            a_lo += blk_prep[6 * q + 2 * k + 1];
        }
        for (int q = threadIdx.x; q < n_pair; q += NT) {
            two_sum_acc(p_hi, p_lo, blk_pair[6 * q + 2 * k]);
            p_lo += blk_pair[6 * q + 2 * k + 1];
        }
        block_sum_dd<NT>(a_hi, a_lo, red);
        block_sum_dd<NT>(p_hi, p_lo, red);
        if (threadIdx.x == 0) {
            double hi = 0, lo = 0;
            two_sum_acc(hi, lo, M * bh->vs[k]);
            two_sum_acc(hi, lo, a_hi);
            lo += a_lo;
            two_sum_acc(hi, lo, -0.5 * inv_c2 * p_hi);
            lo += -0.5 * inv_c2 * p_lo;
            out[k] = hi + lo;
        }
        __syncthreads();
    }
}

}  // namespace pn
