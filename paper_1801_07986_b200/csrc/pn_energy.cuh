// pn_energy.cuh -- S5 (1PN energy, Eq. 2.7) and NEXT-3 (1PN momentum, Eq. 2.8): compensated O(N^2) sums.
// Part of the sm_100a kernels of the limited-1PN hot path (arXiv:1801.07986); pn_kernels.cuh includes every part.
#pragma once
#include "pn_common.cuh"

namespace pn {

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
