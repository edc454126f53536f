// pn_pair_cross.cuh -- NEXT-1/2: S1 + the O(N^2) sums of the Cross terms (Eqs. 2.6, 2.3), ordered and unordered pairs.
// Part of the sm_100a kernels of the limited-1PN hot path (arXiv:1801.07986); pn_kernels.cuh includes every part.
#pragma once
#include "pn_common.cuh"
#include "pn_pair_fp64.cuh"

namespace pn {

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

}  // namespace pn
