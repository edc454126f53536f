// pn_pair_fp32.cuh -- S1 variant: fp32 pair arithmetic (packed f32x2 in the symmetric form), fp64 accumulation.
// Part of the sm_100a kernels of the limited-1PN hot path (arXiv:1801.07986); pn_kernels.cuh includes every part.
#pragma once
#include "pn_common.cuh"
#include "pn_pair_fp64.cuh"

namespace pn {

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

}  // namespace pn
