/*
 * pn_oracle.c -- CPU ORACLE for the limited-1PN N-body hot path of arXiv:1801.07986.
 *
 * THIS FILE IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code,
 * header, table or helper with the CUDA path (paper_1801_07986_b200/csrc) and neither
 * includes the other.
 *
 * It is the paper's definition written out as plain loops, in the paper's order and
 * notation (body 0 == the paper's massive object "#1", mass M; bodies 1..N-1 == the
 * low-mass stars i, j).  No blocking, no fusion, no symmetry tricks.
 *
 *   x_ab = x_a - x_b,  r_ab = |x_ab|,  n_ab = x_ab / r_ab,  v_ab = v_a - v_b
 *   (reading R1: the sign printed at PAPER.md:45 would make Eq. 2.1 repulsive)
 *   rho_ij = sqrt(r_ij^2 + eps^2) for star-star pairs only (Eq. 4.2;
 *   DESIGN.md reading R9).
 *
 * What is computed (hot path; the "Cross" terms, Eqs. 2.3 and 2.6, are the NEXT rows of the scope table and are
 * added only when asked for through the *_terms entry points, see below and DESIGN.md "Scope"):
 *   oracle_accel   a_1 : Eq. 2.1 Newtonian term + (1/c^2)[a_1]_BH, Eq. 2.2
 *                  a_i : Eq. 2.4 first two terms + (1/c^2)[a_i]_BH
 *   oracle_step    classical 4th-order Runge-Kutta on (x, v) of all N bodies
 *   oracle_energy  Eq. 2.7 term by term as printed
 *
 * Arithmetic: every operation is carried out in the type `real`.
 *   default build (liboracle_ref.so):  real = long double (x87 80-bit, 64-bit mantissa),
 *       -O2 -ffp-contract=off: used for parity, more accurate than any fp64 summation order.
 *   -DORACLE_FAST (liboracle_fast.so): real = double, -O3: same source, used only as the
 *       timed CPU baseline.  Both builds run the same pin tests.
 * OpenMP (if enabled) parallelises only over the independent outer index i; each output is
 * produced by one thread in a fixed order, so results do not depend on the thread count.
 *
 * Pins (tests/test_oracle_pins.py): hand-evaluated N=2/N=3 values (tests/golden/), Newtonian
 * limit c=inf against an independent numpy evaluation, Newton's third law, full N-body EIH
 * (Einstein-Infeld-Hoffmann) residual scaling in mpmath, test-particle periastron advance
 * 6 pi G M / (c^2 a (1-e^2)), RK4 4th-order convergence, 1PN two-body energy conservation.
 * NEXT rows (Cross terms, Eqs. 2.3 and 2.6; momentum, Eq. 2.8): residual orders lam^3 / lam^2 / lam^3 against the full
 * EIH acceleration and momentum, hand values for two bodies, bit-identity with the hot path at c = inf and for massless
 * stars, two-body finite-mass periastron advance 6 pi G (M + m) / (c^2 a (1 - e^2)) and energy conservation.
 * Softening inside the 1PN star-star energy bracket, the Cross terms and the momentum (every star-star r_ij -> rho_ij,
 * the r_ij^2 numerators and n_ij -> x_ij / rho_ij included, reading R9) is a convention the paper does not fix (exact at
 * eps = 0).  That the convention is APPLIED at every occurrence is pinned by hand values at eps^2 = 11 (rho_AB = 6):
 * tests/golden/n3_345_softened.txt (energy) and n3_345_softened_cross.txt (Eqs. 2.6, 2.3, 2.8, worked line by line).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifdef ORACLE_FAST
typedef double real;
#define R_SQRT(x) sqrt(x)
#else
typedef long double real;
#define R_SQRT(x) sqrtl(x)
#endif

#define ORACLE_OK 0
#define ORACLE_EINVAL (-1)
#define ORACLE_ENOMEM (-2)

int oracle_real_bytes(void) { return (int)sizeof(real); }
int oracle_mantissa_bits(void)
{
#ifdef ORACLE_FAST
    return 53;
#else
    return 64;
#endif
}
int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

static real dot3(const real* a, const real* b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

/* ---------------------------------------------------------------------------------------
 * Acceleration of the massive object #1 (body 0).  PAPER.md:43-49, Eqs. 2.1 and 2.2:
 *   a_1 = - sum_j G m_j x_1j / r_1j^3
 *         + (1/c^2) { sum_j (G m_j x_1j / r_1j^3) ( 5 G M / r_1j - 2 v_j^2 + (3/2)(v_j . n_1j)^2 )
 *                     + 3 sum_j (G m_j / r_1j^3) (v_j . x_1j) v_j }
 * with x_1j = x_1 - x_j (reading R1) and the square on (v_j . n_1j) (reading R2).
 * BH-star distances are never softened (reading R9).
 * ------------------------------------------------------------------------------------- */
static void accel_bh(int64_t N, const real* m, real G, real inv_c2, const real* x, const real* v, real* a1)
{
    const real M = m[0];
    real newt[3] = {0, 0, 0}, pn_a[3] = {0, 0, 0}, pn_b[3] = {0, 0, 0};
    for (int64_t j = 1; j < N; ++j) {
        real x1j[3], n1j[3];
        for (int k = 0; k < 3; ++k) x1j[k] = x[k] - x[3 * j + k];
        const real r = R_SQRT(dot3(x1j, x1j));
        for (int k = 0; k < 3; ++k) n1j[k] = x1j[k] / r;
        const real r3 = r * r * r;
        const real* vj = v + 3 * j;
        const real vj2 = dot3(vj, vj);
        const real vn = dot3(vj, n1j);
        const real bracket = 5 * G * M / r - 2 * vj2 + (real)1.5 * vn * vn;
        const real vx = dot3(vj, x1j);
        for (int k = 0; k < 3; ++k) {
            newt[k] += G * m[j] * x1j[k] / r3;            /* Eq. 2.1, first term (sign below)  */
            pn_a[k] += G * m[j] * x1j[k] / r3 * bracket;  /* Eq. 2.2, first sum                */
            pn_b[k] += G * m[j] / r3 * vx * vj[k];        /* Eq. 2.2, second sum (factor below)*/
        }
    }
    for (int k = 0; k < 3; ++k) a1[k] = -newt[k] + inv_c2 * (pn_a[k] + 3 * pn_b[k]);
}

/* ---------------------------------------------------------------------------------------
 * Acceleration of star i.  PAPER.md:63-68, Eq. 2.4 and the unnumbered [a_i]_BH:
 *   a_i = - G M x_i1 / r_i1^3 - sum_{j != i} G m_j x_ij / rho_ij^3
 *         + (1/c^2) { (G M x_i1 / r_i1^3)(4 G M / r_i1 - v_i^2) + 4 (G M / r_i1^3)(v_i . x_i1) v_i }
 * (exponent 3 on r_ij: reading R4; v_a -> v_i: reading R3; star-star 1/r softened, Eq. 4.2).
 * ------------------------------------------------------------------------------------- */
static void accel_star(int64_t N, const real* m, real G, real inv_c2, real eps2, const real* x, const real* v,
                       int64_t i, real* ai)
{
    const real M = m[0];
    real xi1[3];
    for (int k = 0; k < 3; ++k) xi1[k] = x[3 * i + k] - x[k];
    const real r = R_SQRT(dot3(xi1, xi1));
    const real r3 = r * r * r;
    const real* vi = v + 3 * i;
    const real vi2 = dot3(vi, vi);
    const real vx = dot3(vi, xi1);

    real ss[3] = {0, 0, 0};
    for (int64_t j = 1; j < N; ++j) {
        if (j == i) continue;
        real xij[3];
        for (int k = 0; k < 3; ++k) xij[k] = x[3 * i + k] - x[3 * j + k];
        const real rho = R_SQRT(dot3(xij, xij) + eps2);
        const real rho3 = rho * rho * rho;
        for (int k = 0; k < 3; ++k) ss[k] += G * m[j] * xij[k] / rho3;
    }
    for (int k = 0; k < 3; ++k) {
        const real newt_bh = -G * M * xi1[k] / r3;
        const real pn = G * M * xi1[k] / r3 * (4 * G * M / r - vi2) + 4 * G * M / r3 * vx * vi[k];
        ai[k] = newt_bh - ss[k] + inv_c2 * pn;
    }
}

/* ---------------------------------------------------------------------------------------
 * NEXT rows of the scope table, selected by the `terms` bit mask; terms = 0 is the hot path.
 *
 * ORACLE_CROSS_STAR: [a_i]_Cross, Eq. 2.6, line by line as printed (x_ab = x_a - x_b,
 * v_ij = v_i - v_j: reading R1; "sum_i" of the last line -> sum_j: reading A6; j != i in every sum):
 *   L0  5 G^2 m_i M x_i1 / r_i1^4 - (G m_i / r_i1^3) [ 4 v_i^2 x_i1 - 7 (v_i.x_i1) v_i ]
 *   L1  sum_j G^2 m_j M x_i1 / r_i1^3 ( 4/r_ij + 5/(4 r_j1) + r_i1^2/(4 r_j1^3) - r_ij^2/(4 r_j1^3) )
 *   L2  sum_j G^2 m_j M x_ij / r_ij^3 ( 4/r_i1 + 5/(4 r_j1) - r_i1^2/(4 r_j1^3) + r_ij^2/(4 r_j1^3) )
 *   L3  -(7/2) sum_j G^2 m_j M x_j1 / r_j1^3 ( 1/r_ij - 1/r_i1 )
 *   L4  - sum_j (G m_j / r_i1^3) [ 4 (v_i.v_j) x_i1 - 3 (v_j.x_i1) v_i - 4 (v_i.x_i1) v_j ]
 *   L5  + sum_j (G m_j x_ij / r_ij^3) [ v_i^2 - 2 |v_ij|^2 + (3/2)(v_j.n_ij)^2 ]
 *   L6  + sum_j (G m_j / r_ij^3) [ x_ij.(4 v_i - 3 v_j) ] v_ij
 * Softening (reading R9, a convention, exact at eps = 0): every star-star r_ij above is rho_ij, including the
 * r_ij^2 in the numerators and n_ij = x_ij / rho_ij; distances to the massive object are never softened.
 * ------------------------------------------------------------------------------------- */
#define ORACLE_CROSS_STAR 1
#define ORACLE_CROSS_BH 2

static void cross_star(int64_t N, const real* m, real G, real eps2, const real* x, const real* v, int64_t i, real* out)
{
    const real M = m[0];
    real xi1[3];
    for (int k = 0; k < 3; ++k) xi1[k] = x[3 * i + k] - x[k];
    const real ri1 = R_SQRT(dot3(xi1, xi1));
    const real ri1_3 = ri1 * ri1 * ri1;
    const real* vi = v + 3 * i;
    const real vi2 = dot3(vi, vi);
    const real vixi1 = dot3(vi, xi1);
    real acc[3];
    for (int k = 0; k < 3; ++k) /* L0 */
        acc[k] = 5 * G * G * m[i] * M * xi1[k] / (ri1_3 * ri1) - G * m[i] / ri1_3 * (4 * vi2 * xi1[k] - 7 * vixi1 * vi[k]);
    for (int64_t j = 1; j < N; ++j) {
        if (j == i) continue;
        real xij[3], xj1[3], vij[3], w[3];
        for (int k = 0; k < 3; ++k) {
            xij[k] = x[3 * i + k] - x[3 * j + k];
            xj1[k] = x[3 * j + k] - x[k];
            vij[k] = vi[k] - v[3 * j + k];
            w[k] = 4 * vi[k] - 3 * v[3 * j + k];
        }
        const real* vj = v + 3 * j;
        const real rij2 = dot3(xij, xij) + eps2; /* rho_ij^2 */
        const real rij = R_SQRT(rij2);
        const real rij3 = rij2 * rij;
        const real rj1 = R_SQRT(dot3(xj1, xj1));
        const real rj1_3 = rj1 * rj1 * rj1;
        const real f1 = 4 / rij + 5 / (4 * rj1) + ri1 * ri1 / (4 * rj1_3) - rij2 / (4 * rj1_3);
        const real f2 = 4 / ri1 + 5 / (4 * rj1) - ri1 * ri1 / (4 * rj1_3) + rij2 / (4 * rj1_3);
        const real vn = dot3(vj, xij) / rij;
        const real b5 = vi2 - 2 * dot3(vij, vij) + (real)1.5 * vn * vn;
        const real xw = dot3(xij, w);
        for (int k = 0; k < 3; ++k) {
            acc[k] += G * G * m[j] * M * xi1[k] / ri1_3 * f1;                                              /* L1 */
            acc[k] += G * G * m[j] * M * xij[k] / rij3 * f2;                                               /* L2 */
            acc[k] -= (real)3.5 * G * G * m[j] * M * xj1[k] / rj1_3 * (1 / rij - 1 / ri1);                 /* L3 */
            acc[k] -= G * m[j] / ri1_3 * (4 * dot3(vi, vj) * xi1[k] - 3 * dot3(vj, xi1) * vi[k] - 4 * vixi1 * vj[k]); /* L4 */
            acc[k] += G * m[j] * xij[k] / rij3 * b5;                                                       /* L5 */
            acc[k] += G * m[j] / rij3 * xw * vij[k];                                                       /* L6 */
        }
    }
    for (int k = 0; k < 3; ++k) out[k] = acc[k];
}

/* ---------------------------------------------------------------------------------------
 * ORACLE_CROSS_BH: [a_1]_Cross, Eq. 2.3 (x_1j = x_1 - x_j, x_jk = x_j - x_k; k != j in the sums
 * that contain r_jk, k = j INCLUDED in the velocity sum: reading A6; star-star r_jk softened as above):
 *   4 sum_j G^2 m_j^2 x_1j / r_1j^4
 *   + sum_{j,k} G^2 m_j m_k x_1j / r_1j^3 ( 4/r_1k + 5/(4 r_jk) - r_1k^2/(4 r_jk^3) + r_1j^2/(4 r_jk^3) )
 *   - (7/2) sum_{j,k} G^2 m_j m_k x_jk / (r_jk^3 r_1j)
 *   - sum_{j,k} (G m_j m_k / (M r_1j^3)) [ 4 (v_j.v_k) x_1j - 3 (v_j.x_1j) v_k - 4 (v_k.x_1j) v_j ]
 * ------------------------------------------------------------------------------------- */
static void cross_bh(int64_t N, const real* m, real G, real eps2, const real* x, const real* v, real* out)
{
    const real M = m[0];
    real acc[3] = {0, 0, 0};
    for (int64_t j = 1; j < N; ++j) {
        real x1j[3];
        for (int q = 0; q < 3; ++q) x1j[q] = x[q] - x[3 * j + q];
        const real r1j = R_SQRT(dot3(x1j, x1j));
        const real r1j3 = r1j * r1j * r1j;
        const real* vj = v + 3 * j;
        for (int q = 0; q < 3; ++q) acc[q] += 4 * G * G * m[j] * m[j] * x1j[q] / (r1j3 * r1j);
        for (int64_t k = 1; k < N; ++k) {
            const real* vk = v + 3 * k;
            for (int q = 0; q < 3; ++q)
                acc[q] -= G * m[j] * m[k] / (M * r1j3) *
                          (4 * dot3(vj, vk) * x1j[q] - 3 * dot3(vj, x1j) * vk[q] - 4 * dot3(vk, x1j) * vj[q]);
            if (k == j) continue;
            real x1k[3], xjk[3];
            for (int q = 0; q < 3; ++q) x1k[q] = x[q] - x[3 * k + q], xjk[q] = x[3 * j + q] - x[3 * k + q];
            const real r1k = R_SQRT(dot3(x1k, x1k));
            const real rjk2 = dot3(xjk, xjk) + eps2;
            const real rjk = R_SQRT(rjk2);
            const real rjk3 = rjk2 * rjk;
            const real f = 4 / r1k + 5 / (4 * rjk) - r1k * r1k / (4 * rjk3) + r1j * r1j / (4 * rjk3);
            for (int q = 0; q < 3; ++q) {
                acc[q] += G * G * m[j] * m[k] * x1j[q] / r1j3 * f;
                acc[q] -= (real)3.5 * G * G * m[j] * m[k] * xjk[q] / (rjk3 * r1j);
            }
        }
    }
    for (int q = 0; q < 3; ++q) out[q] = acc[q];
}

/* acc[a] for every body a in rows[0..nrows) (rows == NULL: all bodies, nrows == N). */
static void accel_real(int64_t N, const real* m, real G, real inv_c2, real eps2, const real* x, const real* v,
                       int64_t nrows, const int64_t* rows, int terms, real* acc)
{
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 16)
#endif
    for (int64_t q = 0; q < nrows; ++q) {
        const int64_t a = rows ? rows[q] : q;
        real cr[3] = {0, 0, 0};
        if (a == 0) {
            accel_bh(N, m, G, inv_c2, x, v, acc + 3 * q);
            if (terms & ORACLE_CROSS_BH) cross_bh(N, m, G, eps2, x, v, cr);
        } else {
            accel_star(N, m, G, inv_c2, eps2, x, v, a, acc + 3 * q);
            if (terms & ORACLE_CROSS_STAR) cross_star(N, m, G, eps2, x, v, a, cr);
        }
        for (int k = 0; k < 3; ++k) acc[3 * q + k] += inv_c2 * cr[k];
    }
}

static int check_args(int64_t N, const double* mass, double G, double c, double eps)
{
    if (N < 2 || !mass) return ORACLE_EINVAL;
    if (!(G > 0) || !(c > 0) || !(eps >= 0) || isinf(G) || isinf(eps)) return ORACLE_EINVAL;
    if (!(mass[0] > 0) || isinf(mass[0])) return ORACLE_EINVAL;
    for (int64_t i = 1; i < N; ++i)
        if (!(mass[i] >= 0) || isinf(mass[i])) return ORACLE_EINVAL;
    return ORACLE_OK;
}

static real* to_real(const double* src, int64_t n)
{
    real* dst = (real*)malloc(sizeof(real) * (size_t)n);
    if (dst)
        for (int64_t i = 0; i < n; ++i) dst[i] = (real)src[i];
    return dst;
}

/* pos, vel, acc: host, row-major [N][3] doubles; mass: N doubles, mass[0] = M.  c may be +inf. */
int oracle_accel_rows_terms(int64_t N, const double* mass, double G, double c, double eps, const double* pos,
                            const double* vel, int64_t nrows, const int64_t* rows, int terms, double* acc_rows)
{
    int rc = check_args(N, mass, G, c, eps);
    if (rc) return rc;
    if (terms & ~(ORACLE_CROSS_STAR | ORACLE_CROSS_BH)) return ORACLE_EINVAL;
    if (!pos || !vel || !acc_rows || nrows < 0) return ORACLE_EINVAL;
    if (rows)
        for (int64_t q = 0; q < nrows; ++q)
            if (rows[q] < 0 || rows[q] >= N) return ORACLE_EINVAL;
    real *m = to_real(mass, N), *x = to_real(pos, 3 * N), *v = to_real(vel, 3 * N);
    real* a = (real*)malloc(sizeof(real) * 3 * (size_t)(nrows ? nrows : 1));
    if (!m || !x || !v || !a) {
        free(m), free(x), free(v), free(a);
        return ORACLE_ENOMEM;
    }
    const real inv_c2 = 1 / ((real)c * (real)c);
    accel_real(N, m, (real)G, inv_c2, (real)eps * (real)eps, x, v, nrows, rows, terms, a);
    for (int64_t q = 0; q < 3 * nrows; ++q) acc_rows[q] = (double)a[q];
    free(m), free(x), free(v), free(a);
    return ORACLE_OK;
}

int oracle_accel_rows(int64_t N, const double* mass, double G, double c, double eps, const double* pos,
                      const double* vel, int64_t nrows, const int64_t* rows, double* acc_rows)
{
    return oracle_accel_rows_terms(N, mass, G, c, eps, pos, vel, nrows, rows, 0, acc_rows);
}

int oracle_accel(int64_t N, const double* mass, double G, double c, double eps, const double* pos,
                 const double* vel, double* acc)
{
    return oracle_accel_rows(N, mass, G, c, eps, pos, vel, N, NULL, acc);
}

/* ---------------------------------------------------------------------------------------
 * Classical fourth-order Runge-Kutta, PAPER.md:130, 150 (ref. [22]); reading R13.
 * y = (x, v) of ALL N bodies (the massive object moves too), f(y) = (v, a(x, v)):
 *   k1 = f(y_n); k2 = f(y_n + dt/2 k1); k3 = f(y_n + dt/2 k2); k4 = f(y_n + dt k3)
 *   y_{n+1} = y_n + dt/6 (k1 + 2 k2 + 2 k3 + k4)
 * The acceleration depends on v (1PN), so the velocity stages are formed explicitly.
 * pos, vel are updated in place, nsteps times.
 * ------------------------------------------------------------------------------------- */
int oracle_step_terms(int64_t N, const double* mass, double G, double c, double eps, double* pos, double* vel,
                      double dt, int64_t nsteps, int terms)
{
    int rc = check_args(N, mass, G, c, eps);
    if (rc) return rc;
    if (terms & ~(ORACLE_CROSS_STAR | ORACLE_CROSS_BH)) return ORACLE_EINVAL;
    if (!pos || !vel || nsteps < 0 || !isfinite(dt)) return ORACLE_EINVAL;
    const int64_t n3 = 3 * N;
    real *m = to_real(mass, N), *x = to_real(pos, n3), *v = to_real(vel, n3);
    real* w = (real*)malloc(sizeof(real) * (size_t)n3 * 10);
    if (!m || !x || !v || !w) {
        free(m), free(x), free(v), free(w);
        return ORACLE_ENOMEM;
    }
    real *xs = w, *vs = w + n3;              /* stage state                 */
    real* kx[4] = {w + 2 * n3, w + 3 * n3, w + 4 * n3, w + 5 * n3};
    real* kv[4] = {w + 6 * n3, w + 7 * n3, w + 8 * n3, w + 9 * n3};
    const real inv_c2 = 1 / ((real)c * (real)c), eps2 = (real)eps * (real)eps, h = (real)dt, g = (real)G;
    const real cstage[4] = {0, (real)0.5, (real)0.5, 1};
    for (int64_t s = 0; s < nsteps; ++s) {
        for (int st = 0; st < 4; ++st) {
            for (int64_t q = 0; q < n3; ++q) {
                xs[q] = st ? x[q] + cstage[st] * h * kx[st - 1][q] : x[q];
                vs[q] = st ? v[q] + cstage[st] * h * kv[st - 1][q] : v[q];
            }
            for (int64_t q = 0; q < n3; ++q) kx[st][q] = vs[q];
            accel_real(N, m, g, inv_c2, eps2, xs, vs, N, NULL, terms, kv[st]);
        }
        for (int64_t q = 0; q < n3; ++q) {
            x[q] += h / 6 * (kx[0][q] + 2 * kx[1][q] + 2 * kx[2][q] + kx[3][q]);
            v[q] += h / 6 * (kv[0][q] + 2 * kv[1][q] + 2 * kv[2][q] + kv[3][q]);
        }
    }
    for (int64_t q = 0; q < n3; ++q) pos[q] = (double)x[q], vel[q] = (double)v[q];
    free(m), free(x), free(v), free(w);
    return ORACLE_OK;
}

int oracle_step(int64_t N, const double* mass, double G, double c, double eps, double* pos, double* vel,
                double dt, int64_t nsteps)
{
    return oracle_step_terms(N, mass, G, c, eps, pos, vel, dt, nsteps, 0);
}

/* ---------------------------------------------------------------------------------------
 * Total 1PN energy, Eq. 2.7, term by term in the printed order:
 *   T1 = 1/2 M v_1^2                         T2 = 1/2 sum_i m_i v_i^2
 *   T3 = -1/2 sum_{i != j} G m_i m_j / rho_ij T4 = - sum_i G M m_i / r_1i
 *   (1/c^2) x {
 *   P1 = 3/8 sum_i m_i v_i^4                 P2 = 3/2 sum_i (G M m_i / r_1i) v_i^2
 *   P3 = 1/2 sum_i G^2 M^2 m_i / r_1i^2
 *   P4 = 1/4 sum_{i != j} (G m_i m_j / rho_ij)[6 v_i^2 - 7 v_i.v_j - (n_ij.v_i)(n_ij.v_j)]
 *   P5 = 1/2 sum_i (G M m_i / r_1i)[3 v_1^2 - 7 v_1.v_i - (n_1i.v_1)(n_1i.v_i)]
 *   P6 = sum_{i != j} G^2 M m_i m_j / (rho_ij r_1i)
 *   P7 = 1/2 sum_{i, j} G^2 M m_i m_j / (r_1i r_1j)      (i = j included: reading R5) }
 * Star-star inverse distances use rho_ij and n_ij = x_ij / rho_ij (reading R9).
 * terms_out (optional): 11 doubles T1..T4, P1..P7 (P's WITHOUT the 1/c^2 factor).
 * ------------------------------------------------------------------------------------- */
int oracle_energy(int64_t N, const double* mass, double G_, double c, double eps, const double* pos,
                  const double* vel, double* E_out, double* terms_out)
{
    int rc = check_args(N, mass, G_, c, eps);
    if (rc) return rc;
    if (!pos || !vel || !E_out) return ORACLE_EINVAL;
    real *m = to_real(mass, N), *x = to_real(pos, 3 * N), *v = to_real(vel, 3 * N);
    real* row = (real*)calloc((size_t)N * 4, sizeof(real)); /* per-i partial sums of T3, P4, P6, P7 */
    if (!m || !x || !v || !row) {
        free(m), free(x), free(v), free(row);
        return ORACLE_ENOMEM;
    }
    const real G = (real)G_, M = m[0], inv_c2 = 1 / ((real)c * (real)c), eps2 = (real)eps * (real)eps;
    const real* v1 = v;
    real T1 = (real)0.5 * M * dot3(v1, v1), T2 = 0, T3 = 0, T4 = 0;
    real P1 = 0, P2 = 0, P3 = 0, P4 = 0, P5 = 0, P6 = 0, P7 = 0;

    for (int64_t i = 1; i < N; ++i) {
        real x1i[3], n1i[3];
        for (int k = 0; k < 3; ++k) x1i[k] = x[k] - x[3 * i + k];
        const real r1i = R_SQRT(dot3(x1i, x1i));
        for (int k = 0; k < 3; ++k) n1i[k] = x1i[k] / r1i;
        const real* vi = v + 3 * i;
        const real vi2 = dot3(vi, vi);
        T2 += (real)0.5 * m[i] * vi2;
        T4 -= G * M * m[i] / r1i;
        P1 += (real)0.375 * m[i] * vi2 * vi2;
        P2 += (real)1.5 * (G * M * m[i] / r1i) * vi2;
        P3 += (real)0.5 * G * G * M * M * m[i] / (r1i * r1i);
        P5 += (real)0.5 * (G * M * m[i] / r1i) *
              (3 * dot3(v1, v1) - 7 * dot3(v1, vi) - dot3(n1i, v1) * dot3(n1i, vi));
    }
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 16)
#endif
    for (int64_t i = 1; i < N; ++i) {
        real x1i[3];
        for (int k = 0; k < 3; ++k) x1i[k] = x[k] - x[3 * i + k];
        const real r1i = R_SQRT(dot3(x1i, x1i));
        const real* vi = v + 3 * i;
        const real vi2 = dot3(vi, vi);
        real t3 = 0, p4 = 0, p6 = 0, p7 = 0;
        for (int64_t j = 1; j < N; ++j) {
            real x1j[3];
            for (int k = 0; k < 3; ++k) x1j[k] = x[k] - x[3 * j + k];
            const real r1j = R_SQRT(dot3(x1j, x1j));
            p7 += (real)0.5 * G * G * M * m[i] * m[j] / (r1i * r1j);
            if (j == i) continue;
            real xij[3], nij[3];
            for (int k = 0; k < 3; ++k) xij[k] = x[3 * i + k] - x[3 * j + k];
            const real rho = R_SQRT(dot3(xij, xij) + eps2);
            for (int k = 0; k < 3; ++k) nij[k] = xij[k] / rho;
            const real* vj = v + 3 * j;
            t3 -= (real)0.5 * G * m[i] * m[j] / rho;
            p4 += (real)0.25 * (G * m[i] * m[j] / rho) *
                  (6 * vi2 - 7 * dot3(vi, vj) - dot3(nij, vi) * dot3(nij, vj));
            p6 += G * G * M * m[i] * m[j] / (rho * r1i);
        }
        row[4 * i + 0] = t3, row[4 * i + 1] = p4, row[4 * i + 2] = p6, row[4 * i + 3] = p7;
    }
    for (int64_t i = 1; i < N; ++i) T3 += row[4 * i], P4 += row[4 * i + 1], P6 += row[4 * i + 2], P7 += row[4 * i + 3];

    const real E = T1 + T2 + T3 + T4 + inv_c2 * (P1 + P2 + P3 + P4 + P5 + P6 + P7);
    *E_out = (double)E;
    if (terms_out) {
        const real t[11] = {T1, T2, T3, T4, P1, P2, P3, P4, P5, P6, P7};
        for (int k = 0; k < 11; ++k) terms_out[k] = (double)t[k];
    }
    free(m), free(x), free(v), free(row);
    return ORACLE_OK;
}

/* ---------------------------------------------------------------------------------------
 * NEXT-3 of the scope table: total 1PN momentum, Eq. 2.8.  The extraction garbles the indices of the
 * second sum in the braces ("sum_i (G m_i m_j / r_1j)[v_i + (v_i.n_ij) n_ij]").  Reading R16: the 1PN
 * momentum of the parent (EIH) theory, sum_a m_a v_a (1 + v_a^2 / 2c^2) - (1/2c^2) sum_{a != b} (G m_a m_b / r_ab)
 * [v_a + (v_a.n_ab) n_ab], with every term kept that is needed for the error order the paper states,
 * O(G m_i^3 v_i / (c^2 M r)):
 *   P = M v_1 + sum_i m_i v_i (1 + v_i^2 / 2c^2)
 *       - (1/2c^2) { sum_i (G M m_i / r_1i) [ v_i + (v_i.n_1i) n_1i ]            (a = star i, b = #1; printed)
 *                  + sum_i (G M m_i / r_1i) [ v_1 + (v_1.n_1i) n_1i ]            (a = #1, b = star i; O(m^2) as v_1 = O(m))
 *                  + sum_{i != j} (G m_i m_j / rho_ij) [ v_i + (v_i.n_ij) n_ij ] }   (stars; softened, n_ij = x_ij / rho_ij)
 * Dropped: (1/2c^2) M v_1^2 v_1 = O(m^3).  Pinned by the O(lam^3) residual against the EIH momentum.
 * ------------------------------------------------------------------------------------- */
int oracle_momentum(int64_t N, const double* mass, double G_, double c, double eps, const double* pos,
                    const double* vel, double* P_out)
{
    int rc = check_args(N, mass, G_, c, eps);
    if (rc) return rc;
    if (!pos || !vel || !P_out) return ORACLE_EINVAL;
    real *m = to_real(mass, N), *x = to_real(pos, 3 * N), *v = to_real(vel, 3 * N);
    real* row = (real*)calloc((size_t)N * 3, sizeof(real));
    if (!m || !x || !v || !row) {
        free(m), free(x), free(v), free(row);
        return ORACLE_ENOMEM;
    }
    const real G = (real)G_, M = m[0], inv_c2 = 1 / ((real)c * (real)c), eps2 = (real)eps * (real)eps;
    const real* v1 = v;
    real P[3], B[3] = {0, 0, 0}, S[3] = {0, 0, 0};
    for (int k = 0; k < 3; ++k) P[k] = M * v1[k];
    for (int64_t i = 1; i < N; ++i) {
        real x1i[3], n1i[3];
        for (int k = 0; k < 3; ++k) x1i[k] = x[k] - x[3 * i + k];
        const real r1i = R_SQRT(dot3(x1i, x1i));
        for (int k = 0; k < 3; ++k) n1i[k] = x1i[k] / r1i;
        const real* vi = v + 3 * i;
        const real vi2 = dot3(vi, vi);
        for (int k = 0; k < 3; ++k) {
            P[k] += m[i] * vi[k] * (1 + (real)0.5 * inv_c2 * vi2);
            B[k] += G * M * m[i] / r1i * (vi[k] + dot3(vi, n1i) * n1i[k]);
            B[k] += G * M * m[i] / r1i * (v1[k] + dot3(v1, n1i) * n1i[k]);
        }
    }
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 16)
#endif
    for (int64_t i = 1; i < N; ++i) {
        const real* vi = v + 3 * i;
        real acc[3] = {0, 0, 0};
        for (int64_t j = 1; j < N; ++j) {
            if (j == i) continue;
            real xij[3], nij[3];
            for (int k = 0; k < 3; ++k) xij[k] = x[3 * i + k] - x[3 * j + k];
            const real rho = R_SQRT(dot3(xij, xij) + eps2);
            for (int k = 0; k < 3; ++k) nij[k] = xij[k] / rho;
            for (int k = 0; k < 3; ++k) acc[k] += G * m[i] * m[j] / rho * (vi[k] + dot3(vi, nij) * nij[k]);
        }
        for (int k = 0; k < 3; ++k) row[3 * i + k] = acc[k];
    }
    for (int64_t i = 1; i < N; ++i)
        for (int k = 0; k < 3; ++k) S[k] += row[3 * i + k];
    for (int k = 0; k < 3; ++k) P_out[k] = (double)(P[k] - (real)0.5 * inv_c2 * (B[k] + S[k]));
    free(m), free(x), free(v), free(row);
    return ORACLE_OK;
}
