/*
 * pn.h -- C-ABI of libpn.so: the limited first-order post-Newtonian (1PN) N-body hot path of
 * arXiv:1801.07986 (Tatekawa) on one NVIDIA B200 (sm_100a).
 *
 * Citations are /root/reference/PAPER.md:<line> (+ equation).  Notation: body 0 is the paper's
 * massive object "#1" (mass M); bodies 1..N-1 are the low-mass stars i, j.
 * x_ab = x_a - x_b, r_ab = |x_ab|, n_ab = x_ab / r_ab (reading R1);
 * rho_ij = sqrt(r_ij^2 + eps^2) between stars only (Eq. 4.2).
 *
 * What one force evaluation computes (the "hot path"; the Cross terms, Eqs. 2.3 and 2.6, are
 * outside it -- DESIGN.md "Scope"):
 *   a_1 = sum_j (G m_j / r_1j^3) { -x_1j + (1/c^2)[ (5 G M / r_1j - 2 v_j^2 + (3/2)(v_j.n_1j)^2) x_1j
 *                                                   + 3 (v_j.x_1j) v_j ] }      PAPER.md:43-49, Eqs. 2.1, 2.2
 *   a_i = - G M x_i1 / r_i1^3 - sum_{j != i} G m_j x_ij / rho_ij^3
 *         + (1/c^2)(G M / r_i1^3)[ (4 G M / r_i1 - v_i^2) x_i1 + 4 (v_i.x_i1) v_i ]   PAPER.md:63-68, Eq. 2.4
 *
 * General rules
 *   - Every function returns PN_OK (0) or a negative PN_E* code; pn_last_error() gives the text.
 *   - "dev" pointers are CUDA device pointers on the context's device; "host" pointers are
 *     ordinary host memory.  All arrays are fp64, row-major [N][3] unless stated.
 *   - The caller owns every buffer it passes; the library copies what it needs during the call
 *     (stream-ordered) and never retains or frees caller pointers.
 *   - All work is enqueued on the context's stream (pn_set_stream; default: the legacy default
 *     stream).  Calls with only device arguments are asynchronous; calls that take or return host
 *     data synchronise that stream before returning.
 *   - A context is single-stream and single-threaded: pn_accel, pn_step, pn_energy and pn_momentum share
 *     the context's scratch buffers (partial sums, the block partials of a_1 and their ticket counter),
 *     so calls on one context must not run concurrently -- one stream at a time, one host thread at a
 *     time.  pn_set_stream orders the new stream after everything already enqueued on the old one.
 *     Use one context per stream for concurrent work.
   - Small-system path (PN_PAIR_AUTO, fewer than 3072 stars): its one-launch kernels synchronise their blocks with a grid
     barrier whose wait is bounded; a launch that gives up (about half a minute; it cannot happen while every block is
     resident) leaves invalid results.  Calls that synchronise report it at once (PN_ECUDA); callers that only use the
     asynchronous calls learn of it from the NEXT pn_set_state / pn_get_state / pn_accel / pn_step on the context, which
     look at a word in mapped host memory that the kernel sets (no copy, no synchronisation in the normal case).
 *   - A context belongs to the CUDA device that was current in pn_create; every later call must be made
 *     with that device current (PN_EINVAL otherwise; pn_destroy switches to it by itself).
 *   - Size limit: 2 <= N <= 2^24 bodies (PN_EINVAL beyond; star indices and tile counts are 32-bit, the
 *     partial-sum buffer grows as 3 KB per star: 12.9 GB at N = 2^22, 51.5 GB at N = 2^24).
 *   - There is no CPU fallback: without a CUDA device pn_create fails with PN_ECUDA.
 *   - Coincident bodies (BH-star distance 0, or two stars at distance 0 with eps = 0) give
 *     inf/NaN, propagated, not trapped.  With eps = 0 the self term j = i is skipped by index.
 */
#ifndef PN_H_
#define PN_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PN_OK 0
#define PN_EINVAL (-1) /* bad argument: N < 2 or N > 2^24, wrong current device, null pointer, non-finite/negative mass, M <= 0, G <= 0, c <= 0 or NaN,
                          eps < 0 or NaN, non-finite dt, nsteps < 0, unknown option/value */
#define PN_ECUDA (-2)  /* a CUDA call failed (text in pn_last_error) or no device */
#define PN_ESTATE (-3) /* pn_step / pn_energy / pn_get_state before any pn_set_state */
#define PN_ENOMEM (-4) /* host or device allocation failed */

/* pn_set_option keys */
#define PN_OPT_PAIR_PRECISION 1 /* PN_FP64 (default) | PN_FP32_PAIR: arithmetic of the O(N^2) star-star pair loop */
#define PN_OPT_USE_GRAPH 2      /* 1 (default): pn_step replays a captured CUDA graph; 0: plain launches (neither applies to
                                   the small-system path, see PN_PAIR_AUTO: that is one cooperative launch per call) */
#define PN_OPT_TIME_PAIR 3      /* 1: bracket the pair stage of every force evaluation with CUDA events (pn_step: event-record
                                   nodes inside a one-step CUDA graph; plain launches when PN_OPT_USE_GRAPH is 0); read with
                                   pn_get_pair_time.  2: as 1, but in pn_step only the first of the four force evaluations
                                   of a step is bracketed (a quarter of the instrumentation).  0 (default) */
#define PN_OPT_J_SPLIT 4        /* 0 (default): automatic; > 0: force the number of j-chunks per i-tile (tiled kernel) */
#define PN_OPT_PAIR_KERNEL 5    /* which fp64 star-star kernel: PN_PAIR_AUTO (default) | PN_PAIR_TILED | PN_PAIR_SYMMETRIC */

#define PN_OPT_EQUAL_MASS 6     /* 1 (default): when every star has the same mass (checked in pn_create) the symmetric
                                   kernels accumulate rho^-3 d on both sides and apply the common G m once per partial sum
                                   (9 instead of 10 FP64, 10 instead of 11 FP32 instructions per ordered pair); 0: always
                                   the general-mass form */

#define PN_OPT_CROSS_TERMS 7    /* 0 (default): the hot path of north_star; PN_CROSS_STAR: add [a_i]_Cross, Eq. 2.6
                                   (PAPER.md:70-86), to every star's acceleration -- the first NEXT row of the scope table:
                                   its O(N^2) sums are fused into an fp64 pair kernel that also produces the Newtonian
                                   star-star term, its O(N) parts go into the epilogue.  From 6144 stars on that kernel
                                   evaluates every UNORDERED pair once for both stars (38 FP64 instructions per ordered
                                   pair, 37 with equal masses), below every ordered pair (54); PN_OPT_PAIR_KERNEL = PN_PAIR_SYMMETRIC /
                                   PN_PAIR_TILED forces either.  PN_CROSS_STAR | PN_CROSS_BH: also [a_1]_Cross, Eq. 2.3
                                   (PAPER.md:51-57), the second NEXT row -- the paper's full limited-1PN force (one more
                                   O(N^2) sum per star in the same kernel, 42 / 59 instructions per pair; the rest is O(N)).
                                   Applies to pn_accel and pn_step; pn_energy is Eq. 2.7 either way.  The Cross path is fp64
                                   only: while it is on, PN_OPT_PAIR_PRECISION has no effect. */
#define PN_CROSS_STAR 1
#define PN_CROSS_BH 2

/* PN_OPT_PAIR_PRECISION values */
#define PN_FP64 0      /* fp64 pair arithmetic and accumulation (parity 1e-12) */
#define PN_FP32_PAIR 1 /* fp32 pair arithmetic on two-float positions, fp64 accumulation (parity 1e-5) */

/* PN_OPT_PAIR_KERNEL values (either pair precision) */
#define PN_PAIR_AUTO 0      /* symmetric for N - 1 >= 3072 stars (unit tiles of 128 stars, 512 from 36000 stars on).  Below
                               (fp64; with the Cross terms: up to 1279 stars): the small-system path -- ONE cooperative kernel launch runs a whole
                               pn_step call (every stage of every step) or one pn_accel, every ordered pair, 15 instructions;
                               it needs a device with cooperative launch and as many SMs as blocks (else: tiled) */
#define PN_PAIR_TILED 1     /* every ordered pair (i, j): 15 FP64 (18 FP32) instructions per ordered pair */
#define PN_PAIR_SYMMETRIC 2 /* every unordered pair once, applied to both stars (Newton's third law, exact for the
                               softened Newtonian term of Eq. 2.4): 10 FP64 (11 FP32) instructions per ordered pair */

typedef struct pn_ctx pn_ctx; /* opaque; owns all internal device buffers */

/* Problem statement of the paper: one massive object + N-1 stars, constants G, c and
 * the star-star Plummer softening eps.  2 <= N <= 2^24.  masses_host: N host doubles, copied; masses_host[0] = M > 0,
 * stars >= 0.  c may be +inf (pure Newtonian).  Uses the current CUDA device, and stays on it.  *out is set to NULL on
 * failure (pn_last_error(NULL) has the text). */
int pn_create(pn_ctx** out, int64_t N, const double* masses_host, double G, double c, double softening);
int pn_destroy(pn_ctx* ctx); /* synchronises, frees everything; NULL is allowed */

int pn_set_stream(pn_ctx* ctx, void* cuda_stream); /* a cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); the new
                                                      stream waits for the work already enqueued on the old one.  The OLD
                                                      stream must still exist at this call: switch first, destroy it afterwards
                                                      (the CUDA runtime does not validate a destroyed handle -- recording on one
                                                      crashed inside the driver when tried on a B200).  If the runtime does
                                                      report an error for the old stream, the call waits for the whole device
                                                      instead and still switches */
int pn_set_option(pn_ctx* ctx, int key, int value);

/* Integrator state (x, v) of all N bodies.  [N][3] each. */
int pn_set_state(pn_ctx* ctx, const double* pos_dev, const double* vel_dev);
int pn_get_state(pn_ctx* ctx, double* pos_dev, double* vel_dev);
int pn_set_state_host(pn_ctx* ctx, const double* pos_host, const double* vel_host); /* H2D inside; synchronous */
int pn_get_state_host(pn_ctx* ctx, double* pos_host, double* vel_host);             /* D2H inside; synchronous */

/* One force evaluation (equations above) at the given (pos, vel): acc[0] = a_1, acc[i] = a_i.  Does not read or
 * modify the integrator state.  pos, vel, acc: [N][3]. */
int pn_accel(pn_ctx* ctx, const double* pos_dev, const double* vel_dev, double* acc_dev);
int pn_accel_host(pn_ctx* ctx, const double* pos_host, const double* vel_host, double* acc_host); /* synchronous */

/* nsteps steps of the paper's integrator, the classical fourth-order Runge-Kutta method with
 * fixed dt, on the internal state: y = (x, v) of all N bodies, f = (v, a(x, v)), 4 force evaluations per step,
 * weights (1, 2, 2, 1)/6.  The stage update is fused into the kernel that finishes each force evaluation. */
int pn_step(pn_ctx* ctx, double dt, int64_t nsteps);

/* Total 1PN energy of the internal state, Eq. 2.7 with the star-star distances softened;
 * O(N^2) pair sum in compensated fp64.  Synchronises the stream; *E_host is a host double. */
int pn_energy(pn_ctx* ctx, double* E_host);

/* Total 1PN momentum of the internal state, Eq. 2.8 (the third NEXT row of the scope table) in the
 * reading R16 of DESIGN.md: the EIH momentum with every term kept that the paper's error order needs.  P_host: 3 host
 * doubles.  O(N^2) pair sum over the unordered star pairs in compensated fp64.  Synchronises the stream. */
int pn_momentum(pn_ctx* ctx, double* P_host);

/* Bookkeeping for benchmarks. */
int pn_get_launch_count(pn_ctx* ctx, int64_t* n_kernels_host);          /* kernels launched (graph nodes count) */
int pn_get_pair_time(pn_ctx* ctx, double* ms_total_host, int64_t* n_launches_host, int reset); /* PN_OPT_TIME_PAIR: sum of
                                                                            the bracketed pair-stage times and their count
                                                                            since the last reset; synchronises the stream.
                                                                            On the small-system path (PN_PAIR_AUTO) there is
                                                                            no separate pair stage: both come back 0 */
int pn_get_epilogue_time(pn_ctx* ctx, double* ms_total_host, int64_t* n_intervals_host, int reset); /* PN_OPT_TIME_PAIR = 1 and
                                                                            pn_step on its CUDA graph: sum and count of the intervals
                                                                            from the end of one bracketed pair stage to the start
                                                                            of the next one inside a step (3 per step) -- each is
                                                                            one fused epilogue (S2 + S3 + S4, with the Cross terms
                                                                            also their O(N) preparation kernels) plus the launch
                                                                            gaps around it.  For the HBM figure of the O(N) kernels
                                                                            at large N; 0 otherwise.  Synchronises the stream */
int pn_get_pair_config(pn_ctx* ctx, int32_t* cfg_host); /* 8 ints: threads/block, i per thread, j-tile, partial-sum
                                                           slots (j-splits / groups), grid blocks, padded N_s, pipe
                                                           instructions per ordered pair, variant (0 fp64 tiled,
                                                           1 fp32 tiled, 2 fp64 symmetric, 3 fp32 symmetric,
                                                           4 fp64 symmetric, equal-mass form,
                                                           5 fp64 ordered pairs with the Cross terms of Eq. 2.6,
                                                           6 the same with the O(N^2) sum of Eq. 2.3) */

/* The one entry point for callers that cannot allocate device memory (paper_1801_07986_b200/csrc/pn_noalloc.cu).
 * Every other call needs a pn_ctx, and pn_create obtains its work buffers with cudaMalloc.  That rules the library out
 * for a program whose own pool already owns (nearly) all of the GPU's memory or that runs under a fixed memory quota --
 * a further cudaMalloc fails there -- and for a time-critical loop that cannot accept the device-wide stall of
 * cudaMalloc / cudaFree.  This call needs no context and never calls cudaMalloc, cudaFree or an allocating library
 * routine.
 *
 * Computes a_1, the acceleration of the massive object from all stars, Eqs. 2.1 + 2.2 -- the same
 * quantity as row 0 of pn_accel's output on the hot path -- and writes its three components to a1_dev.
 *   N            bodies, 2 <= N <= 1 + PN_NOALLOC_MAX_STARS; PN_EINVAL with a message beyond (nothing is launched)
 *   masses_dev   N device doubles, masses_dev[0] = M; NOT validated (they stay on the device): NaN / negative values propagate
 *   pos_dev, vel_dev   device, fp64, row-major [N][3], body 0 first; vel_dev[0] (v_1) is not used (reading R7)
 *   G > 0 finite; c > 0, +inf for the Newtonian limit
 *   a1_dev       3 device doubles, written by the kernel
 *   cuda_stream  a cudaStream_t (NULL: the legacy default stream); the call is asynchronous on it
 *   errbuf_host / errbuf_len   optional host buffer that receives the error text (pn_last_error does not cover this call)
 * All pointers belong to the caller and are used only during the call's stream-ordered work.
 *
 * The kernel's scratch memory (one partial sum per thread block + a block counter) is a fixed 98 560-byte array inside
 * the library image: every GPU on which the process uses libpn.so holds it until the process exits, and its size is
 * what limits N.  The FIRST call on each device looks up that array's device address (cudaGetSymbolAddress, with that
 * device current), which may load the library's code onto the device: make it during start-up, before any stream
 * capture.  Later calls on that device enqueue one 256-byte memset (the counter must start at zero; the array keeps
 * the previous call's contents) and one kernel.  All calls on a device share the array: calls that overlap on the GPU
 * (different streams, threads or contexts without ordering between them) race and give wrong results -- keep them on
 * one stream or order them with events. */
#define PN_NOALLOC_MAX_STARS (1 << 20)
int pn_bh_accel_noalloc(int64_t N, const double* masses_dev, const double* pos_dev, const double* vel_dev, double G, double c,
                        double* a1_dev, void* cuda_stream, char* errbuf_host, size_t errbuf_len);

const char* pn_last_error(pn_ctx* ctx); /* ctx may be NULL: last error of a failed pn_create in this thread */
const char* pn_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PN_H_ */
