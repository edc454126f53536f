// pn_api.cu -- C-ABI (include/pn.h) of the limited-1PN hot path on B200.  Host-side orchestration only:
// every step of the path runs in the kernels of pn_kernels.cuh.  No CPU fallback exists.
#include "../../include/pn.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "pn_kernels.cuh"

using namespace pn;

namespace {

// threads per epilogue block: 32 stars x (threads / 32) warps that share the partial-sum slots.  8 warps for the hot path: at
// N_s = 16383 the 50 MB of partials come out of L2 and the read is bound by bytes in flight (RK4 step 0.706 -> 0.692 ms;
// 12 and 16 warps and 2 slots per thread in flight are slower, 4 warps x 8 slots equal); no difference once they stream from HBM.
constexpr int kEpiNT = 256;
constexpr int kEpiNTCross = 128;  // 7 - 8 components per slot: 4 warps measure 0.6 % ahead
constexpr int kNT = 128;        // threads per block of the pair / energy / epilogue kernels
constexpr int kTJ = 128;        // j records per shared-memory tile
constexpr int kGraphBatch = 16; // RK4 steps captured in the batched graph
constexpr int kCrossI = 2;      // i-stars per thread of pair_cross_fp64_kernel
constexpr int kCrossTJ = 64;    // its j tile (112 B records)
#ifndef PN_CROSS_SYM_MINB
#define PN_CROSS_SYM_MINB 8
#endif
constexpr int kCrossSymMinB = PN_CROSS_SYM_MINB;  // one-warp blocks per SM of pair_cross_sym_kernel
constexpr int kCrossSymMinStars = 6144; // below: the ordered-pair kernel (too few work items for the triangular grid)
constexpr int kCrossSymMaxGroups = 128; // its partial-sum slots

thread_local std::string g_create_error;

}  // namespace

struct pn_ctx {
    int64_t N = 0;
    int n_stars = 0, np = 0;
    double G = 0, c = 0, eps = 0, M = 0, GM = 0, inv_c2 = 0, eps2 = 0;
    int device = 0, n_sm = 148;  // the CUDA device the context was created on, its SM count
    cudaStream_t stream = nullptr;
    cudaStream_t cap_stream = nullptr;
    cudaEvent_t stream_ev = nullptr;  // orders a new stream after the old one in pn_set_stream
    std::string err;

    // options
    int precision = PN_FP64, use_graph = 1, time_pair = 0, j_split_opt = 0, kernel_opt = PN_PAIR_AUTO, eqm_opt = 1;
    int cross = 0;            // PN_OPT_CROSS_TERMS mask
    CRec* crec = nullptr;     // cross mode: per-star records, block partials and totals of the O(N) sums, 7/8-component partials
    double *cblk = nullptr, *csum = nullptr, *part6 = nullptr;
    int c_split = 1, c_tiles_per_split = 0;
    int c_T = 0, c_m = 0, c_G = 0;  // symmetric Cross kernel: unit tiles of 64 stars in c_G groups of c_m
    double* blk_mom = nullptr;  // pn_momentum scratch
    bool equal_mass = false;  // every star has the same mass > 0
    double gm_eq = 0;

    // pair-kernel launch configuration
    int ipt = 1, n_itiles = 0, n_tiles = 0, n_split = 1, tiles_per_split = 0, max_split = 1;
    // symmetric pair kernel: unit tile U = 32 W I stars, T unit tiles in G groups of m
    int sym_kind = 0, sym_I = 0, sym_W = 0, sym_U = 0, sym_T = 0, sym_m = 0, sym_G = 0;
    // small-system path (small_path_kernel, one cooperative launch per pn_step / pn_accel call): i-stars per warp, blocks
    int small_ok = 0, small_IW = 0, small_blocks = 0;
    double* small_part = nullptr;      // [2][4 small_blocks][3] per-warp partials of a_1
    unsigned int* small_bar = nullptr; // [2]: arrival counter of the grid barrier, give-up flag (small_check)
    unsigned int* small_host_flag = nullptr; // mapped host word the kernel sets when it gives up (small_poll: no copy, no sync)
    bool small_used = false;           // a small-path launch since the last check
    XVRec* small_xv = nullptr;         // [2][np] exchanged stage state of the small-system path with the Cross terms
    unsigned int small_bar_base = 0;   // its value when the next launch starts

    // device buffers.  Two stage sets: [0] integrator state, [1] scratch for pn_accel.
    JRec* jrec[2] = {nullptr, nullptr};
    double* v[2] = {nullptr, nullptr};
    BhState* bh[2] = {nullptr, nullptr};
    double *x0 = nullptr, *v0 = nullptr, *sx = nullptr, *sv = nullptr;
    double* part = nullptr;
    double* bh_part = nullptr;
    unsigned int* ticket = nullptr;
    StepParams* prm = nullptr;
    double *io_pos = nullptr, *io_vel = nullptr, *io_acc = nullptr;  // staging for the *_host entry points
    ERec* erec = nullptr;
    FRec* frec = nullptr;  // two-float records of the fp32-pair variant, rebuilt before every pair launch (tiled kernel)
    FPair* fpair = nullptr;  // the same for pairs of consecutive stars: packed operands of the symmetric f32x2 kernel
    double *blk_prep = nullptr, *blk_pair = nullptr, *d_energy = nullptr;
    int e_blocks = 1;            // blocks of the energy / momentum pair kernels
    long long e_per_block = 1;   // tile pairs (it <= jt) each of them walks

    bool have_state = false;
    double dt_dev = NAN;

    cudaGraphExec_t graph1 = nullptr, graphB = nullptr;
    // timed one-step graph (PN_OPT_TIME_PAIR with graphs): event-record nodes around the pair stage of each RK4 stage;
    // the events are swapped for fresh ones before every launch
    cudaGraph_t graphT_src = nullptr;
    cudaGraphExec_t graphT = nullptr;
    cudaEvent_t tev[8] = {};
    cudaGraphNode_t tnode[8] = {};
    int cap_ev = -1;  // >= 0 while the timed graph is captured: next template event
    int graph_split = -1, graph_precision = -1, graph_sym = -1, graph_eqm = -1;

    int64_t n_launch = 0;
    std::vector<cudaEvent_t> ev;  // pairs (start, stop); a bounded pool, folded into the two sums below when it fills
    size_t ev_used = 0;
    double pair_ms_folded = 0;
    int64_t pair_n_folded = 0;
    std::vector<char> ev_chain;   // per event pair: 1 = it follows the previous pair inside one captured RK4 step, so the time
                                  // from that pair's stop to this pair's start is one epilogue (pn_get_epilogue_time)
    double epi_ms_folded = 0;
    int64_t epi_n_folded = 0;
};

namespace {

int fail(pn_ctx* ctx, int code, const char* fmt, ...)
{
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (ctx)
        ctx->err = buf;
    else
        g_create_error = buf;
    return code;
}

#define PN_CUDA(ctx, call)                                                                                  \
    do {                                                                                                    \
        cudaError_t e_ = (call);                                                                            \
        if (e_ != cudaSuccess)                                                                              \
            return fail(ctx, PN_ECUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

template <typename T>
cudaError_t dalloc(T** p, size_t n)
{
    return cudaMalloc(reinterpret_cast<void**>(p), n * sizeof(T));
}

void choose_split(pn_ctx* c)
{
    int s = c->j_split_opt;
    if (s <= 0) {
        // ~28 blocks per SM (4 resident) keeps the tail of the last wave small; at least one tile per block
        s = (c->n_sm * 28 + c->n_itiles - 1) / c->n_itiles;
    }
    if (s > c->n_tiles) s = c->n_tiles;
    if (s > c->max_split) s = c->max_split;
    if (s < 1) s = 1;
    c->tiles_per_split = (c->n_tiles + s - 1) / s;
    c->n_split = (c->n_tiles + c->tiles_per_split - 1) / c->tiles_per_split;
}

constexpr int kSymMaxGroups = 128;  // partial-sum slots of the symmetric kernel (tail granularity vs epilogue traffic)

// Symmetric (Newton's third law) kernel variants, by problem size (measured on a B200, profiles/r2_ncu_summary.md): the
// j-split form (4 warps share one 128 x 128 unit-tile pair: work items a quarter as long) where the grid is small,
// one-warp blocks around N_s = 16384, 512-star unit tiles (4 warps, 128 i-stars each) from 36000 stars on, where the
// tile prologue and flush weigh least.
enum { SYM_W1_U128 = 0, SYM_JS_U128 = 1, SYM_W4_U512 = 2 };

void choose_sym(pn_ctx* c)
{
    // measured with the Gray-code walk (profiles/r2_ncu_summary.md section 4): one-warp blocks win only right below 16384 stars,
    // where 128 one-tile groups give 8256 items of one 128 x 128 tile pair (N_s = 16383: 0.772 against 0.758; at 15359 the
    // j-split form is ahead again, 0.746 against 0.726); everywhere else below 36000 stars the j-split form, whose items are a
    // quarter as long; 512-star tiles from 36000 stars on
    if (c->n_stars < 16000)
        c->sym_kind = SYM_JS_U128;
    else if (c->n_stars <= 16384)
        c->sym_kind = SYM_W1_U128;
    else if (c->n_stars < 36000)
        c->sym_kind = SYM_JS_U128;
    else
        c->sym_kind = SYM_W4_U512;
    // diagnostics only (bench.py --variants: the table behind the thresholds above): PN_SYM_FORM=w1|js|u512 in the environment
    // of pn_create forces a form.  The form fixes the padding and the buffer sizes, hence creation time and not pn_set_option.
    if (const char* f = std::getenv("PN_SYM_FORM")) {
        if (!std::strcmp(f, "w1")) c->sym_kind = SYM_W1_U128;
        else if (!std::strcmp(f, "js")) c->sym_kind = SYM_JS_U128;
        else if (!std::strcmp(f, "u512")) c->sym_kind = SYM_W4_U512;
    }
    c->sym_I = 4;
    c->sym_W = (c->sym_kind == SYM_W1_U128) ? 1 : 4;
    c->sym_U = (c->sym_kind == SYM_W4_U512) ? 512 : 128;
}

void choose_sym_groups(pn_ctx* c)
{
    c->sym_T = c->np / c->sym_U;
    c->sym_m = (c->sym_T + kSymMaxGroups - 1) / kSymMaxGroups;
    c->sym_G = (c->sym_T + c->sym_m - 1) / c->sym_m;
}

bool use_sym(const pn_ctx* c)
{
    if (c->kernel_opt == PN_PAIR_SYMMETRIC) return true;
    if (c->kernel_opt == PN_PAIR_TILED) return false;
    return c->n_stars >= 3072;
}

// small systems: the whole call in one cooperative launch (fp64 hot path only; PN_PAIR_TILED / PN_PAIR_SYMMETRIC ask for
// the multi-kernel path by name)
bool use_small(const pn_ctx* c)
{
    return c->small_ok && c->kernel_opt == PN_PAIR_AUTO && c->precision == PN_FP64 && !c->cross;
}

// ... and with the Cross terms up to kSmallCrossMaxStars stars (the per-star Cross records of every star must fit in shared memory)
bool use_small_cross(const pn_ctx* c)
{
    return c->small_ok && c->small_xv && c->kernel_opt == PN_PAIR_AUTO && c->cross && c->n_stars <= kSmallCrossMaxStars;
}

bool use_eqm(const pn_ctx* c) { return c->equal_mass && c->eqm_opt && use_sym(c) && !use_small(c); }

// kernels of the pair stage of one force evaluation (the epilogue is counted by the callers)
int kernels_per_eval(const pn_ctx* c) { return c->cross ? 3 : (c->precision == PN_FP32_PAIR ? 2 : 1); }

// Cross terms: every unordered pair once from kCrossSymMinStars stars on (PN_PAIR_TILED / PN_PAIR_SYMMETRIC force either kernel)
bool cross_sym(const pn_ctx* c)
{
    return c->kernel_opt == PN_PAIR_SYMMETRIC || (c->kernel_opt == PN_PAIR_AUTO && c->n_stars >= kCrossSymMinStars);
}

int active_split(const pn_ctx* c) { return c->cross ? (cross_sym(c) ? c->c_G : c->c_split) : (use_sym(c) ? c->sym_G : c->n_split); }

void destroy_graphs(pn_ctx* c)
{
    if (c->graph1) cudaGraphExecDestroy(c->graph1), c->graph1 = nullptr;
    if (c->graphB) cudaGraphExecDestroy(c->graphB), c->graphB = nullptr;
    if (c->graphT) cudaGraphExecDestroy(c->graphT), c->graphT = nullptr;
    if (c->graphT_src) cudaGraphDestroy(c->graphT_src), c->graphT_src = nullptr;
}

// ---- small-system path ------------------------------------------------------------------------------------------
constexpr int kSmallMaxStars = 3071;
constexpr int kSmallMaxIW = 6;

template <int MODE, int IW, bool MASK>
const void* small_kernel_ptr()
{
    constexpr int JU = IW == 1 ? 8 : (IW == 2 ? 4 : 2);
    return reinterpret_cast<const void*>(small_path_kernel<MODE, IW, JU, MASK>);
}

template <int MODE>
const void* small_kernel(int iw, bool mask)
{
    switch (iw) {
        case 1: return mask ? small_kernel_ptr<MODE, 1, true>() : small_kernel_ptr<MODE, 1, false>();
        case 2: return mask ? small_kernel_ptr<MODE, 2, true>() : small_kernel_ptr<MODE, 2, false>();
        case 3: return mask ? small_kernel_ptr<MODE, 3, true>() : small_kernel_ptr<MODE, 3, false>();
        case 4: return mask ? small_kernel_ptr<MODE, 4, true>() : small_kernel_ptr<MODE, 4, false>();
        case 5: return mask ? small_kernel_ptr<MODE, 5, true>() : small_kernel_ptr<MODE, 5, false>();
        default: return mask ? small_kernel_ptr<MODE, 6, true>() : small_kernel_ptr<MODE, 6, false>();
    }
}

int small_launch_common(pn_ctx* c, const void* fn, void** args, size_t smem, int64_t n_eval);

// one cooperative launch: mode MODE_RK4 runs nsteps classical RK4 steps on the integrator state (stage set 0, with stage
// set 1 as the second position buffer), MODE_ACCEL one force evaluation on stage set 1
int launch_small(pn_ctx* c, int mode, double dt, int64_t nsteps, double* acc_out)
{
    SmallArgs a;
    const int set = (mode == MODE_RK4) ? 0 : 1;
    a.jrec[0] = c->jrec[set], a.jrec[1] = c->jrec[1];
    a.v = c->v[set];
    a.x0 = c->x0, a.v0 = c->v0, a.sx = c->sx, a.sv = c->sv;
    a.bh = c->bh[set];
    a.bh_part = c->small_part;
    a.bar = c->small_bar;
    a.host_flag = c->small_host_flag;
    a.acc_out = acc_out;
    a.n_stars = c->n_stars, a.np = c->np;
    a.GM = c->GM, a.inv_c2 = c->inv_c2, a.eps2 = c->eps2, a.dt = dt;
    a.nsteps = nsteps;
    a.bar_base = c->small_bar_base;
    const bool mask = (c->eps2 == 0.0);
    const void* fn = (mode == MODE_RK4) ? small_kernel<MODE_RK4>(c->small_IW, mask) : small_kernel<MODE_ACCEL>(c->small_IW, mask);
    void* args[] = {&a};
    const size_t smem = (size_t)c->np * sizeof(JRec);
    return small_launch_common(c, fn, args, smem, (mode == MODE_RK4) ? 4 * nsteps : 1);
}

// one cooperative launch of a small-system kernel; on success the host's copy of the barrier counter moves on
int small_launch_common(pn_ctx* c, const void* fn, void** args, size_t smem, int64_t n_eval)
{
    // blocks of two grids that both spin at their own barrier must never share the device half and half: cooperative launches
    // of this process run one after the other (each waits for the event the previous one recorded, on whatever stream)
    static std::mutex g_small_mu;
    static cudaEvent_t g_small_ev[16] = {};
    std::lock_guard<std::mutex> lock(g_small_mu);
    cudaEvent_t& chain = g_small_ev[c->device & 15];
    if (chain)
        PN_CUDA(c, cudaStreamWaitEvent(c->stream, chain, 0));
    else
        PN_CUDA(c, cudaEventCreateWithFlags(&chain, cudaEventDisableTiming));
    cudaError_t e = cudaLaunchCooperativeKernel(fn, dim3(c->small_blocks), dim3(kSmallNT), args, smem, c->stream);
    if (e == cudaErrorCooperativeLaunchTooLarge || e == cudaErrorLaunchOutOfResources) {
        // the blocks cannot all be resident (SMs taken by another client of the device): nothing was launched; the callers fall
        // back to the multi-kernel path for the rest of this context's life
        cudaGetLastError();
        c->small_ok = 0;
        return PN_ESTATE;
    }
    PN_CUDA(c, e);
    PN_CUDA(c, cudaEventRecord(chain, c->stream));
    c->small_used = true;
    c->small_bar_base += (unsigned int)((uint64_t)n_eval * (uint64_t)c->small_blocks);  // modulo 2^32, like the counter
    return PN_OK;
}

template <int MODE, bool BHX>
const void* small_cross_kernel_ptr(int iw)
{
    switch (iw) {
        case 1: return reinterpret_cast<const void*>(small_cross_kernel<MODE, 1, BHX>);
        case 2: return reinterpret_cast<const void*>(small_cross_kernel<MODE, 2, BHX>);
        default: return reinterpret_cast<const void*>(small_cross_kernel<MODE, 3, BHX>);
    }
}

const void* small_cross_fn(int mode, int iw, bool bhx)
{
    if (mode == MODE_RK4) return bhx ? small_cross_kernel_ptr<MODE_RK4, true>(iw) : small_cross_kernel_ptr<MODE_RK4, false>(iw);
    return bhx ? small_cross_kernel_ptr<MODE_ACCEL, true>(iw) : small_cross_kernel_ptr<MODE_ACCEL, false>(iw);
}

// the same with the Cross terms (PN_OPT_CROSS_TERMS): small_cross_kernel
int launch_small_cross(pn_ctx* c, int mode, double dt, int64_t nsteps, double* acc_out)
{
    SmallCrossArgs a;
    const int set = (mode == MODE_RK4) ? 0 : 1;
    a.jrec_in = c->jrec[set], a.jrec_out = c->jrec[0];
    a.v = c->v[set];
    a.x0 = c->x0, a.v0 = c->v0, a.sx = c->sx, a.sv = c->sv;
    a.bh = c->bh[set];
    a.xv = c->small_xv;
    a.bh_part = c->small_part;
    a.bar = c->small_bar;
    a.host_flag = c->small_host_flag;
    a.acc_out = acc_out;
    a.n_stars = c->n_stars, a.np = c->np;
    a.GM = c->GM, a.inv_c2 = c->inv_c2, a.eps2 = c->eps2, a.dt = dt;
    a.nsteps = nsteps;
    a.bar_base = c->small_bar_base;
    void* args[] = {&a};
    return small_launch_common(c, small_cross_fn(mode, c->small_IW, (c->cross & PN_CROSS_BH) != 0), args,
                               (size_t)c->np * kSmallCrossBytesPerStar, (mode == MODE_RK4) ? 4 * nsteps : 1);
}

// sizes the small-system path and checks that the device can run it (cooperative launch, shared memory, residency)
cudaError_t prepare_small(pn_ctx* c)
{
    c->small_ok = 0;
    if (c->n_stars > kSmallMaxStars) return cudaSuccess;
    int coop = 0;
    cudaError_t e = cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, c->device);
    if (e != cudaSuccess || !coop) return e;
    const int warps = 4 * c->n_sm;
    c->small_IW = std::min(kSmallMaxIW, std::max(1, (c->n_stars + warps - 1) / warps));
    c->small_blocks = (c->n_stars + 4 * c->small_IW - 1) / (4 * c->small_IW);
    if (c->small_blocks > c->n_sm) return cudaSuccess;  // one block per SM: every block must be resident
    // the attribute belongs to the kernel, not to the context: always the largest size any context may ask of it
    const int smem = ((kSmallMaxStars + 255) / 256 * 256) * (int)sizeof(JRec);
    for (int mode = 0; mode < 2; ++mode)
        for (int mask = 0; mask < 2; ++mask) {
            const void* fn = mode ? small_kernel<MODE_RK4>(c->small_IW, mask != 0) : small_kernel<MODE_ACCEL>(c->small_IW, mask != 0);
            e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
            if (e != cudaSuccess) return e;
        }
    e = dalloc(&c->small_part, 2 * 3 * (size_t)4 * c->small_blocks);
    if (e == cudaSuccess) e = dalloc(&c->small_bar, 2);
    if (e == cudaSuccess) e = cudaMemset(c->small_bar, 0, 2 * sizeof(unsigned int));
    if (e == cudaSuccess && !c->small_host_flag) {
        e = cudaHostAlloc(reinterpret_cast<void**>(&c->small_host_flag), sizeof(unsigned int), cudaHostAllocMapped);
        if (e == cudaSuccess) *c->small_host_flag = 0;
    }
    if (e == cudaSuccess) c->small_ok = 1;
    return e;
}

// ---- launches ---------------------------------------------------------------------------------------------
template <int I, int JU, int MINB, bool MASK>
void launch_pair_fp64(pn_ctx* c, int set, cudaStream_t st)
{
    dim3 grid(c->n_itiles, c->n_split);
    pair_fp64_kernel<I, JU, MINB, kNT, kTJ, MASK><<<grid, kNT, 0, st>>>(c->jrec[set], c->part, c->np, c->tiles_per_split, c->eps2);
}

// symmetric kernels <I, W, MINB>: one block per work item (group pair), W warps
template <int I, int W, int MINB, bool JS>
cudaError_t prepare_sym()
{
    const int bytes = kSymSmemBytes<I, W, JS>;
    cudaError_t e = cudaFuncSetAttribute(pair_sym_fp64_kernel<I, W, MINB, false, false, JS>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(pair_sym_fp64_kernel<I, W, MINB, true, false, JS>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(pair_sym_fp64_kernel<I, W, MINB, false, true, JS>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(pair_sym_fp64_kernel<I, W, MINB, true, true, JS>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    return e;
}

template <int W, int MINB>
cudaError_t prepare_sym32()
{
    const int bytes = kSym32SmemBytes<W>;
    cudaError_t e = cudaFuncSetAttribute(pair_sym_fp32_kernel<W, MINB, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(pair_sym_fp32_kernel<W, MINB, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(pair_sym_fp32_kernel<W, MINB, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(pair_sym_fp32_kernel<W, MINB, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    return e;
}

template <int W, int MINB, bool MASK, bool EQM>
void launch_pair_sym32_v(pn_ctx* c, cudaStream_t st)
{
    const int items = c->sym_G * (c->sym_G + 1) / 2;
    pair_sym_fp32_kernel<W, MINB, MASK, EQM><<<items, 32 * W, kSym32SmemBytes<W>, st>>>(c->fpair, c->part, c->np, c->sym_T, c->sym_m,
                                                                                      (float)c->eps2, c->gm_eq);
}

template <int W, int MINB>
void launch_pair_sym32(pn_ctx* c, cudaStream_t st)
{
    const bool mask = (c->eps2 == 0.0), eqm = use_eqm(c);
    if (mask)
        eqm ? launch_pair_sym32_v<W, MINB, true, true>(c, st) : launch_pair_sym32_v<W, MINB, true, false>(c, st);
    else
        eqm ? launch_pair_sym32_v<W, MINB, false, true>(c, st) : launch_pair_sym32_v<W, MINB, false, false>(c, st);
}

template <int I, int W, int MINB, bool JS, bool MASK, bool EQM>
void launch_pair_sym_v(pn_ctx* c, int set, cudaStream_t st)
{
    const int items = c->sym_G * (c->sym_G + 1) / 2;
    pair_sym_fp64_kernel<I, W, MINB, MASK, EQM, JS><<<items, 32 * W, kSymSmemBytes<I, W, JS>, st>>>(c->jrec[set], c->part, c->np, c->sym_T,
                                                                                                   c->sym_m, c->eps2, c->gm_eq, 0);
}

template <int I, int W, int MINB, bool JS>
void launch_pair_sym(pn_ctx* c, int set, cudaStream_t st)
{
    const bool mask = (c->eps2 == 0.0), eqm = use_eqm(c);
    if (mask)
        eqm ? launch_pair_sym_v<I, W, MINB, JS, true, true>(c, set, st) : launch_pair_sym_v<I, W, MINB, JS, true, false>(c, set, st);
    else
        eqm ? launch_pair_sym_v<I, W, MINB, JS, false, true>(c, set, st) : launch_pair_sym_v<I, W, MINB, JS, false, false>(c, set, st);
}

constexpr size_t kMaxEvents = 4096;  // PN_OPT_TIME_PAIR event pool: 2048 timed launches between folds

// adds the elapsed times of the recorded event pairs to the running sums and recycles the pool (synchronises the stream)
int fold_events(pn_ctx* c)
{
    if (c->ev_used == 0) return PN_OK;
    PN_CUDA(c, cudaStreamSynchronize(c->stream));
    for (size_t q = 0; q + 1 < c->ev_used; q += 2) {
        float ms = 0;
        PN_CUDA(c, cudaEventElapsedTime(&ms, c->ev[q], c->ev[q + 1]));
        c->pair_ms_folded += ms;
        if (q / 2 < c->ev_chain.size() && c->ev_chain[q / 2]) {
            PN_CUDA(c, cudaEventElapsedTime(&ms, c->ev[q - 1], c->ev[q]));
            c->epi_ms_folded += ms;
            c->epi_n_folded += 1;
        }
    }
    c->ev_chain.assign(c->ev_chain.size(), 0);
    c->pair_n_folded += (int64_t)(c->ev_used / 2);
    c->ev_used = 0;
    return PN_OK;
}

int reserve_events(pn_ctx* c, size_t n)
{
    if (c->ev_used + n > kMaxEvents)
        if (int rc = fold_events(c)) return rc;
    while (c->ev_used + n > c->ev.size()) {
        cudaEvent_t e;
        PN_CUDA(c, cudaEventCreate(&e));
        c->ev.push_back(e);
    }
    return PN_OK;
}

int launch_pair(pn_ctx* c, int set, cudaStream_t st, bool timed)
{
    if (timed && c->cap_ev >= 0) {
        PN_CUDA(c, cudaEventRecordWithFlags(c->tev[c->cap_ev], st, cudaEventRecordExternal));  // a real event-record node
    } else if (timed) {
        if (int rc = reserve_events(c, 2)) return rc;
        PN_CUDA(c, cudaEventRecord(c->ev[c->ev_used], st));
    }
    const bool mask = (c->eps2 == 0.0);
    if (c->cross) {  // NEXT-1: star-star Newtonian + pair part of [a_i]_Cross in one ordered-pair pass (fp64)
        const int nb = c->np / kNT;
        const bool ceqm = cross_sym(c) && c->equal_mass && c->eqm_opt;  // equal-mass form of the symmetric Cross kernel
        cross_prep_kernel<kNT><<<nb, kNT, 0, st>>>(c->jrec[set], c->v[set], c->bh[set], c->crec, c->cblk, c->n_stars, c->np, c->GM,
                                                  ceqm ? 1.0 / c->gm_eq : 1.0);
        cross_sum_kernel<<<1, 256, 0, st>>>(c->cblk, nb, c->csum);
        const double GM4 = 4.0 * c->GM;
        if (cross_sym(c)) {  // every unordered pair once
            const int items = c->c_G * (c->c_G + 1) / 2;
            const bool bhx = (c->cross & PN_CROSS_BH) != 0;
#define PN_LAUNCH_CSYM(B, E)                                                                                                          \
    pair_cross_sym_kernel<kCrossSymMinB, B, E><<<items, 32, kCrossSymSmemBytes<B>, st>>>(c->crec, c->part6, c->np, c->c_T, c->c_m, c->eps2, \
                                                                                         GM4, c->gm_eq)
            if (bhx)
                ceqm ? PN_LAUNCH_CSYM(true, true) : PN_LAUNCH_CSYM(true, false);
            else
                ceqm ? PN_LAUNCH_CSYM(false, true) : PN_LAUNCH_CSYM(false, false);
#undef PN_LAUNCH_CSYM
        } else {
            dim3 grid(c->np / (kCrossI * kNT), c->c_split);
            if (c->cross & PN_CROSS_BH)
                pair_cross_fp64_kernel<kCrossI, 2, kNT, kCrossTJ, true><<<grid, kNT, 0, st>>>(c->crec, c->part6, c->np, c->c_tiles_per_split,
                                                                                             c->eps2, GM4);
            else
                pair_cross_fp64_kernel<kCrossI, 2, kNT, kCrossTJ, false><<<grid, kNT, 0, st>>>(c->crec, c->part6, c->np, c->c_tiles_per_split,
                                                                                              c->eps2, GM4);
        }
    } else if (c->precision == PN_FP32_PAIR) {
        if (use_sym(c))
            split_pair_kernel<<<(c->np + 255) / 256, 256, 0, st>>>(c->jrec[set], c->fpair, c->n_stars, c->np);
        else
            split_kernel<<<(c->np + 255) / 256, 256, 0, st>>>(c->jrec[set], c->frec, c->n_stars, c->np);
        PN_CUDA(c, cudaGetLastError());
        dim3 grid(c->n_itiles, c->n_split);
        const float e2 = (float)c->eps2;
        if (use_sym(c)) {
            if (c->sym_U == 128)
                launch_pair_sym32<1, 12>(c, st);
            else
                launch_pair_sym32<4, 3>(c, st);
        } else if (c->ipt == 2)
            mask ? pair_fp32_kernel<2, kNT, kTJ, 32, true><<<grid, kNT, 0, st>>>(c->frec, c->part, c->np, c->tiles_per_split, e2)
                 : pair_fp32_kernel<2, kNT, kTJ, 32, false><<<grid, kNT, 0, st>>>(c->frec, c->part, c->np, c->tiles_per_split, e2);
        else
            mask ? pair_fp32_kernel<1, kNT, kTJ, 32, true><<<grid, kNT, 0, st>>>(c->frec, c->part, c->np, c->tiles_per_split, e2)
                 : pair_fp32_kernel<1, kNT, kTJ, 32, false><<<grid, kNT, 0, st>>>(c->frec, c->part, c->np, c->tiles_per_split, e2);
    } else if (use_sym(c)) {
        if (c->sym_kind == SYM_JS_U128)
            launch_pair_sym<4, 4, 3, true>(c, set, st);
        else if (c->sym_kind == SYM_W1_U128)
            launch_pair_sym<4, 1, 12, false>(c, set, st);
        else
            launch_pair_sym<4, 4, 3, false>(c, set, st);
    } else if (c->ipt == 2)
        mask ? launch_pair_fp64<2, 4, 4, true>(c, set, st) : launch_pair_fp64<2, 4, 4, false>(c, set, st);
    else
        mask ? launch_pair_fp64<1, 8, 4, true>(c, set, st) : launch_pair_fp64<1, 8, 4, false>(c, set, st);
    PN_CUDA(c, cudaGetLastError());
    if (timed && c->cap_ev >= 0) {
        PN_CUDA(c, cudaEventRecordWithFlags(c->tev[c->cap_ev + 1], st, cudaEventRecordExternal));
        c->cap_ev += 2;
    } else if (timed) {
        PN_CUDA(c, cudaEventRecord(c->ev[c->ev_used + 1], st));
        c->ev_used += 2;
    }
    return PN_OK;
}

EpiArgs epi_args(pn_ctx* c, int set, double* acc_out)
{
    EpiArgs a;
    a.jrec = c->jrec[set];
    a.v = c->v[set];
    a.part = c->cross ? c->part6 : c->part;
    a.csum = c->csum;
    a.x0 = c->x0, a.v0 = c->v0, a.sx = c->sx, a.sv = c->sv;
    a.bh = c->bh[set];
    a.bh_part = c->bh_part;
    a.ticket = c->ticket;
    a.acc_out = acc_out;
    a.prm = c->prm;
    a.n_stars = c->n_stars, a.np = c->np, a.n_split = active_split(c);
    a.GM = c->GM, a.inv_c2 = c->inv_c2;
    return a;
}

// one classical-RK4 step = 4 x (pair kernel, fused epilogue)
int enqueue_rk4_step(pn_ctx* c, cudaStream_t st, bool timed)
{
    const EpiArgs a = epi_args(c, 0, nullptr);
    const int grid = c->np / kEpiStars;
    for (int stage = 0; stage < 4; ++stage) {
        int rc = launch_pair(c, 0, st, timed && (c->time_pair != 2 || stage == 0));
        if (rc) return rc;
        if (c->cross & PN_CROSS_BH)
            epilogue_kernel<MODE_RK4, kEpiNTCross, 2><<<grid, kEpiNTCross, 0, st>>>(a, stage);
        else if (c->cross)
            epilogue_kernel<MODE_RK4, kEpiNTCross, 1><<<grid, kEpiNTCross, 0, st>>>(a, stage);
        else
            epilogue_kernel<MODE_RK4, kEpiNT, 0><<<grid, kEpiNT, 0, st>>>(a, stage);
        PN_CUDA(c, cudaGetLastError());
    }
    return PN_OK;
}

int build_graph(pn_ctx* c, int nrep, cudaGraphExec_t* out)
{
    cudaGraph_t g = nullptr;
    PN_CUDA(c, cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal));
    int rc = PN_OK;
    for (int r = 0; r < nrep && rc == PN_OK; ++r) rc = enqueue_rk4_step(c, c->cap_stream, false);
    cudaError_t e = cudaStreamEndCapture(c->cap_stream, &g);
    if (rc != PN_OK) {
        if (g) cudaGraphDestroy(g);
        return rc;
    }
    if (e != cudaSuccess) return fail(c, PN_ECUDA, "cudaStreamEndCapture failed: %s", cudaGetErrorString(e));
    e = cudaGraphInstantiate(out, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) return fail(c, PN_ECUDA, "cudaGraphInstantiate failed: %s", cudaGetErrorString(e));
    return PN_OK;
}

// the event-record nodes of the captured timed graph, by template event
int find_timed_nodes(pn_ctx* c)
{
    size_t n = 0;
    PN_CUDA(c, cudaGraphGetNodes(c->graphT_src, nullptr, &n));
    std::vector<cudaGraphNode_t> nodes(n);
    PN_CUDA(c, cudaGraphGetNodes(c->graphT_src, nodes.data(), &n));
    int found = 0;
    for (cudaGraphNode_t nd : nodes) {
        cudaGraphNodeType t;
        PN_CUDA(c, cudaGraphNodeGetType(nd, &t));
        if (t != cudaGraphNodeTypeEventRecord) continue;
        cudaEvent_t ev;
        PN_CUDA(c, cudaGraphEventRecordNodeGetEvent(nd, &ev));
        for (int q = 0; q < 8; ++q)
            if (ev == c->tev[q]) c->tnode[q] = nd, ++found;
    }
    const int want = (c->time_pair == 2) ? 2 : 8;
    if (found != want) return fail(c, PN_ECUDA, "timed graph: %d of %d event-record nodes found", found, want);
    return PN_OK;
}

// One RK4 step with event-record nodes around the pair stage of each of the 4 force evaluations.
int build_timed_graph(pn_ctx* c)
{
    for (int q = 0; q < 8; ++q)
        if (!c->tev[q]) PN_CUDA(c, cudaEventCreate(&c->tev[q]));
    PN_CUDA(c, cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeThreadLocal));
    c->cap_ev = 0;
    int rc = enqueue_rk4_step(c, c->cap_stream, true);
    c->cap_ev = -1;
    cudaError_t e = cudaStreamEndCapture(c->cap_stream, &c->graphT_src);
    if (rc == PN_OK && e != cudaSuccess) rc = fail(c, PN_ECUDA, "cudaStreamEndCapture (timed graph) failed: %s", cudaGetErrorString(e));
    if (rc == PN_OK) rc = find_timed_nodes(c);
    if (rc == PN_OK) {
        e = cudaGraphInstantiate(&c->graphT, c->graphT_src, 0);
        if (e != cudaSuccess) rc = fail(c, PN_ECUDA, "cudaGraphInstantiate (timed graph) failed: %s", cudaGetErrorString(e));
    }
    if (rc != PN_OK) {  // nothing half-built survives a failure: the next call starts from scratch
        destroy_graphs(c);
        for (cudaGraphNode_t& nd : c->tnode) nd = nullptr;
    }
    return rc;
}

// every entry point: the context must exist and its device must be the calling thread's current device (device
// pointers and kernel launches of a context belong to the device it was created on)
int check_ctx(pn_ctx* c)
{
    if (!c) return fail(nullptr, PN_EINVAL, "null context");
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return fail(c, PN_ECUDA, "cudaGetDevice failed");
    }
    if (dev != c->device)
        return fail(c, PN_EINVAL, "the context lives on CUDA device %d but the current device is %d (cudaSetDevice first)", c->device, dev);
    return PN_OK;
}

// after a synchronisation of the context's stream: did a grid barrier of the small-system path give up?  (one 4-byte read)
int small_check(pn_ctx* c)
{
    if (!c->small_used) return PN_OK;
    c->small_used = false;
    unsigned int flag = 0;
    PN_CUDA(c, cudaMemcpy(&flag, c->small_bar + 1, sizeof flag, cudaMemcpyDeviceToHost));
    if (!flag) return PN_OK;
    cudaMemset(c->small_bar, 0, 2 * sizeof(unsigned int));
    if (c->small_host_flag) *reinterpret_cast<volatile unsigned int*>(c->small_host_flag) = 0;
    c->small_bar_base = 0;
    c->small_ok = 0;
    return fail(c, PN_ECUDA, "small-system path: a grid barrier timed out (the results of the last pn_step / pn_accel are invalid, set the "
                             "state again); the context uses the multi-kernel path from now on");
}

// Device-only callers (pn_step, then pn_accel or pn_get_state with their own stream synchronisation) never reach small_check.
// The kernel that gives up also sets a word in mapped host memory; every asynchronous entry point looks at it first (a plain
// host read: no copy, no synchronisation), so a failed launch is reported by the NEXT call on the context at the latest.
int small_poll(pn_ctx* c)
{
    if (!c->small_host_flag || !*reinterpret_cast<volatile unsigned int*>(c->small_host_flag)) return PN_OK;
    PN_CUDA(c, cudaStreamSynchronize(c->stream));  // the launch that gave up drains within the barrier's bound
    c->small_used = true;
    return small_check(c);
}

}  // namespace

// =================================================================================================== C-ABI ==
extern "C" {

const char* pn_version(void) { return "pn-b200 0.1 (sm_100a)"; }

const char* pn_last_error(pn_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

int pn_create(pn_ctx** out, int64_t N, const double* masses, double G, double c, double softening)
{
    if (!out) return fail(nullptr, PN_EINVAL, "pn_create: out is null");
    *out = nullptr;
    if (N < 2 || N > (int64_t)1 << 24) return fail(nullptr, PN_EINVAL, "pn_create: N = %lld out of range [2, 2^24]", (long long)N);
    if (!masses) return fail(nullptr, PN_EINVAL, "pn_create: masses is null");
    if (!(G > 0) || std::isinf(G)) return fail(nullptr, PN_EINVAL, "pn_create: G must be finite and > 0");
    if (!(c > 0)) return fail(nullptr, PN_EINVAL, "pn_create: c must be > 0 (+inf allowed)");
    if (!(softening >= 0) || std::isinf(softening)) return fail(nullptr, PN_EINVAL, "pn_create: softening must be finite and >= 0");
    if (!(masses[0] > 0) || std::isinf(masses[0])) return fail(nullptr, PN_EINVAL, "pn_create: masses[0] = M must be finite and > 0");
    for (int64_t i = 1; i < N; ++i)
        if (!(masses[i] >= 0) || std::isinf(masses[i]))
            return fail(nullptr, PN_EINVAL, "pn_create: masses[%lld] must be finite and >= 0", (long long)i);

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(nullptr, PN_ECUDA, "pn_create: no CUDA device (this library has no CPU fallback)");
    }

    pn_ctx* ctx = new (std::nothrow) pn_ctx;
    if (!ctx) return fail(nullptr, PN_ENOMEM, "pn_create: out of host memory");
    if (cudaGetDevice(&ctx->device) != cudaSuccess ||
        cudaDeviceGetAttribute(&ctx->n_sm, cudaDevAttrMultiProcessorCount, ctx->device) != cudaSuccess || ctx->n_sm < 1) {
        cudaGetLastError();
        delete ctx;
        return fail(nullptr, PN_ECUDA, "pn_create: cannot query the current CUDA device");
    }
    ctx->N = N;
    ctx->n_stars = (int)(N - 1);
    ctx->G = G, ctx->c = c, ctx->eps = softening, ctx->M = masses[0];
    ctx->GM = G * masses[0];
    ctx->inv_c2 = std::isinf(c) ? 0.0 : 1.0 / (c * c);
    ctx->eps2 = softening * softening;
    ctx->equal_mass = masses[1] > 0;
    for (int64_t i = 2; i < N && ctx->equal_mass; ++i) ctx->equal_mass = (masses[i] == masses[1]);
    ctx->gm_eq = G * masses[1];

    // i per thread: larger i-tiles amortise the shared-memory broadcast; small N needs more blocks instead
    ctx->ipt = ctx->n_stars >= 3072 ? 2 : 1;
    choose_sym(ctx);
    const int ti = std::max(std::max(ctx->ipt * kNT, ctx->sym_U), kCrossI * kNT);  // powers of two: np suits every pair kernel
    ctx->np = (ctx->n_stars + ti - 1) / ti * ti;
    choose_sym_groups(ctx);
    ctx->n_itiles = ctx->np / (ctx->ipt * kNT);
    ctx->n_tiles = ctx->np / kTJ;
    ctx->max_split = std::min(ctx->n_tiles, 64);
    choose_split(ctx);

#define CREATE_CUDA(call)                                                                   \
    do {                                                                                    \
        cudaError_t e_ = (call);                                                            \
        if (e_ != cudaSuccess) {                                                            \
            int code_ = (e_ == cudaErrorMemoryAllocation) ? PN_ENOMEM : PN_ECUDA;           \
            fail(nullptr, code_, "pn_create: %s failed: %s", #call, cudaGetErrorString(e_)); \
            pn_destroy(ctx);                                                                \
            return code_;                                                                   \
        }                                                                                   \
    } while (0)

    const size_t np = ctx->np;
    CREATE_CUDA(cudaStreamCreateWithFlags(&ctx->cap_stream, cudaStreamNonBlocking));
    CREATE_CUDA(cudaEventCreateWithFlags(&ctx->stream_ev, cudaEventDisableTiming));
    for (int s = 0; s < 2; ++s) {
        CREATE_CUDA(dalloc(&ctx->jrec[s], np));
        CREATE_CUDA(dalloc(&ctx->v[s], 3 * np));
        CREATE_CUDA(dalloc(&ctx->bh[s], 1));
        CREATE_CUDA(cudaMemset(ctx->v[s], 0, 3 * np * sizeof(double)));
        CREATE_CUDA(cudaMemset(ctx->bh[s], 0, sizeof(BhState)));
    }
    CREATE_CUDA(dalloc(&ctx->x0, 3 * np));
    CREATE_CUDA(dalloc(&ctx->v0, 3 * np));
    CREATE_CUDA(dalloc(&ctx->sx, 3 * np));
    CREATE_CUDA(dalloc(&ctx->sv, 3 * np));
    CREATE_CUDA((prepare_sym<4, 1, 12, false>()));
    CREATE_CUDA((prepare_sym<4, 4, 3, true>()));
    CREATE_CUDA((prepare_sym<4, 4, 3, false>()));
    CREATE_CUDA((prepare_sym32<1, 12>()));
    CREATE_CUDA((prepare_sym32<4, 3>()));
    CREATE_CUDA(prepare_small(ctx));
    CREATE_CUDA(dalloc(&ctx->part, (size_t)std::max(ctx->max_split, ctx->sym_G) * 3 * np));
    CREATE_CUDA(dalloc(&ctx->bh_part, 3 * (np / kEpiStars)));
    CREATE_CUDA(dalloc(&ctx->ticket, 1));
    CREATE_CUDA(cudaMemset(ctx->ticket, 0, sizeof(unsigned int)));
    CREATE_CUDA(dalloc(&ctx->prm, 1));
    CREATE_CUDA(dalloc(&ctx->io_pos, 3 * (size_t)N));
    CREATE_CUDA(dalloc(&ctx->io_vel, 3 * (size_t)N));
    CREATE_CUDA(dalloc(&ctx->io_acc, 3 * (size_t)N));
    CREATE_CUDA(dalloc(&ctx->erec, np));
    CREATE_CUDA(dalloc(&ctx->frec, np));
    CREATE_CUDA(dalloc(&ctx->fpair, np / 2));
    {
        const int n_it = (int)(np / kNT);
        // the energy / momentum pair kernels share out the n_it (n_it + 1) / 2 tile pairs (it <= jt) evenly: one full wave of
        // blocks (7 of 72 registers x 128 threads per SM), every block the same number of consecutive pairs
        const long long n_pairs = (long long)n_it * (n_it + 1) / 2;
        const long long want = (long long)ctx->n_sm * 7;
        ctx->e_per_block = std::max(1LL, (n_pairs + want - 1) / want);
        ctx->e_blocks = (int)((n_pairs + ctx->e_per_block - 1) / ctx->e_per_block);
        CREATE_CUDA(dalloc(&ctx->blk_prep, 4 * (size_t)n_it));
        CREATE_CUDA(dalloc(&ctx->blk_pair, 2 * (size_t)ctx->e_blocks));
        CREATE_CUDA(dalloc(&ctx->d_energy, 1));
    }

    // j records: mass constants for real stars; pad stars far away with zero mass
    {
        std::vector<JRec> h(np);
        for (size_t s = 0; s < np; ++s) {
            JRec r;
            r.x = r.y = r.z = kPadPos;
            const double gm = (s < (size_t)ctx->n_stars) ? G * masses[s + 1] : 0.0;
            r.gm = gm, r.g15 = 1.5 * gm, r.g1875 = 1.875 * gm;
            h[s] = r;
        }
        for (int s = 0; s < 2; ++s)
            CREATE_CUDA(cudaMemcpy(ctx->jrec[s], h.data(), np * sizeof(JRec), cudaMemcpyHostToDevice));
    }
#undef CREATE_CUDA
    *out = ctx;
    return PN_OK;
}

int pn_destroy(pn_ctx* c)
{
    if (!c) return PN_OK;
    int prev = -1;
    cudaGetDevice(&prev);
    if (prev != c->device) cudaSetDevice(c->device);
    cudaDeviceSynchronize();
    destroy_graphs(c);
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    for (cudaEvent_t e : c->tev)
        if (e) cudaEventDestroy(e);
    if (c->stream_ev) cudaEventDestroy(c->stream_ev);
    for (int s = 0; s < 2; ++s) cudaFree(c->jrec[s]), cudaFree(c->v[s]), cudaFree(c->bh[s]);
    cudaFree(c->x0), cudaFree(c->v0), cudaFree(c->sx), cudaFree(c->sv);
    cudaFree(c->part), cudaFree(c->bh_part), cudaFree(c->ticket), cudaFree(c->prm);
    cudaFree(c->io_pos), cudaFree(c->io_vel), cudaFree(c->io_acc);
    cudaFree(c->crec), cudaFree(c->cblk), cudaFree(c->csum), cudaFree(c->part6), cudaFree(c->blk_mom);
    cudaFree(c->small_part), cudaFree(c->small_bar), cudaFree(c->small_xv);
    if (c->small_host_flag) cudaFreeHost(c->small_host_flag);
    cudaFree(c->frec), cudaFree(c->fpair), cudaFree(c->erec), cudaFree(c->blk_prep), cudaFree(c->blk_pair), cudaFree(c->d_energy);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    cudaGetLastError();
    if (prev >= 0 && prev != c->device) cudaSetDevice(prev);
    delete c;
    return PN_OK;
}

int pn_set_stream(pn_ctx* c, void* s)
{
    if (int rc = check_ctx(c)) return rc;
    cudaStream_t ns = static_cast<cudaStream_t>(s);
    if (ns != c->stream) {
        // pn_accel and pn_step share the context's scratch (partial sums, the a_1 block partials and their ticket):
        // work already enqueued on the old stream must finish before anything enqueued on the new one touches it
        // If the runtime rejects the old stream (e.g. a handle it recognises as invalid), everything on the device is waited
        // for instead and the context moves to the new stream all the same.  This is no licence to destroy the old stream
        // first: the runtime does not validate a destroyed handle (cudaEventRecord on one crashed in the driver when tried);
        // pn.h asks callers to switch first and destroy afterwards.
        cudaError_t e = cudaEventRecord(c->stream_ev, c->stream);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(ns, c->stream_ev, 0);
        if (e != cudaSuccess) {
            cudaGetLastError();  // clear it: not this call's failure
            c->stream = ns;      // never stay bound to a dead handle
            PN_CUDA(c, cudaDeviceSynchronize());
        }
        c->stream = ns;
    }
    return PN_OK;
}

int pn_set_option(pn_ctx* c, int key, int value)
{
    if (int rc = check_ctx(c)) return rc;
    switch (key) {
        case PN_OPT_PAIR_PRECISION:
            if (value != PN_FP64 && value != PN_FP32_PAIR) return fail(c, PN_EINVAL, "pn_set_option: unknown pair precision %d", value);
            c->precision = value;
            return PN_OK;
        case PN_OPT_USE_GRAPH:
            if (value != 0 && value != 1) return fail(c, PN_EINVAL, "pn_set_option: PN_OPT_USE_GRAPH takes 0 or 1");
            c->use_graph = value;
            return PN_OK;
        case PN_OPT_TIME_PAIR:
            if (value < 0 || value > 2) return fail(c, PN_EINVAL, "pn_set_option: PN_OPT_TIME_PAIR takes 0, 1 or 2");
            if ((value == 2) != (c->time_pair == 2)) destroy_graphs(c);  // the timed graph has 8 or 2 event nodes
            c->time_pair = value;
            return PN_OK;
        case PN_OPT_PAIR_KERNEL:
            if (value != PN_PAIR_AUTO && value != PN_PAIR_TILED && value != PN_PAIR_SYMMETRIC)
                return fail(c, PN_EINVAL, "pn_set_option: unknown pair kernel %d", value);
            if (value != c->kernel_opt) destroy_graphs(c);
            c->kernel_opt = value;
            return PN_OK;
        case PN_OPT_CROSS_TERMS: {
            if (value != 0 && value != PN_CROSS_STAR && value != (PN_CROSS_STAR | PN_CROSS_BH))
                return fail(c, PN_EINVAL, "pn_set_option: PN_OPT_CROSS_TERMS takes 0, PN_CROSS_STAR or PN_CROSS_STAR | PN_CROSS_BH");
            if (value && !c->part6) {  // buffers of the cross path, on first use (part6 is allocated last)
                cudaFree(c->crec), cudaFree(c->cblk), cudaFree(c->csum);  // left over from a failed earlier attempt
                c->crec = nullptr, c->cblk = nullptr, c->csum = nullptr;
                const size_t np = c->np;
                const int n_it = c->np / (kCrossI * kNT), n_t = c->np / kCrossTJ;
                int s = std::max(1, std::min(std::min((c->n_sm * 16 + n_it - 1) / n_it, n_t), 64));
                c->c_tiles_per_split = (n_t + s - 1) / s;
                c->c_split = (n_t + c->c_tiles_per_split - 1) / c->c_tiles_per_split;
                c->c_T = c->np / kCrossSymU;
                c->c_m = (c->c_T + kCrossSymMaxGroups - 1) / kCrossSymMaxGroups;
                c->c_G = (c->c_T + c->c_m - 1) / c->c_m;
                PN_CUDA(c, cudaFuncSetAttribute(pair_cross_sym_kernel<kCrossSymMinB, true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kCrossSymSmemBytes<true>));
                PN_CUDA(c, cudaFuncSetAttribute(pair_cross_sym_kernel<kCrossSymMinB, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kCrossSymSmemBytes<true>));
                PN_CUDA(c, cudaFuncSetAttribute(pair_cross_sym_kernel<kCrossSymMinB, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kCrossSymSmemBytes<false>));
                PN_CUDA(c, cudaFuncSetAttribute(pair_cross_sym_kernel<kCrossSymMinB, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kCrossSymSmemBytes<false>));
                PN_CUDA(c, dalloc(&c->crec, np));
                PN_CUDA(c, dalloc(&c->cblk, (np / kNT) * kCrossSums));
                PN_CUDA(c, dalloc(&c->csum, kCrossSums));
                PN_CUDA(c, dalloc(&c->part6, (size_t)std::max(c->c_split, c->c_G) * 8 * np));
            }
            if (value && c->small_ok && c->n_stars <= kSmallCrossMaxStars && !c->small_xv) {  // small-system path with the Cross terms
                const size_t np = c->np;
                for (int mode = 0; mode < 2; ++mode)
                    for (int bhx = 0; bhx < 2; ++bhx)
                        PN_CUDA(c, cudaFuncSetAttribute(small_cross_fn(mode, c->small_IW, bhx != 0), cudaFuncAttributeMaxDynamicSharedMemorySize,
                                                        ((kSmallCrossMaxStars + 255) / 256 * 256) * kSmallCrossBytesPerStar));
                std::vector<XVRec> h(2 * np);  // pad entries are never written by the kernel: far away, at rest, for good
                for (XVRec& r : h) r.x = r.y = r.z = kPadPos, r.vx = r.vy = r.vz = 0.0;
                XVRec* xv = nullptr;
                PN_CUDA(c, dalloc(&xv, 2 * np));
                cudaError_t e = cudaMemcpy(xv, h.data(), h.size() * sizeof(XVRec), cudaMemcpyHostToDevice);
                if (e != cudaSuccess) {
                    cudaFree(xv);
                    PN_CUDA(c, e);
                }
                c->small_xv = xv;
            }
            c->cross = value;
            destroy_graphs(c);
            return PN_OK;
        }
        case PN_OPT_EQUAL_MASS:
            if (value != 0 && value != 1) return fail(c, PN_EINVAL, "pn_set_option: PN_OPT_EQUAL_MASS takes 0 or 1");
            c->eqm_opt = value;
            return PN_OK;
        case PN_OPT_J_SPLIT:
            if (value < 0) return fail(c, PN_EINVAL, "pn_set_option: PN_OPT_J_SPLIT must be >= 0");
            c->j_split_opt = value;
            choose_split(c);
            return PN_OK;
        default:
            return fail(c, PN_EINVAL, "pn_set_option: unknown key %d", key);
    }
}

int pn_set_state(pn_ctx* c, const double* pos, const double* vel)
{
    if (int rc = check_ctx(c)) return rc;
    if (int rc = small_poll(c)) return rc;  // a small-system launch that gave up since the last call
    if (!pos || !vel) return fail(c, PN_EINVAL, "pn_set_state: null pointer");
    const int grid = (c->n_stars + 255) / 256;
    pack_kernel<<<grid, 256, 0, c->stream>>>(pos, vel, c->jrec[0], c->v[0], c->x0, c->v0, c->bh[0], c->n_stars, c->np, 1);
    PN_CUDA(c, cudaGetLastError());
    c->n_launch += 1;
    c->have_state = true;
    return PN_OK;
}

int pn_get_state(pn_ctx* c, double* pos, double* vel)
{
    if (int rc = check_ctx(c)) return rc;
    if (int rc = small_poll(c)) return rc;  // a small-system launch that gave up since the last call
    if (!pos || !vel) return fail(c, PN_EINVAL, "pn_get_state: null pointer");
    if (!c->have_state) return fail(c, PN_ESTATE, "pn_get_state: no state set");
    const int grid = (c->n_stars + 255) / 256;
    unpack_kernel<<<grid, 256, 0, c->stream>>>(c->x0, c->v0, c->bh[0], pos, vel, c->n_stars, c->np);
    PN_CUDA(c, cudaGetLastError());
    c->n_launch += 1;
    return PN_OK;
}

int pn_set_state_host(pn_ctx* c, const double* pos, const double* vel)
{
    if (int rc = check_ctx(c)) return rc;
    if (!pos || !vel) return fail(c, PN_EINVAL, "pn_set_state_host: null pointer");
    const size_t bytes = 3 * (size_t)c->N * sizeof(double);
    PN_CUDA(c, cudaMemcpyAsync(c->io_pos, pos, bytes, cudaMemcpyHostToDevice, c->stream));
    PN_CUDA(c, cudaMemcpyAsync(c->io_vel, vel, bytes, cudaMemcpyHostToDevice, c->stream));
    if (int rc = pn_set_state(c, c->io_pos, c->io_vel)) return rc;
    PN_CUDA(c, cudaStreamSynchronize(c->stream));
    return PN_OK;
}

int pn_get_state_host(pn_ctx* c, double* pos, double* vel)
{
    if (int rc = check_ctx(c)) return rc;
    if (!pos || !vel) return fail(c, PN_EINVAL, "pn_get_state_host: null pointer");
    if (int rc = pn_get_state(c, c->io_pos, c->io_vel)) return rc;
    const size_t bytes = 3 * (size_t)c->N * sizeof(double);
    PN_CUDA(c, cudaMemcpyAsync(pos, c->io_pos, bytes, cudaMemcpyDeviceToHost, c->stream));
    PN_CUDA(c, cudaMemcpyAsync(vel, c->io_vel, bytes, cudaMemcpyDeviceToHost, c->stream));
    PN_CUDA(c, cudaStreamSynchronize(c->stream));
    if (int rc = small_check(c)) return rc;
    return PN_OK;
}

int pn_accel(pn_ctx* c, const double* pos, const double* vel, double* acc)
{
    if (int rc = check_ctx(c)) return rc;
    if (int rc = small_poll(c)) return rc;  // a small-system launch that gave up since the last call
    if (!pos || !vel || !acc) return fail(c, PN_EINVAL, "pn_accel: null pointer");
    const int grid_pack = (c->n_stars + 255) / 256;
    pack_kernel<<<grid_pack, 256, 0, c->stream>>>(pos, vel, c->jrec[1], c->v[1], nullptr, nullptr, c->bh[1], c->n_stars, c->np, 0);
    PN_CUDA(c, cudaGetLastError());
    if (use_small(c) || use_small_cross(c)) {
        const int rc = c->cross ? launch_small_cross(c, MODE_ACCEL, 0.0, 0, acc) : launch_small(c, MODE_ACCEL, 0.0, 0, acc);
        if (rc == PN_OK) {
            c->n_launch += 2;
            return PN_OK;
        }
        if (c->small_ok) return rc;  // a real error; otherwise: cooperative launch not possible right now, multi-kernel path
    }
    if (int rc = launch_pair(c, 1, c->stream, c->time_pair != 0)) return rc;
    const EpiArgs a = epi_args(c, 1, acc);
    if (c->cross & PN_CROSS_BH)
        epilogue_kernel<MODE_ACCEL, kEpiNTCross, 2><<<c->np / kEpiStars, kEpiNTCross, 0, c->stream>>>(a, 0);
    else if (c->cross)
        epilogue_kernel<MODE_ACCEL, kEpiNTCross, 1><<<c->np / kEpiStars, kEpiNTCross, 0, c->stream>>>(a, 0);
    else
        epilogue_kernel<MODE_ACCEL, kEpiNT, 0><<<c->np / kEpiStars, kEpiNT, 0, c->stream>>>(a, 0);
    PN_CUDA(c, cudaGetLastError());
    c->n_launch += 2 + kernels_per_eval(c);
    return PN_OK;
}

int pn_accel_host(pn_ctx* c, const double* pos, const double* vel, double* acc)
{
    if (int rc = check_ctx(c)) return rc;
    if (!pos || !vel || !acc) return fail(c, PN_EINVAL, "pn_accel_host: null pointer");
    const size_t bytes = 3 * (size_t)c->N * sizeof(double);
    PN_CUDA(c, cudaMemcpyAsync(c->io_pos, pos, bytes, cudaMemcpyHostToDevice, c->stream));
    PN_CUDA(c, cudaMemcpyAsync(c->io_vel, vel, bytes, cudaMemcpyHostToDevice, c->stream));
    if (int rc = pn_accel(c, c->io_pos, c->io_vel, c->io_acc)) return rc;
    PN_CUDA(c, cudaMemcpyAsync(acc, c->io_acc, bytes, cudaMemcpyDeviceToHost, c->stream));
    PN_CUDA(c, cudaStreamSynchronize(c->stream));
    if (int rc = small_check(c)) return rc;
    return PN_OK;
}

int pn_step(pn_ctx* c, double dt, int64_t nsteps)
{
    if (int rc = check_ctx(c)) return rc;
    if (int rc = small_poll(c)) return rc;  // a small-system launch that gave up since the last call
    if (!std::isfinite(dt)) return fail(c, PN_EINVAL, "pn_step: dt must be finite");
    if (nsteps < 0) return fail(c, PN_EINVAL, "pn_step: nsteps must be >= 0");
    if (!c->have_state) return fail(c, PN_ESTATE, "pn_step: no state set (call pn_set_state first)");
    if (nsteps == 0) return PN_OK;
    if (use_small(c) || use_small_cross(c)) {  // every stage of every step in one cooperative launch (PN_OPT_USE_GRAPH / PN_OPT_TIME_PAIR do not apply)
        const int rc = c->cross ? launch_small_cross(c, MODE_RK4, dt, nsteps, nullptr) : launch_small(c, MODE_RK4, dt, nsteps, nullptr);
        if (rc == PN_OK) {
            c->n_launch += 1;
            return PN_OK;
        }
        if (c->small_ok) return rc;  // a real error; otherwise: cooperative launch not possible right now, multi-kernel path
    }
    if (!(dt == c->dt_dev)) {
        StepParams p;
        p.dt = dt;
        PN_CUDA(c, cudaMemcpyAsync(c->prm, &p, sizeof p, cudaMemcpyHostToDevice, c->stream));
        PN_CUDA(c, cudaStreamSynchronize(c->stream));  // p lives on this stack frame
        c->dt_dev = dt;
    }
    const bool eager = !c->use_graph;
    if (eager) {
        for (int64_t s = 0; s < nsteps; ++s)
            if (int rc = enqueue_rk4_step(c, c->stream, c->time_pair != 0)) return rc;
        c->n_launch += 4 * (1 + kernels_per_eval(c)) * nsteps;
        return PN_OK;
    }
    if (c->graph_split != c->n_split || c->graph_precision != c->precision || c->graph_sym != (int)use_sym(c) ||
        c->graph_eqm != (int)use_eqm(c)) {
        destroy_graphs(c);
        c->graph_split = c->n_split, c->graph_precision = c->precision, c->graph_sym = (int)use_sym(c), c->graph_eqm = (int)use_eqm(c);
    }
    if (c->time_pair) {  // one-step graph whose event-record nodes get fresh events from the pool before every launch
        if (!c->graphT)
            if (int rc = build_timed_graph(c)) return rc;
        for (int64_t s = 0; s < nsteps; ++s) {
            const int ne = (c->time_pair == 2) ? 2 : 8;
            if (int rc = reserve_events(c, ne)) return rc;
            for (int q = 0; q < ne; ++q)
                PN_CUDA(c, cudaGraphExecEventRecordNodeSetEvent(c->graphT, c->tnode[q], c->ev[c->ev_used + q]));
            PN_CUDA(c, cudaGraphLaunch(c->graphT, c->stream));
            if (ne == 8) {  // four bracketed pair stages in one step: between two of them lies exactly one epilogue
                const size_t base = c->ev_used / 2;
                if (c->ev_chain.size() < base + 4) c->ev_chain.resize(base + 4, 0);
                c->ev_chain[base] = 0, c->ev_chain[base + 1] = c->ev_chain[base + 2] = c->ev_chain[base + 3] = 1;
            }
            c->ev_used += ne;
        }
        c->n_launch += 4 * (1 + kernels_per_eval(c)) * nsteps;
        return PN_OK;
    }
    int64_t left = nsteps;
    if (left >= kGraphBatch) {
        if (!c->graphB)
            if (int rc = build_graph(c, kGraphBatch, &c->graphB)) return rc;
        for (; left >= kGraphBatch; left -= kGraphBatch) PN_CUDA(c, cudaGraphLaunch(c->graphB, c->stream));
    }
    if (left > 0) {
        if (!c->graph1)
            if (int rc = build_graph(c, 1, &c->graph1)) return rc;
        for (; left > 0; --left) PN_CUDA(c, cudaGraphLaunch(c->graph1, c->stream));
    }
    c->n_launch += 4 * (1 + kernels_per_eval(c)) * nsteps;
    return PN_OK;
}

int pn_energy(pn_ctx* c, double* E)
{
    if (int rc = check_ctx(c)) return rc;
    if (!E) return fail(c, PN_EINVAL, "pn_energy: null pointer");
    if (!c->have_state) return fail(c, PN_ESTATE, "pn_energy: no state set");
    const int n_it = c->np / kNT;
    energy_prep_kernel<kNT><<<n_it, kNT, 0, c->stream>>>(c->jrec[0], c->v[0], c->bh[0], c->erec, c->blk_prep, c->n_stars, c->np,
                                                        c->GM, c->G, c->inv_c2);
    PN_CUDA(c, cudaGetLastError());
    energy_pair_kernel<kNT, kTJ><<<c->e_blocks, kNT, 0, c->stream>>>(c->erec, c->blk_pair, c->n_stars, c->np, c->e_per_block, c->eps2, c->G,
                                                              c->inv_c2);
    PN_CUDA(c, cudaGetLastError());
    energy_final_kernel<256><<<1, 256, 0, c->stream>>>(c->blk_prep, n_it, c->blk_pair, c->e_blocks, c->bh[0], c->M, c->GM,
                                                       c->G, c->inv_c2, c->d_energy);
    PN_CUDA(c, cudaGetLastError());
    c->n_launch += 3;
    PN_CUDA(c, cudaMemcpyAsync(E, c->d_energy, sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    PN_CUDA(c, cudaStreamSynchronize(c->stream));
    if (int rc = small_check(c)) return rc;
    return PN_OK;
}

int pn_momentum(pn_ctx* c, double* P)
{
    if (int rc = check_ctx(c)) return rc;
    if (!P) return fail(c, PN_EINVAL, "pn_momentum: null pointer");
    if (!c->have_state) return fail(c, PN_ESTATE, "pn_momentum: no state set");
    const int n_it = c->np / kNT;
    if (!c->blk_mom) {  // [n_it][6] + [e_blocks][6] + 3 results, on first use
        PN_CUDA(c, dalloc(&c->blk_mom, 6 * ((size_t)n_it + c->e_blocks) + 3));
    }
    double* blk_prep = c->blk_mom;
    double* blk_pair = c->blk_mom + 6 * (size_t)n_it;
    double* d_out = blk_pair + 6 * (size_t)c->e_blocks;
    energy_prep_kernel<kNT><<<n_it, kNT, 0, c->stream>>>(c->jrec[0], c->v[0], c->bh[0], c->erec, c->blk_prep, c->n_stars, c->np,
                                                        c->GM, c->G, c->inv_c2);  // builds the ERec stream
    momentum_prep_kernel<kNT><<<n_it, kNT, 0, c->stream>>>(c->jrec[0], c->v[0], c->bh[0], blk_prep, c->n_stars, c->np, c->GM, c->G,
                                                          c->inv_c2);
    momentum_pair_kernel<kNT, kTJ><<<c->e_blocks, kNT, 0, c->stream>>>(c->erec, blk_pair, c->n_stars, c->np, c->e_per_block, c->eps2, c->G);
    momentum_final_kernel<256><<<1, 256, 0, c->stream>>>(blk_prep, n_it, blk_pair, c->e_blocks, c->bh[0], c->M, c->inv_c2, d_out);
    PN_CUDA(c, cudaGetLastError());
    c->n_launch += 4;
    PN_CUDA(c, cudaMemcpyAsync(P, d_out, 3 * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    PN_CUDA(c, cudaStreamSynchronize(c->stream));
    if (int rc = small_check(c)) return rc;
    return PN_OK;
}

int pn_get_launch_count(pn_ctx* c, int64_t* n)
{
    if (int rc = check_ctx(c)) return rc;
    if (!n) return fail(c, PN_EINVAL, "pn_get_launch_count: null pointer");
    *n = c->n_launch;
    return PN_OK;
}

int pn_get_pair_time(pn_ctx* c, double* ms_total, int64_t* n_launches, int reset)
{
    if (int rc = check_ctx(c)) return rc;
    if (!ms_total || !n_launches) return fail(c, PN_EINVAL, "pn_get_pair_time: null pointer");
    if (int rc = fold_events(c)) return rc;
    *ms_total = c->pair_ms_folded;
    *n_launches = c->pair_n_folded;
    if (reset) c->pair_ms_folded = 0, c->pair_n_folded = 0;
    return PN_OK;
}

int pn_get_epilogue_time(pn_ctx* c, double* ms_total, int64_t* n_intervals, int reset)
{
    if (int rc = check_ctx(c)) return rc;
    if (!ms_total || !n_intervals) return fail(c, PN_EINVAL, "pn_get_epilogue_time: null pointer");
    if (int rc = fold_events(c)) return rc;
    *ms_total = c->epi_ms_folded;
    *n_intervals = c->epi_n_folded;
    if (reset) c->epi_ms_folded = 0, c->epi_n_folded = 0;
    return PN_OK;
}

int pn_get_pair_config(pn_ctx* c, int32_t* cfg)
{
    if (int rc = check_ctx(c)) return rc;
    if (!cfg) return fail(c, PN_EINVAL, "pn_get_pair_config: null pointer");
    if (use_small(c)) {
        cfg[0] = kSmallNT, cfg[1] = c->small_IW, cfg[2] = 32, cfg[3] = 1, cfg[4] = c->small_blocks, cfg[5] = c->np, cfg[6] = 15, cfg[7] = 7;
        return PN_OK;
    }
    if (use_small_cross(c)) {  // 12 / 13: the small-system path with the Cross terms (ordered pairs: 54 / 59 instructions)
        const bool bhx = (c->cross & PN_CROSS_BH) != 0;
        cfg[0] = kSmallNT, cfg[1] = c->small_IW, cfg[2] = 32, cfg[3] = 1, cfg[4] = c->small_blocks, cfg[5] = c->np;
        cfg[6] = bhx ? 59 : 54, cfg[7] = bhx ? 13 : 12;
        return PN_OK;
    }
    if (c->cross && cross_sym(c)) {
        cfg[0] = 32, cfg[1] = kCrossSymI, cfg[2] = kCrossSymU, cfg[3] = c->c_G;
        cfg[4] = c->c_G * (c->c_G + 1) / 2, cfg[5] = c->np;
        const bool bhx = (c->cross & PN_CROSS_BH) != 0, ceqm = c->equal_mass && c->eqm_opt;
        cfg[6] = bhx ? (ceqm ? 40 : 42) : (ceqm ? 37 : 38), cfg[7] = (bhx ? 9 : 8) + (ceqm ? 2 : 0);  // 10 / 11: equal-mass form
        return PN_OK;
    }
    if (c->cross) {
        cfg[0] = kNT, cfg[1] = kCrossI, cfg[2] = kCrossTJ, cfg[3] = c->c_split;
        cfg[4] = (c->np / (kCrossI * kNT)) * c->c_split, cfg[5] = c->np;
        cfg[6] = (c->cross & PN_CROSS_BH) ? 59 : 54, cfg[7] = (c->cross & PN_CROSS_BH) ? 6 : 5;
        return PN_OK;
    }
    if (use_sym(c)) {
        cfg[0] = (c->precision == PN_FP32_PAIR && c->sym_U == 128) ? 32 : 32 * c->sym_W, cfg[1] = c->sym_I, cfg[2] = c->sym_U, cfg[3] = c->sym_G;
        cfg[4] = c->sym_G * (c->sym_G + 1) / 2, cfg[5] = c->np;
        cfg[6] = (c->precision == PN_FP32_PAIR) ? (use_eqm(c) ? 10 : 11) : (use_eqm(c) ? 9 : 10);
        cfg[7] = (c->precision == PN_FP32_PAIR) ? 3 : (use_eqm(c) ? 4 : 2);
        return PN_OK;
    }
    cfg[0] = kNT, cfg[1] = c->ipt, cfg[2] = kTJ, cfg[3] = c->n_split;
    cfg[4] = c->n_itiles * c->n_split, cfg[5] = c->np, cfg[6] = (c->precision == PN_FP32_PAIR) ? 18 : 15, cfg[7] = c->precision;
    return PN_OK;
}

}  // extern "C"
