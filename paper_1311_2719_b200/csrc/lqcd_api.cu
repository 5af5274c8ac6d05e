// lqcd_api.cu -- the C-ABI of include/lqcd.h: context, workspace carving, kernel launches and
// the host side of the conjugate gradient (the paper's congrad).
//
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -shared ... (build.py)
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "../../include/lqcd.h"
#include "cg_kernels.cuh"
#include "cg_persistent.cuh"
#include "stag_dslash.cuh"
#include "stag_dslash_f32x2.cuh"
#include "wilson_dslash.cuh"

using namespace lqcd;

namespace {

constexpr int kStagBlock = 128;
#ifndef LQCD_WILSON_BLOCK
#define LQCD_WILSON_BLOCK 128
#endif
constexpr int kWilsonBlock = LQCD_WILSON_BLOCK;
#ifndef LQCD_F32X2_BLOCK
#define LQCD_F32X2_BLOCK 128
#endif
constexpr int kF32x2Block = LQCD_F32X2_BLOCK;  // threads per block of the two-sites-per-thread fp32 kernels
constexpr int kVecBlock = 256;
constexpr int kReorderTile = 64;
constexpr size_t kAlign = 256;

typedef StagArgs<cplx> StagArgsD;
typedef StagArgs<cplxf> StagArgsF;

size_t align_up(size_t n) { return (n + kAlign - 1) / kAlign * kAlign; }

}  // namespace

struct lqcd_ctx {
    int L[4];
    int fermion;
    Geom g;
    size_t nvec;  // complex numbers per CG vector
    // workspace layout (byte offsets)
    size_t off_gauge, off_r, off_p, off_t, off_sc, off_ticket, off_partials, off_hist, off_stage;
    size_t off_stage_b, off_stage_x;  // inside the staging area, after the canonical gauge copy
    size_t off_gauge_f, off_xf, off_rf, off_pf, off_tf;  // fp32 copies for the mixed-precision solver (staggered)
    size_t ws_needed;
    size_t max_blocks;
    // bound workspace
    char* ws;
    cudaStream_t stream;
    bool gauge_loaded;
    bool gauge_f_ready;  // the fp32 link copy matches the loaded fp64 one
    // options
    int cg_mode;
    int check_every;
    int recon;  // 18 or 12 stored reals per link
    int congrad_precision;  // 64 or 32: which solver lqcd_congrad_host runs
    int f32_pairs;          // fp32 kernels of the mixed solver: two sites per thread with 128-bit loads
    int stag_block;         // 0 auto (stag_block_for), or 32 / 64 / 128 threads per block of the fp64 staggered kernels
    int persistent;         // -1 auto, 0 never, 1 always: the CG loop as one cooperative kernel (cg_persistent.cuh)
    bool cg_mode_set;       // LQCD_OPT_CG_MODE was set by the caller: the automatic choice above then respects LQCD_CG_SYNC
    int last_path;          // LQCD_PATH_* of the last lqcd_cg_solve-type call (lqcd_last_cg_path)
    int persist_chunk;      // LQCD_OPT_PERSISTENT_CHUNK: iterations per launch of the cooperative kernel
    int nsm;                // multiprocessors of the device the workspace was bound on (148 on B200 until then)
    bool links_fit_l2;  // the stored link field is at most a third of the L2 (set by lqcd_load_gauge)
    bool wilson_eo;  // set while lqcd_wilson_solve_eo runs: the CG works on Mhat^+ Mhat, even half of the vectors
    // host side
    CgScalars* h_sc;  // pinned, 2 slots
    cudaEvent_t ev[2];
    bool host_ready;
    long long launches;
    int last_iters;
    char err[320];

    cplx* gauge() const { return (cplx*)(ws + off_gauge); }
    cplx* r() const { return (cplx*)(ws + off_r); }
    cplx* p() const { return (cplx*)(ws + off_p); }
    cplx* t() const { return (cplx*)(ws + off_t); }
    cplxf* gauge_f() const { return (cplxf*)(ws + off_gauge_f); }
    cplxf* xf() const { return (cplxf*)(ws + off_xf); }
    cplxf* rf() const { return (cplxf*)(ws + off_rf); }
    cplxf* pf() const { return (cplxf*)(ws + off_pf); }
    cplxf* tf() const { return (cplxf*)(ws + off_tf); }
    CgScalars* sc() const { return (CgScalars*)(ws + off_sc); }
    double* hist() const { return (double*)(ws + off_hist); }
    ReduceScratch rs() const
    {
        ReduceScratch s;
        s.partials = (double*)(ws + off_partials);
        s.ticket = (unsigned int*)(ws + off_ticket);
        return s;
    }
};

namespace {

int fail(lqcd_ctx* c, int code, const char* fmt, ...)
{
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof c->err, fmt, ap);
        va_end(ap);
    }
    return code;
}

#define LQCD_CUDA(call)                                                                                  \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess)                                                                           \
            return fail(ctx, LQCD_ECUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, \
                        __LINE__);                                                                       \
    } while (0)

#define LQCD_LAUNCH_CHECK()                                                                              \
    do {                                                                                                 \
        ctx->launches++;                                                                                 \
        cudaError_t e_ = cudaGetLastError();                                                             \
        if (e_ != cudaSuccess)                                                                           \
            return fail(ctx, LQCD_ECUDA, "kernel launch failed: %s (%s:%d)", cudaGetErrorString(e_),     \
                        __FILE__, __LINE__);                                                             \
    } while (0)

int check_ready(lqcd_ctx* ctx, bool need_gauge)
{
    if (!ctx) return LQCD_EARG;
    if (!ctx->ws) return fail(ctx, LQCD_ESTATE, "workspace not set (call lqcd_set_workspace)");
    if (need_gauge && !ctx->gauge_loaded) return fail(ctx, LQCD_ESTATE, "gauge field not loaded (call lqcd_load_gauge)");
    return LQCD_OK;
}

unsigned int blocks_for(size_t n, int block) { return (unsigned int)((n + block - 1) / block); }

VecLayout vec_layout(const lqcd_ctx* ctx)
{
    VecLayout l;
    if (ctx->wilson_eo) {
        l.n = 12 * (size_t)ctx->g.Vh;
        l.inner = (size_t)ctx->g.Vh;
        l.stride = (size_t)ctx->g.V;
    } else {
        l.n = l.inner = l.stride = ctx->nvec;
    }
    return l;
}

unsigned int vec_grid(const lqcd_ctx* ctx)
{
    size_t b = (vec_layout(ctx).n + kVecBlock - 1) / kVecBlock;
    size_t cap = (size_t)ctx->nsm * 8;   // eight 256-thread blocks per multiprocessor: one wave of the vector kernels
    if (cap > 4096) cap = 4096;          // the partial-sum area has V/32 + 4096 slots (lqcd_create)
    if (b > cap) b = cap;
    if (b < 1) b = 1;
    return (unsigned int)b;
}

// ---------------------------------------------------------------- staggered launches
StagArgsD stag_args(const lqcd_ctx* ctx, int parity, const cplx* in, cplx* out)
{
    StagArgsD a;
    memset(&a, 0, sizeof a);
    a.g = ctx->g;
    a.parity = parity;
    a.gauge = ctx->gauge();
    a.in = in;
    a.out = out;
    a.sc = ctx->sc();
    a.rs = ctx->rs();
    a.hist = ctx->hist();
    return a;
}

// Threads per block of the fp64 staggered kernels.  128 on lattices that fill the machine; small lattices
// are latency-bound and gain from more, smaller blocks (B200, us per CG iteration / plain Dslash at
// 128, 64, 32 threads: 16^4 30.4 / 10.3, 27.2 / 7.3, 25.9 / 6.3; 4^4 20.7 / 6.2, 18.7 / 4.6, 17.1 / 4.2;
// 32^4 234.9, 242.6, 267.3 per iteration: profiles/r01_bench.md).
int stag_block_for(const lqcd_ctx* ctx)
{
    if (ctx->stag_block) return ctx->stag_block;  // LQCD_OPT_STAG_BLOCK
    const long long blocks128 = ((long long)ctx->g.Vh + 127) / 128;
    if (blocks128 < 2 * ctx->nsm) return 32;
    if (blocks128 < 8 * ctx->nsm) return 64;
    return 128;
}

template <int EPI, int BLOCK>
int launch_stag_block(lqcd_ctx* ctx, const StagArgsD& a)
{
    const unsigned int grid = blocks_for(ctx->g.Vh, BLOCK);
    if (ctx->recon == 12)
        stag_dslash_kernel<EPI, BLOCK, 12, cplx><<<grid, BLOCK, 0, ctx->stream>>>(a);
    else
        stag_dslash_kernel<EPI, BLOCK, 18, cplx><<<grid, BLOCK, 0, ctx->stream>>>(a);
    LQCD_LAUNCH_CHECK();
    return LQCD_OK;
}

template <int EPI>
int launch_stag(lqcd_ctx* ctx, const StagArgsD& a)
{
    const int block = stag_block_for(ctx);
    if (block == 32) return launch_stag_block<EPI, 32>(ctx, a);
    if (block == 64) return launch_stag_block<EPI, 64>(ctx, a);
    return launch_stag_block<EPI, kStagBlock>(ctx, a);
}

// fp32 instantiations: only the two kernels of the inner iteration of the mixed-precision solver
StagArgsF stag_args_f(const lqcd_ctx* ctx, int parity, const cplxf* in, cplxf* out)
{
    StagArgsF a;
    memset(&a, 0, sizeof a);
    a.g = ctx->g;
    a.parity = parity;
    a.gauge = ctx->gauge_f();
    a.in = in;
    a.out = out;
    a.sc = ctx->sc();
    a.rs = ctx->rs();
    a.hist = ctx->hist();
    return a;
}

template <int EPI>
int launch_stag_f(lqcd_ctx* ctx, const StagArgsF& a)
{
    if (ctx->f32_pairs && ctx->g.Lh % 2 == 0) {  // two sites per thread, 128-bit loads (stag_dslash_f32x2.cuh)
        const unsigned int grid2 = blocks_for((size_t)ctx->g.Vh / 2, kF32x2Block);
        if (ctx->recon == 12)
            stag_dslash_f32x2_kernel<EPI, kF32x2Block, 12><<<grid2, kF32x2Block, 0, ctx->stream>>>(a);
        else
            stag_dslash_f32x2_kernel<EPI, kF32x2Block, 18><<<grid2, kF32x2Block, 0, ctx->stream>>>(a);
        LQCD_LAUNCH_CHECK();
        return LQCD_OK;
    }
    const unsigned int grid = blocks_for(ctx->g.Vh, kStagBlock);
    if (ctx->recon == 12)
        stag_dslash_kernel<EPI, kStagBlock, 12, cplxf><<<grid, kStagBlock, 0, ctx->stream>>>(a);
    else
        stag_dslash_kernel<EPI, kStagBlock, 18, cplxf><<<grid, kStagBlock, 0, ctx->stream>>>(a);
    LQCD_LAUNCH_CHECK();
    return LQCD_OK;
}

// ---------------------------------------------------------------- Wilson launches
WilsonArgs wilson_args(const lqcd_ctx* ctx, int parity, const cplx* in, cplx* out, double kappa)
{
    WilsonArgs a;
    memset(&a, 0, sizeof a);
    a.g = ctx->g;
    a.parity = parity;
    a.gauge = ctx->gauge();
    a.in = in;
    a.out = out;
    a.kappa = kappa;
    a.sc = ctx->sc();
    a.rs = ctx->rs();
    a.hist = ctx->hist();
    return a;
}

template <int EPI, bool DAGGER, int LINKS>
int launch_wilson_policy(lqcd_ctx* ctx, const WilsonArgs& a)
{
    // one-parity kernels: one block per tile of Vh; full-lattice kernels: tiles of the two parities alternate
    const unsigned int tiles = blocks_for(ctx->g.Vh, kWilsonBlock);
    const unsigned int grid = wilson_one_parity(EPI) ? tiles : 2 * tiles;
    if (ctx->recon == 12)
        wilson_dslash_kernel<EPI, DAGGER, kWilsonBlock, 12, LINKS><<<grid, kWilsonBlock, 0, ctx->stream>>>(a);
    else
        wilson_dslash_kernel<EPI, DAGGER, kWilsonBlock, 18, LINKS><<<grid, kWilsonBlock, 0, ctx->stream>>>(a);
    LQCD_LAUNCH_CHECK();
    return LQCD_OK;
}

template <int EPI, bool DAGGER>
int launch_wilson(lqcd_ctx* ctx, const WilsonArgs& a)
{
    // Link cache policy (device_common.cuh): a full-lattice kernel uses every link twice within a short time
    // (wilson_thread_site) -> through L2; a one-parity kernel uses every link once per launch -> streamed,
    // unless the whole field stays in L2 from launch to launch (ctx->links_fit_l2).
    if (!wilson_one_parity(EPI) || ctx->links_fit_l2) return launch_wilson_policy<EPI, DAGGER, LP_L2>(ctx, a);
    return launch_wilson_policy<EPI, DAGGER, LP_STREAM>(ctx, a);
}

// ---------------------------------------------------------------- operator pieces
// t = "first half" of A applied to v (D_oe v  or  M v), optionally with the norm/alpha epilogue.
int op_first(lqcd_ctx* ctx, double param, const cplx* v, bool with_norm)
{
    if (ctx->fermion == LQCD_STAGGERED) {
        StagArgsD a = stag_args(ctx, LQCD_ODD, v, ctx->t());
        a.m2 = param * param;
        return with_norm ? launch_stag<SE_NORM>(ctx, a) : launch_stag<SE_PLAIN>(ctx, a);
    }
    WilsonArgs a = wilson_args(ctx, 0, v, ctx->t(), param);
    return with_norm ? launch_wilson<WE_M_NORM, false>(ctx, a) : launch_wilson<WE_M, false>(ctx, a);
}

// Even-odd preconditioned Wilson: t_e = Mhat v_e (DAGGER = false) or Mhat^+ v_e
// (true), Mhat = 1 - kappa^2 D_eo D_oe, through the odd half of the scratch vector t.  `dst` receives
// the even half of the result; with_norm adds tt = |result|^2 and alpha = rr/tt.
template <bool DAGGER>
int eo_mhat(lqcd_ctx* ctx, double kappa, const cplx* v, cplx* dst, bool with_norm)
{
    int rc = launch_wilson<WE_PLAIN, DAGGER>(ctx, wilson_args(ctx, LQCD_ODD, v, ctx->t(), 0.0));
    if (rc) return rc;
    WilsonArgs a = wilson_args(ctx, LQCD_EVEN, ctx->t(), dst, -kappa * kappa);
    a.p = v;
    return with_norm ? launch_wilson<WE_EO_XPAY_NORM, DAGGER>(ctx, a) : launch_wilson<WE_EO_XPAY, DAGGER>(ctx, a);
}

int eo_iteration_kernels(lqcd_ctx* ctx, double kappa, cplx* x)
{
    int rc = eo_mhat<false>(ctx, kappa, ctx->p(), ctx->t(), true);  // t_e = Mhat p, alpha = rr/|t_e|^2
    if (rc) return rc;
    // w_o = D^+_oe t_e into the odd half of t; Ap = t_e - kappa^2 D^+_eo w_o fused with the x / r updates
    rc = launch_wilson<WE_PLAIN, true>(ctx, wilson_args(ctx, LQCD_ODD, ctx->t(), ctx->t(), 0.0));
    if (rc) return rc;
    WilsonArgs a = wilson_args(ctx, LQCD_EVEN, ctx->t(), nullptr, -kappa * kappa);
    a.p = ctx->t();
    a.b = ctx->p();
    a.x = x;
    a.r = ctx->r();
    return launch_wilson<WE_EO_CGUPDATE, true>(ctx, a);
}

int cg_iteration_kernels(lqcd_ctx* ctx, double param, cplx* x)
{
    if (ctx->wilson_eo) return eo_iteration_kernels(ctx, param, x);
    int rc = op_first(ctx, param, ctx->p(), true);  // S1 + S2
    if (rc) return rc;
    if (ctx->fermion == LQCD_STAGGERED) {           // S3
        StagArgsD a = stag_args(ctx, LQCD_EVEN, ctx->t(), nullptr);
        a.m2 = param * param;
        a.p = ctx->p();
        a.x = x;
        a.r = ctx->r();
        return launch_stag<SE_CGUPDATE>(ctx, a);
    }
    WilsonArgs a = wilson_args(ctx, 0, ctx->t(), nullptr, param);
    a.p = ctx->p();
    a.x = x;
    a.r = ctx->r();
    return launch_wilson<WE_CGUPDATE, true>(ctx, a);
}

int cg_pupdate(lqcd_ctx* ctx, cplx* x)  // S5 (Wilson: preceded by the x += alpha p of S3, see cg_xpupdate_kernel)
{
    if (ctx->fermion == LQCD_WILSON)
        cg_xpupdate_kernel<kVecBlock><<<vec_grid(ctx), kVecBlock, 0, ctx->stream>>>(ctx->r(), ctx->p(), x, vec_layout(ctx), ctx->sc(),
                                                                                 ctx->rs());
    else
        cg_pupdate_kernel<kVecBlock, cplx><<<vec_grid(ctx), kVecBlock, 0, ctx->stream>>>(ctx->r(), ctx->p(), vec_layout(ctx), ctx->sc(),
                                                                                  ctx->rs());
    LQCD_LAUNCH_CHECK();
    return LQCD_OK;
}

int enqueue_batch(lqcd_ctx* ctx, double param, cplx* x, int batch)
{
    for (int k = 0; k < batch; ++k) {
        int rc = cg_iteration_kernels(ctx, param, x);
        if (rc) return rc;
        rc = cg_pupdate(ctx, x);
        if (rc) return rc;
    }
    return LQCD_OK;
}

struct GraphHolder {
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    ~GraphHolder()
    {
        if (exec) cudaGraphExecDestroy(exec);
        if (graph) cudaGraphDestroy(graph);
    }
};

int read_scalars(lqcd_ctx* ctx, int slot)
{
    LQCD_CUDA(cudaMemcpyAsync(&ctx->h_sc[slot], ctx->sc(), sizeof(CgScalars), cudaMemcpyDeviceToHost, ctx->stream));
    LQCD_CUDA(cudaEventRecord(ctx->ev[slot], ctx->stream));
    return LQCD_OK;
}

int ensure_host(lqcd_ctx* ctx)
{
    if (ctx->host_ready) return LQCD_OK;
    LQCD_CUDA(cudaHostAlloc((void**)&ctx->h_sc, 2 * sizeof(CgScalars), cudaHostAllocDefault));
    LQCD_CUDA(cudaEventCreateWithFlags(&ctx->ev[0], cudaEventDisableTiming));
    LQCD_CUDA(cudaEventCreateWithFlags(&ctx->ev[1], cudaEventDisableTiming));
    ctx->host_ready = true;
    return LQCD_OK;
}

// ---------------------------------------------------------------- the loop as one cooperative kernel
// Used for the fp64 staggered CG where an iteration is bounded by its kernel boundaries: the links fit the
// L2 (ctx->links_fit_l2), so the three kernels of an iteration take a few microseconds each.
bool use_persistent(const lqcd_ctx* ctx)
{
    if (ctx->fermion != LQCD_STAGGERED || ctx->wilson_eo) return false;
    if (ctx->persistent >= 0) return ctx->persistent == 1;
    // automatic: never against an explicit request for the paper's loop with its host-side exit test
    if (ctx->cg_mode_set && ctx->cg_mode == LQCD_CG_SYNC) return false;
    return ctx->links_fit_l2;
}

// Iterations one launch of the cooperative kernel may run.  Its grid barrier counts arrivals in 32 bits from
// zero at launch: three barriers per iteration and at most one block per multiprocessor, so 2^20 iterations
// stay far below 2^32 arrivals (3 * 2^20 * 1024 blocks = 2^31.6); longer solves continue in a fresh launch
// (the scalars round-trip through CgScalars, the iterates do not change).
constexpr int kPersistChunk = 1 << 20;

template <int RECON>
int launch_persistent_recon(lqcd_ctx* ctx, double mass, cplx* x, int niter)
{
    PersistArgs a;
    memset(&a, 0, sizeof a);
    a.g = ctx->g;
    a.gauge = ctx->gauge();
    a.p = ctx->p();
    a.t = ctx->t();
    a.x = x;
    a.r = ctx->r();
    a.m2 = mass * mass;
    a.sc = ctx->sc();
    a.hist = ctx->hist();
    a.partials = ctx->rs().partials;
    a.bar = ctx->rs().ticket + 16;  // the 256-byte ticket area: word 0 = reduction ticket, word 16 = grid barrier
    a.nvb = (int)blocks_for(ctx->g.Vh, 32);
    a.vgrid = (int)vec_grid(ctx);
    a.niter = niter;
    if ((size_t)(2 * a.nvb + a.vgrid) > ctx->max_blocks) return fail(ctx, LQCD_ENOMEM, "partial-sum area too small for the persistent kernel");
    int dev = 0, nsm = 0, per_sm = 0, coop = 0;
    LQCD_CUDA(cudaGetDevice(&dev));
    LQCD_CUDA(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    if (!coop) return fail(ctx, LQCD_ECUDA, "device does not support cooperative launches");
    LQCD_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    LQCD_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, stag_cg_persistent_kernel<RECON>, kPersistBlock, 0));
    if (per_sm < 1) return fail(ctx, LQCD_ECUDA, "persistent CG kernel does not fit an SM");
    // one block per SM at most, eight virtual blocks (warps) per block at a time
    long long grid = (a.nvb + kPersistBlock / 32 - 1) / (kPersistBlock / 32);
    if (grid > nsm) grid = nsm;
    LQCD_CUDA(cudaMemsetAsync(a.bar, 0, sizeof(unsigned int), ctx->stream));
    void* params[] = { (void*)&a };
    LQCD_CUDA(cudaLaunchCooperativeKernel((const void*)stag_cg_persistent_kernel<RECON>, dim3((unsigned int)grid), dim3(kPersistBlock),
                                          params, 0, ctx->stream));
    ctx->launches++;
    return LQCD_OK;
}

int launch_persistent(lqcd_ctx* ctx, double mass, cplx* x, int niter)
{
    return ctx->recon == 12 ? launch_persistent_recon<12>(ctx, mass, x, niter) : launch_persistent_recon<18>(ctx, mass, x, niter);
}

// Init (S6) and the iteration loop (S1-S5) of the conjugate gradient on A x = b.  On return the
// stream is idle and ctx->h_sc[0] holds the final scalars (iter, rr_new, thresh, bb).
int cg_run(lqcd_ctx* ctx, double mass_or_kappa, double tol, int maxiter, const cplx* b, cplx* x)
{
    int rc;
    // S6: p = r = b, x = 0, rr = bb = pp = |b|^2
    cg_init_kernel<kVecBlock><<<vec_grid(ctx), kVecBlock, 0, ctx->stream>>>(b, x, ctx->r(), ctx->p(), vec_layout(ctx), ctx->sc(),
                                                                           ctx->rs(), ctx->hist(), tol, maxiter);
    LQCD_LAUNCH_CHECK();

    CgScalars* h = ctx->h_sc;
    ctx->last_path = LQCD_PATH_HOST_LOOP;
    if (use_persistent(ctx)) {
        // one launch runs the loop to the exit rule (or maxiter); the scalars come back once
        ctx->last_path = LQCD_PATH_PERSISTENT;
        int left = maxiter > 0 ? maxiter : 0;
        do {
            const int chunk = left < ctx->persist_chunk ? left : ctx->persist_chunk;
            if (chunk > 0) {
                rc = launch_persistent(ctx, mass_or_kappa, x, chunk);
                if (rc) return rc;
            }
            left -= chunk;
            rc = read_scalars(ctx, 0);
            if (rc) return rc;
            LQCD_CUDA(cudaEventSynchronize(ctx->ev[0]));
        } while (left > 0 && !h[0].done);
    } else if (ctx->cg_mode == LQCD_CG_SYNC) {
        // The paper's loop: one scalar comes back per iteration, the exit test runs on the host
        // (PAPER.md:75-76, :91-93, :100).
        rc = read_scalars(ctx, 0);
        if (rc) return rc;
        LQCD_CUDA(cudaEventSynchronize(ctx->ev[0]));
        while (!h[0].done) {
            rc = cg_iteration_kernels(ctx, mass_or_kappa, x);
            if (rc) return rc;
            rc = read_scalars(ctx, 0);
            if (rc) return rc;
            LQCD_CUDA(cudaEventSynchronize(ctx->ev[0]));
            if (h[0].done && ctx->fermion != LQCD_WILSON) break;
            rc = cg_pupdate(ctx, x);  // Wilson: also after the exit rule has fired -- the kernel holds the last x += alpha p
            if (rc) return rc;
            if (h[0].done) break;
        }
    } else {
        // Same kernels, same order; batches of `check_every` iterations are enqueued while the
        // previous batch's scalars are still on their way to the host.  Once the device sets
        // `done`, every later kernel returns at once, so x, r and the iteration count are exactly
        // those of the synchronous loop.
        const int batch = ctx->check_every;
        // LQCD_CG_GRAPH: the batch is captured once and replayed with one graph launch instead of
        // 3*batch kernel launches (launch-bound small lattices).  The legacy default stream cannot
        // be captured; there the batch is enqueued kernel by kernel as in LQCD_CG_ASYNC.
        GraphHolder gh;
        if (ctx->cg_mode == LQCD_CG_GRAPH && ctx->stream != nullptr && maxiter > 0) {
            const long long counted = ctx->launches;
            LQCD_CUDA(cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeThreadLocal));
            rc = enqueue_batch(ctx, mass_or_kappa, x, batch);
            cudaError_t ce = cudaStreamEndCapture(ctx->stream, &gh.graph);
            if (rc) return rc;
            LQCD_CUDA(ce);
            LQCD_CUDA(cudaGraphInstantiate(&gh.exec, gh.graph, 0));
            ctx->launches = counted;  // capturing launched nothing
        }
        int slot = 0;
        bool pending[2] = { false, false };
        bool finished = false;
        long long enqueued = 0;
        while (!finished) {
            if (enqueued < (long long)maxiter) {
                if (gh.exec) {
                    LQCD_CUDA(cudaGraphLaunch(gh.exec, ctx->stream));
                    ctx->launches += (ctx->wilson_eo ? 5LL : 3LL) * batch;
                } else {
                    rc = enqueue_batch(ctx, mass_or_kappa, x, batch);
                    if (rc) return rc;
                }
                enqueued += batch;
            }
            rc = read_scalars(ctx, slot);
            if (rc) return rc;
            pending[slot] = true;
            const int other = slot ^ 1;
            if (pending[other]) {
                LQCD_CUDA(cudaEventSynchronize(ctx->ev[other]));
                pending[other] = false;
                if (h[other].done) finished = true;
            }
            slot = other;
        }
        // drain: the newest snapshot has the final values
        LQCD_CUDA(cudaStreamSynchronize(ctx->stream));
        rc = read_scalars(ctx, 0);
        if (rc) return rc;
        LQCD_CUDA(cudaEventSynchronize(ctx->ev[0]));
    }

    ctx->last_iters = h[0].iter;
    return LQCD_OK;
}

// ---------------------------------------------------------------- mixed precision
int mixed_iteration_kernels(lqcd_ctx* ctx, double mass)  // S1 + S2, S3 on the fp32 copies
{
    StagArgsF a = stag_args_f(ctx, LQCD_ODD, ctx->pf(), ctx->tf());
    a.m2 = mass * mass;
    int rc = launch_stag_f<SE_NORM>(ctx, a);
    if (rc) return rc;
    a = stag_args_f(ctx, LQCD_EVEN, ctx->tf(), nullptr);
    a.m2 = mass * mass;
    a.p = ctx->pf();
    a.x = ctx->xf();
    a.r = ctx->rf();
    return launch_stag_f<SE_CGUPDATE_MIXED>(ctx, a);
}

int mixed_pupdate(lqcd_ctx* ctx)  // S5 on the fp32 copies
{
    if (ctx->f32_pairs && ctx->nvec % 2 == 0) {
        cg_pupdate_f32x2_kernel<kVecBlock><<<vec_grid(ctx), kVecBlock, 0, ctx->stream>>>(ctx->rf(), ctx->pf(), ctx->nvec, ctx->sc(),
                                                                                       ctx->rs());
        LQCD_LAUNCH_CHECK();
        return LQCD_OK;
    }
    cg_pupdate_kernel<kVecBlock, cplxf><<<vec_grid(ctx), kVecBlock, 0, ctx->stream>>>(ctx->rf(), ctx->pf(), vec_layout(ctx),
                                                                                      ctx->sc(), ctx->rs());
    LQCD_LAUNCH_CHECK();
    return LQCD_OK;
}

int mixed_batch(lqcd_ctx* ctx, double mass, int batch)
{
    for (int k = 0; k < batch; ++k) {
        int rc = mixed_iteration_kernels(ctx, mass);
        if (rc) return rc;
        rc = mixed_pupdate(ctx);
        if (rc) return rc;
    }
    return LQCD_OK;
}

// The reliable update, all fp64: x += xs, xs = 0; r = b - A x; rs = fl32(r); <r,r>, beta, exit test;
// then the p-update the paused iteration was waiting for.  Enqueued by the host only after a
// snapshot of the scalars showed `pause` with every earlier update completed.
int mixed_reliable_update(lqcd_ctx* ctx, double mass, const cplx* b, cplx* x)
{
    mixed_accumulate_kernel<kVecBlock><<<vec_grid(ctx), kVecBlock, 0, ctx->stream>>>(x, ctx->xf(), ctx->nvec, ctx->sc(), 1);
    LQCD_LAUNCH_CHECK();
    int rc = launch_stag<SE_PLAIN>(ctx, stag_args(ctx, LQCD_ODD, x, ctx->t()));
    if (rc) return rc;
    StagArgsD a = stag_args(ctx, LQCD_EVEN, ctx->t(), nullptr);
    a.m2 = mass * mass;
    a.p = x;
    a.b = b;
    a.rf = ctx->rf();
    rc = launch_stag<SE_RELIABLE>(ctx, a);
    if (rc) return rc;
    return mixed_pupdate(ctx);
}

int cg_run_mixed(lqcd_ctx* ctx, double mass, double tol, double delta, int maxiter, const cplx* b, cplx* x)
{
    int rc;
    ctx->last_path = LQCD_PATH_HOST_LOOP;
    if (!ctx->gauge_f_ready) {
        const size_t n = (size_t)ctx->g.V * 4 * (size_t)(ctx->recon / 2);
        gauge_narrow_kernel<<<ctx->nsm * 8, 256, 0, ctx->stream>>>(ctx->gauge(), ctx->gauge_f(), n);
        LQCD_LAUNCH_CHECK();
        ctx->gauge_f_ready = true;
    }
    cg_init_mixed_kernel<kVecBlock><<<vec_grid(ctx), kVecBlock, 0, ctx->stream>>>(
        b, x, ctx->xf(), ctx->rf(), ctx->pf(), ctx->nvec, ctx->sc(), ctx->rs(), ctx->hist(), tol, delta, maxiter);
    LQCD_LAUNCH_CHECK();

    CgScalars* h = ctx->h_sc;
    const bool sync = ctx->cg_mode == LQCD_CG_SYNC;
    const int batch = sync ? 1 : ctx->check_every;
    GraphHolder gh;
    if (ctx->cg_mode == LQCD_CG_GRAPH && ctx->stream != nullptr && maxiter > 0) {
        const long long counted = ctx->launches;
        LQCD_CUDA(cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeThreadLocal));
        rc = mixed_batch(ctx, mass, batch);
        cudaError_t ce = cudaStreamEndCapture(ctx->stream, &gh.graph);
        if (rc) return rc;
        LQCD_CUDA(ce);
        LQCD_CUDA(cudaGraphInstantiate(&gh.exec, gh.graph, 0));
        ctx->launches = counted;
    }
    // As cg_run, with one more device-side state: `pause`.  Iterations enqueued after the device
    // paused are no-ops, so the iterates do not depend on the batch size or on when the host notices.
    int slot = 0, updates_enqueued = 0;
    bool pending[2] = { false, false };
    bool finished = maxiter <= 0;
    while (!finished) {
        if (gh.exec) {
            LQCD_CUDA(cudaGraphLaunch(gh.exec, ctx->stream));
            ctx->launches += 3LL * batch;
        } else {
            rc = mixed_batch(ctx, mass, batch);
            if (rc) return rc;
        }
        rc = read_scalars(ctx, slot);
        if (rc) return rc;
        pending[slot] = true;
        const int look = sync ? slot : slot ^ 1;
        if (pending[look]) {
            LQCD_CUDA(cudaEventSynchronize(ctx->ev[look]));
            pending[look] = false;
            if (h[look].done) {
                finished = true;
            } else if (h[look].pause && h[look].nupd == updates_enqueued) {
                rc = mixed_reliable_update(ctx, mass, b, x);
                if (rc) return rc;
                ++updates_enqueued;
            }
        }
        slot ^= 1;
    }
    // whatever the fp32 iteration still holds goes into x (nothing after a converged exit: xs = 0)
    mixed_accumulate_kernel<kVecBlock><<<vec_grid(ctx), kVecBlock, 0, ctx->stream>>>(x, ctx->xf(), ctx->nvec, ctx->sc(), 0);
    LQCD_LAUNCH_CHECK();
    LQCD_CUDA(cudaStreamSynchronize(ctx->stream));
    rc = read_scalars(ctx, 0);
    if (rc) return rc;
    LQCD_CUDA(cudaEventSynchronize(ctx->ev[0]));
    ctx->last_iters = h[0].iter;
    return LQCD_OK;
}

}  // namespace

// =========================================================================== C-ABI
extern "C" {

int lqcd_create(lqcd_ctx** out, int L0, int L1, int L2, int L3, int fermion_type)
{
    if (!out) return LQCD_EARG;
    *out = nullptr;
    if (fermion_type != LQCD_STAGGERED && fermion_type != LQCD_WILSON) return LQCD_EARG;
    const int L[4] = { L0, L1, L2, L3 };
    long long V = 1;
    for (int mu = 0; mu < 4; ++mu) {
        if (L[mu] < 2 || (L[mu] & 1)) return LQCD_EDIM;
        V *= L[mu];
        if (V > (1LL << 30)) return LQCD_EDIM;  // int32 tables and 32-bit half-lattice indices
    }
    lqcd_ctx* c = (lqcd_ctx*)calloc(1, sizeof(lqcd_ctx));
    if (!c) return LQCD_ENOMEM;
    memcpy(c->L, L, sizeof L);
    c->fermion = fermion_type;
    c->g.Lh = L0 / 2;
    c->g.L1 = L1;
    c->g.L2 = L2;
    c->g.L3 = L3;
    c->g.s1 = c->g.Lh;
    c->g.s2 = c->g.Lh * L1;
    c->g.s3 = c->g.Lh * L1 * L2;
    c->g.V = V;
    c->g.Vh = (int)(V / 2);
    c->nvec = fermion_type == LQCD_STAGGERED ? 3 * (size_t)(V / 2) : 12 * (size_t)V;
    c->max_blocks = (size_t)V / 32 + 4096;
    c->cg_mode = LQCD_CG_ASYNC;
    c->check_every = 4;
    c->recon = 18;
    c->congrad_precision = 64;
    c->f32_pairs = 1;
    c->persistent = -1;
    c->cg_mode_set = false;
    c->persist_chunk = kPersistChunk;
    c->last_path = LQCD_PATH_NONE;
    c->nsm = 148;

    size_t off = 0;
    const size_t vec_bytes = align_up(c->nvec * sizeof(cplx));
    c->off_gauge = off;      off += align_up((size_t)V * 36 * sizeof(cplx));
    c->off_r = off;          off += vec_bytes;
    c->off_p = off;          off += vec_bytes;
    c->off_t = off;          off += vec_bytes;
    c->off_sc = off;         off += align_up(sizeof(CgScalars));
    c->off_ticket = off;     off += kAlign;
    c->off_partials = off;   off += align_up(c->max_blocks * sizeof(double));
    c->off_hist = off;       off += align_up((size_t)kHistCap * sizeof(double));
    c->off_stage = off;
    const size_t stage_u = align_up((size_t)V * 36 * sizeof(cplx));
    c->off_stage_b = off + stage_u;
    c->off_stage_x = c->off_stage_b + vec_bytes;
    size_t stage = stage_u + 2 * vec_bytes;
    const size_t tables = align_up((size_t)V * 9 * sizeof(int32_t));
    if (tables > stage) stage = tables;
    off += stage;
    if (fermion_type == LQCD_STAGGERED) {
        const size_t vecf_bytes = align_up(c->nvec * sizeof(cplxf));
        c->off_gauge_f = off;  off += align_up((size_t)V * 36 * sizeof(cplxf));
        c->off_xf = off;       off += vecf_bytes;
        c->off_rf = off;       off += vecf_bytes;
        c->off_pf = off;       off += vecf_bytes;
        c->off_tf = off;       off += vecf_bytes;
    }
    c->ws_needed = off;
    *out = c;
    return LQCD_OK;
}

int lqcd_destroy(lqcd_ctx* ctx)
{
    if (!ctx) return LQCD_EARG;
    if (ctx->host_ready) {
        cudaFreeHost(ctx->h_sc);
        cudaEventDestroy(ctx->ev[0]);
        cudaEventDestroy(ctx->ev[1]);
    }
    free(ctx);
    return LQCD_OK;
}

size_t lqcd_workspace_bytes(const lqcd_ctx* ctx) { return ctx ? ctx->ws_needed : 0; }

int lqcd_set_workspace(lqcd_ctx* ctx, void* workspace_dev, size_t bytes, void* cuda_stream)
{
    if (!ctx) return LQCD_EARG;
    if (!workspace_dev) return fail(ctx, LQCD_EARG, "workspace pointer is null");
    if (((uintptr_t)workspace_dev) % kAlign) return fail(ctx, LQCD_EARG, "workspace must be 256-byte aligned");
    if (bytes < ctx->ws_needed)
        return fail(ctx, LQCD_ENOMEM, "workspace too small: %zu bytes given, %zu needed", bytes, ctx->ws_needed);
    int ndev = 0;
    LQCD_CUDA(cudaGetDeviceCount(&ndev));
    if (ndev < 1) return fail(ctx, LQCD_ECUDA, "no CUDA device");
    int rc = ensure_host(ctx);
    if (rc) return rc;
    int dev = 0, nsm = 0;
    LQCD_CUDA(cudaGetDevice(&dev));
    LQCD_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
    if (nsm > 0) ctx->nsm = nsm;
    ctx->ws = (char*)workspace_dev;
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->gauge_loaded = false;
    ctx->gauge_f_ready = false;
    LQCD_CUDA(cudaMemsetAsync(ctx->ws + ctx->off_sc, 0, align_up(sizeof(CgScalars)) + kAlign, ctx->stream));
    return LQCD_OK;
}

int lqcd_set_option(lqcd_ctx* ctx, int option, int value)
{
    if (!ctx) return LQCD_EARG;
    if (option == LQCD_OPT_CG_MODE) {
        if (value < LQCD_CG_SYNC || value > LQCD_CG_GRAPH) return fail(ctx, LQCD_EARG, "bad CG mode %d", value);
        ctx->cg_mode = value;
        ctx->cg_mode_set = true;
        return LQCD_OK;
    }
    if (option == LQCD_OPT_CG_CHECK_EVERY) {
        if (value < 1 || value > 1024) return fail(ctx, LQCD_EARG, "check_every must be in 1..1024");
        ctx->check_every = value;
        return LQCD_OK;
    }
    if (option == LQCD_OPT_RECONSTRUCT) {
        if (value != 18 && value != 12) return fail(ctx, LQCD_EARG, "reconstruct must be 18 or 12");
        if (value != ctx->recon) ctx->gauge_loaded = ctx->gauge_f_ready = false;  // the internal copies have the other layout
        ctx->recon = value;
        return LQCD_OK;
    }
    if (option == LQCD_OPT_CONGRAD_PRECISION) {
        if (value != 64 && !(value == 32 && ctx->fermion == LQCD_STAGGERED))
            return fail(ctx, LQCD_EARG, "congrad precision must be 64, or 32 on a staggered context");
        ctx->congrad_precision = value;
        return LQCD_OK;
    }
    if (option == LQCD_OPT_F32_PAIRS) {
        if (value != 0 && value != 1) return fail(ctx, LQCD_EARG, "f32_pairs must be 0 or 1");
        ctx->f32_pairs = value;
        return LQCD_OK;
    }
    if (option == LQCD_OPT_STAG_BLOCK) {
        if (value != 0 && value != 32 && value != 64 && value != 128) return fail(ctx, LQCD_EARG, "stag_block must be 0 (auto), 32, 64 or 128");
        ctx->stag_block = value;
        return LQCD_OK;
    }
    if (option == LQCD_OPT_PERSISTENT_CHUNK) {
        if (value < 1 || value > kPersistChunk) return fail(ctx, LQCD_EARG, "persistent chunk must be in 1..%d", kPersistChunk);
        ctx->persist_chunk = value;
        return LQCD_OK;
    }
    if (option == LQCD_OPT_PERSISTENT) {
        if (value < -1 || value > 1) return fail(ctx, LQCD_EARG, "persistent must be -1 (auto), 0 or 1");
        ctx->persistent = value;
        return LQCD_OK;
    }
    return fail(ctx, LQCD_EARG, "unknown option %d", option);
}

int lqcd_load_gauge(lqcd_ctx* ctx, const double* u_dev)
{
    int rc = check_ready(ctx, false);
    if (rc) return rc;
    if (!u_dev) return fail(ctx, LQCD_EARG, "u_dev is null");
    const size_t V = (size_t)ctx->g.V;
    const unsigned int grid = blocks_for(V, kReorderTile);
    if (ctx->recon == 12)
        gauge_reorder_kernel<256, kReorderTile, 12, cplx><<<grid, 256, 0, ctx->stream>>>((const cplx*)u_dev, ctx->gauge(),
                                                                                         (size_t)ctx->g.Vh);
    else
        gauge_reorder_kernel<256, kReorderTile, 18, cplx><<<grid, 256, 0, ctx->stream>>>((const cplx*)u_dev, ctx->gauge(),
                                                                                         (size_t)ctx->g.Vh);
    LQCD_LAUNCH_CHECK();
    ctx->gauge_f_ready = false;
    ctx->gauge_loaded = true;
    // B200: 126 MB of L2 in two partitions; data read by all SMs is cached in both, so about half of it is
    // usable for a field every SM reads (75 MB of links at 16^3 x 32 were measured NOT to stay resident).
    int dev = 0, l2 = 0;
    LQCD_CUDA(cudaGetDevice(&dev));
    LQCD_CUDA(cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev));
    ctx->links_fit_l2 = V * 4 * (size_t)(ctx->recon / 2) * sizeof(cplx) <= (size_t)l2 / 3;
    return LQCD_OK;
}

int lqcd_get_tables(lqcd_ctx* ctx, int32_t* iup_host, int32_t* idn_host, int32_t* lex2eo_host)
{
    int rc = check_ready(ctx, false);
    if (rc) return rc;
    const size_t V = (size_t)ctx->g.V;
    int32_t* d = (int32_t*)(ctx->ws + ctx->off_stage);
    tables_kernel<<<blocks_for(V, 256), 256, 0, ctx->stream>>>(ctx->g, d, d + 4 * V, d + 8 * V);
    LQCD_LAUNCH_CHECK();
    if (iup_host) LQCD_CUDA(cudaMemcpyAsync(iup_host, d, 4 * V * sizeof(int32_t), cudaMemcpyDeviceToHost, ctx->stream));
    if (idn_host)
        LQCD_CUDA(cudaMemcpyAsync(idn_host, d + 4 * V, 4 * V * sizeof(int32_t), cudaMemcpyDeviceToHost, ctx->stream));
    if (lex2eo_host)
        LQCD_CUDA(cudaMemcpyAsync(lex2eo_host, d + 8 * V, V * sizeof(int32_t), cudaMemcpyDeviceToHost, ctx->stream));
    LQCD_CUDA(cudaStreamSynchronize(ctx->stream));
    return LQCD_OK;
}

int lqcd_dslash(lqcd_ctx* ctx, int out_parity, const double* in_dev, double* out_dev)
{
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    if (!in_dev || !out_dev) return fail(ctx, LQCD_EARG, "null vector pointer");
    if (in_dev == out_dev) return fail(ctx, LQCD_EARG, "in and out must not alias");
    if (out_parity != LQCD_EVEN && out_parity != LQCD_ODD) return fail(ctx, LQCD_EARG, "bad parity %d", out_parity);
    if (ctx->fermion == LQCD_STAGGERED) return launch_stag<SE_PLAIN>(ctx, stag_args(ctx, out_parity, (const cplx*)in_dev, (cplx*)out_dev));
    return launch_wilson<WE_PLAIN, false>(ctx, wilson_args(ctx, out_parity, (const cplx*)in_dev, (cplx*)out_dev, 0.0));
}

int lqcd_dslash_sweep(lqcd_ctx* ctx, int first_out_parity, double* a_dev, double* b_dev, int reps)
{
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    if (!a_dev || !b_dev || a_dev == b_dev) return fail(ctx, LQCD_EARG, "null or aliased vector pointer");
    if (first_out_parity != LQCD_EVEN && first_out_parity != LQCD_ODD) return fail(ctx, LQCD_EARG, "bad parity %d", first_out_parity);
    if (reps < 0) return fail(ctx, LQCD_EARG, "reps must be >= 0");
    for (int k = 0; k < reps; ++k) {
        rc = lqcd_dslash(ctx, (first_out_parity + k) & 1, (k & 1) ? b_dev : a_dev, (k & 1) ? a_dev : b_dev);
        if (rc) return rc;
    }
    return LQCD_OK;
}

int lqcd_apply_MdagM(lqcd_ctx* ctx, double mass_or_kappa, const double* in_dev, double* out_dev)
{
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    if (!in_dev || !out_dev) return fail(ctx, LQCD_EARG, "null vector pointer");
    if (in_dev == out_dev) return fail(ctx, LQCD_EARG, "in and out must not alias");
    rc = op_first(ctx, mass_or_kappa, (const cplx*)in_dev, false);
    if (rc) return rc;
    if (ctx->fermion == LQCD_STAGGERED) {
        StagArgsD a = stag_args(ctx, LQCD_EVEN, ctx->t(), (cplx*)out_dev);
        a.m2 = mass_or_kappa * mass_or_kappa;
        a.p = (const cplx*)in_dev;
        return launch_stag<SE_MDAGM>(ctx, a);
    }
    return launch_wilson<WE_M, true>(ctx, wilson_args(ctx, 0, ctx->t(), (cplx*)out_dev, mass_or_kappa));
}


int lqcd_cg_solve(lqcd_ctx* ctx, double mass_or_kappa, double tol, int maxiter, const double* b_dev, double* x_dev,
                  int* iters, double* true_residual)
{
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    if (!b_dev || !x_dev || !iters || !true_residual) return fail(ctx, LQCD_EARG, "null pointer argument");
    if (b_dev == x_dev) return fail(ctx, LQCD_EARG, "b and x must not alias");
    if (!(tol >= 0.0) || maxiter < 0) return fail(ctx, LQCD_EARG, "tol must be >= 0 and maxiter >= 0");
    const cplx* b = (const cplx*)b_dev;
    cplx* x = (cplx*)x_dev;
    CgScalars* h = ctx->h_sc;
    rc = cg_run(ctx, mass_or_kappa, tol, maxiter, b, x);
    if (rc) return rc;

    // S7: true residual |b - A x| / |b| with a fresh application of A
    rc = op_first(ctx, mass_or_kappa, x, false);
    if (rc) return rc;
    if (ctx->fermion == LQCD_STAGGERED) {
        StagArgsD a = stag_args(ctx, LQCD_EVEN, ctx->t(), nullptr);
        a.m2 = mass_or_kappa * mass_or_kappa;
        a.p = x;
        a.b = b;
        rc = launch_stag<SE_RESIDUAL>(ctx, a);
    } else {
        WilsonArgs a = wilson_args(ctx, 0, ctx->t(), nullptr, mass_or_kappa);
        a.b = b;
        rc = launch_wilson<WE_RESIDUAL, true>(ctx, a);
    }
    if (rc) return rc;
    rc = read_scalars(ctx, 0);
    if (rc) return rc;
    LQCD_CUDA(cudaEventSynchronize(ctx->ev[0]));

    *iters = h[0].iter;
    *true_residual = h[0].bb > 0.0 ? sqrt(h[0].res2 / h[0].bb) : 0.0;
    const bool converged = h[0].rr_new <= h[0].thresh;
    return converged ? LQCD_OK : LQCD_MAXITER;
}

int lqcd_cg_solve_mixed(lqcd_ctx* ctx, double mass, double tol, int maxiter, double delta, const double* b_dev,
                        double* x_dev, int* iters, int* reliable_updates, double* true_residual)
{
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    if (ctx->fermion != LQCD_STAGGERED) return fail(ctx, LQCD_EARG, "lqcd_cg_solve_mixed needs a staggered context");
    if (!b_dev || !x_dev || !iters || !reliable_updates || !true_residual) return fail(ctx, LQCD_EARG, "null pointer argument");
    if (b_dev == x_dev) return fail(ctx, LQCD_EARG, "b and x must not alias");
    if (!(tol >= 0.0) || maxiter < 0) return fail(ctx, LQCD_EARG, "tol must be >= 0 and maxiter >= 0");
    if (!(delta > 0.0 && delta < 1.0)) return fail(ctx, LQCD_EARG, "delta must be in (0,1)");
    const cplx* b = (const cplx*)b_dev;
    cplx* x = (cplx*)x_dev;
    CgScalars* h = ctx->h_sc;
    rc = cg_run_mixed(ctx, mass, tol, delta, maxiter, b, x);
    if (rc) return rc;
    const int it = h[0].iter, nupd = h[0].nupd;
    const bool converged = h[0].bb == 0.0 || (h[0].rr_new <= h[0].thresh && !h[0].pause && (nupd > 0));
    // true residual |b - A x| / |b| with a fresh fp64 A (S7)
    rc = op_first(ctx, mass, x, false);
    if (rc) return rc;
    StagArgsD a = stag_args(ctx, LQCD_EVEN, ctx->t(), nullptr);
    a.m2 = mass * mass;
    a.p = x;
    a.b = b;
    rc = launch_stag<SE_RESIDUAL>(ctx, a);
    if (rc) return rc;
    rc = read_scalars(ctx, 0);
    if (rc) return rc;
    LQCD_CUDA(cudaEventSynchronize(ctx->ev[0]));
    *iters = it;
    *reliable_updates = nupd;
    *true_residual = h[0].bb > 0.0 ? sqrt(h[0].res2 / h[0].bb) : 0.0;
    return converged ? LQCD_OK : LQCD_MAXITER;
}

int lqcd_stag_solve_full(lqcd_ctx* ctx, double mass, double tol, int maxiter, const double* b_even_dev,
                         const double* b_odd_dev, double* x_even_dev, double* x_odd_dev, int* iters,
                         double* true_residual)
{
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    if (ctx->fermion != LQCD_STAGGERED) return fail(ctx, LQCD_EARG, "lqcd_stag_solve_full needs a staggered context");
    if (!b_even_dev || !b_odd_dev || !x_even_dev || !x_odd_dev || !iters || !true_residual)
        return fail(ctx, LQCD_EARG, "null pointer argument");
    if (x_even_dev == x_odd_dev || b_even_dev == x_even_dev || b_even_dev == x_odd_dev || b_odd_dev == x_even_dev ||
        b_odd_dev == x_odd_dev)
        return fail(ctx, LQCD_EARG, "b and x vectors must not alias");
    if (!(tol >= 0.0) || maxiter < 0) return fail(ctx, LQCD_EARG, "tol must be >= 0 and maxiter >= 0");
    if (mass == 0.0 || !(mass == mass)) return fail(ctx, LQCD_EARG, "mass must be non-zero (x_o = (b_o - D_oe x_e)/m)");
    const cplx *be = (const cplx*)b_even_dev, *bo = (const cplx*)b_odd_dev;
    cplx *xe = (cplx*)x_even_dev, *xo = (cplx*)x_odd_dev;
    cplx* bp = (cplx*)(ctx->ws + ctx->off_stage_b);  // b' lives in the staging area (idle during device-pointer calls)
    CgScalars* h = ctx->h_sc;

    // 1. source preparation  b' = m b_e - D_eo b_o
    StagArgsD a = stag_args(ctx, LQCD_EVEN, bo, bp);
    a.m2 = mass;
    a.p = be;
    rc = launch_stag<SE_PREP>(ctx, a);
    if (rc) return rc;
    // 2. CG on (m^2 - D_eo D_oe) x_e = b'
    rc = cg_run(ctx, mass, tol, maxiter, bp, xe);
    if (rc) return rc;
    const int cg_iters = h[0].iter;
    const bool converged = h[0].rr_new <= h[0].thresh;
    // 3. reconstruction  x_o = (b_o - D_oe x_e)/m
    a = stag_args(ctx, LQCD_ODD, xe, xo);
    a.m2 = mass;
    a.p = bo;
    rc = launch_stag<SE_RECON>(ctx, a);
    if (rc) return rc;
    // 4. |b - M x|^2 and |b|^2 over both parities with M = m + D applied afresh
    a = stag_args(ctx, LQCD_EVEN, xo, nullptr);
    a.m2 = mass;
    a.p = xe;
    a.b = be;
    a.flag = 0;
    rc = launch_stag<SE_RESIDUAL_M>(ctx, a);
    if (rc) return rc;
    a = stag_args(ctx, LQCD_ODD, xe, nullptr);
    a.m2 = mass;
    a.p = xo;
    a.b = bo;
    a.flag = 1;
    rc = launch_stag<SE_RESIDUAL_M>(ctx, a);
    if (rc) return rc;
    rc = read_scalars(ctx, 0);
    if (rc) return rc;
    LQCD_CUDA(cudaEventSynchronize(ctx->ev[0]));
    *iters = cg_iters;
    *true_residual = h[0].aux > 0.0 ? sqrt(h[0].res2 / h[0].aux) : 0.0;
    return converged ? LQCD_OK : LQCD_MAXITER;
}

int lqcd_wilson_eo_MdagM(lqcd_ctx* ctx, double kappa, const double* in_dev, double* out_dev)
{
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    if (ctx->fermion != LQCD_WILSON) return fail(ctx, LQCD_EARG, "lqcd_wilson_eo_MdagM needs a Wilson context");
    if (!in_dev || !out_dev) return fail(ctx, LQCD_EARG, "null vector pointer");
    if (in_dev == out_dev) return fail(ctx, LQCD_EARG, "in and out must not alias");
    rc = eo_mhat<false>(ctx, kappa, (const cplx*)in_dev, ctx->t(), false);  // t_e = Mhat in_e
    if (rc) return rc;
    // out_e = Mhat^+ t_e: w_o = D^+_oe t_e into the odd half of t, then the diagonal term from t_e
    rc = launch_wilson<WE_PLAIN, true>(ctx, wilson_args(ctx, LQCD_ODD, ctx->t(), ctx->t(), 0.0));
    if (rc) return rc;
    WilsonArgs a = wilson_args(ctx, LQCD_EVEN, ctx->t(), (cplx*)out_dev, -kappa * kappa);
    a.p = ctx->t();
    return launch_wilson<WE_EO_XPAY, true>(ctx, a);
}

int lqcd_wilson_solve_eo(lqcd_ctx* ctx, double kappa, double tol, int maxiter, const double* b_dev, double* x_dev,
                         int* iters, double* true_residual)
{
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    if (ctx->fermion != LQCD_WILSON) return fail(ctx, LQCD_EARG, "lqcd_wilson_solve_eo needs a Wilson context");
    if (!b_dev || !x_dev || !iters || !true_residual) return fail(ctx, LQCD_EARG, "null pointer argument");
    if (b_dev == x_dev) return fail(ctx, LQCD_EARG, "b and x must not alias");
    if (!(tol >= 0.0) || maxiter < 0) return fail(ctx, LQCD_EARG, "tol must be >= 0 and maxiter >= 0");
    const cplx* b = (const cplx*)b_dev;
    cplx* x = (cplx*)x_dev;
    cplx* bh = (cplx*)(ctx->ws + ctx->off_stage_b);  // staging vectors are idle during device-pointer calls
    cplx* c = (cplx*)(ctx->ws + ctx->off_stage_x);
    CgScalars* h = ctx->h_sc;

    // 1. bh_e = b_e + kappa D_eo b_o
    WilsonArgs a = wilson_args(ctx, LQCD_EVEN, b, bh, kappa);
    a.p = b;
    rc = launch_wilson<WE_EO_XPAY, false>(ctx, a);
    if (rc) return rc;
    // 2. c_e = Mhat^+ bh_e
    rc = eo_mhat<true>(ctx, kappa, bh, c, false);
    if (rc) return rc;
    // 3. CG on Mhat^+ Mhat x_e = c_e over the even half of the full-lattice arrays
    ctx->wilson_eo = true;
    rc = cg_run(ctx, kappa, tol, maxiter, c, x);
    ctx->wilson_eo = false;
    if (rc) return rc;
    const int cg_iters = h[0].iter;
    const bool converged = h[0].rr_new <= h[0].thresh;
    // 4. x_o = b_o + kappa D_oe x_e
    a = wilson_args(ctx, LQCD_ODD, x, x, kappa);
    a.p = b;
    rc = launch_wilson<WE_EO_XPAY, false>(ctx, a);
    if (rc) return rc;
    // 5. |b - M x|^2 and |b|^2, M = 1 - kappa D_W, one parity at a time
    for (int parity = 0; parity < 2; ++parity) {
        a = wilson_args(ctx, parity, x, nullptr, -kappa);
        a.p = x;
        a.b = b;
        a.flag = parity;
        rc = launch_wilson<WE_EO_RESIDUAL, false>(ctx, a);
        if (rc) return rc;
    }
    rc = read_scalars(ctx, 0);
    if (rc) return rc;
    LQCD_CUDA(cudaEventSynchronize(ctx->ev[0]));
    *iters = cg_iters;
    *true_residual = h[0].aux > 0.0 ? sqrt(h[0].res2 / h[0].aux) : 0.0;
    return converged ? LQCD_OK : LQCD_MAXITER;
}

int lqcd_congrad_host(lqcd_ctx* ctx, const double* u_host, double mass_or_kappa, double tol, int maxiter,
                      const double* b_host, double* x_host, int* iters, double* true_residual)
{
    int rc = check_ready(ctx, false);
    if (rc) return rc;
    if (!u_host || !b_host || !x_host) return fail(ctx, LQCD_EARG, "null host pointer");
    const size_t V = (size_t)ctx->g.V;
    cplx* su = (cplx*)(ctx->ws + ctx->off_stage);
    cplx* sb = (cplx*)(ctx->ws + ctx->off_stage_b);
    cplx* sx = (cplx*)(ctx->ws + ctx->off_stage_x);
    // copyin(u, r)
    LQCD_CUDA(cudaMemcpyAsync(su, u_host, V * 36 * sizeof(cplx), cudaMemcpyHostToDevice, ctx->stream));
    LQCD_CUDA(cudaMemcpyAsync(sb, b_host, ctx->nvec * sizeof(cplx), cudaMemcpyHostToDevice, ctx->stream));
    rc = lqcd_load_gauge(ctx, (const double*)su);
    if (rc) return rc;
    int nupd = 0;
    const int status = ctx->congrad_precision == 32
                           ? lqcd_cg_solve_mixed(ctx, mass_or_kappa, tol, maxiter, 0.1, (const double*)sb, (double*)sx, iters,
                                                 &nupd, true_residual)
                           : lqcd_cg_solve(ctx, mass_or_kappa, tol, maxiter, (const double*)sb, (double*)sx, iters,
                                           true_residual);
    if (status < 0) return status;
    // copyout(x)
    LQCD_CUDA(cudaMemcpyAsync(x_host, sx, ctx->nvec * sizeof(cplx), cudaMemcpyDeviceToHost, ctx->stream));
    LQCD_CUDA(cudaStreamSynchronize(ctx->stream));
    return status;
}

int lqcd_dslash_host(lqcd_ctx* ctx, int out_parity, const double* in_host, double* out_host)
{
    int rc = check_ready(ctx, true);
    if (rc) return rc;
    if (!in_host || !out_host) return fail(ctx, LQCD_EARG, "null host pointer");
    cplx* sb = (cplx*)(ctx->ws + ctx->off_stage_b);
    cplx* sx = (cplx*)(ctx->ws + ctx->off_stage_x);
    const size_t bytes = ctx->nvec * sizeof(cplx);
    LQCD_CUDA(cudaMemcpyAsync(sb, in_host, bytes, cudaMemcpyHostToDevice, ctx->stream));
    if (ctx->fermion == LQCD_WILSON) LQCD_CUDA(cudaMemsetAsync(sx, 0, bytes, ctx->stream));
    rc = lqcd_dslash(ctx, out_parity, (const double*)sb, (double*)sx);
    if (rc) return rc;
    LQCD_CUDA(cudaMemcpyAsync(out_host, sx, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    LQCD_CUDA(cudaStreamSynchronize(ctx->stream));
    return LQCD_OK;
}

int lqcd_cg_history(lqcd_ctx* ctx, double* rr_host, int capacity)
{
    int rc = check_ready(ctx, false);
    if (rc) return rc;
    if (!rr_host || capacity < 0) return fail(ctx, LQCD_EARG, "bad history buffer");
    int n = ctx->last_iters + 1;
    if (n > kHistCap) n = kHistCap;
    if (n > capacity) n = capacity;
    LQCD_CUDA(cudaMemcpyAsync(rr_host, ctx->hist(), (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    LQCD_CUDA(cudaStreamSynchronize(ctx->stream));
    return n;
}

long long lqcd_kernel_launches(const lqcd_ctx* ctx) { return ctx ? ctx->launches : 0; }

int lqcd_last_cg_path(const lqcd_ctx* ctx) { return ctx ? ctx->last_path : LQCD_EARG; }

const char* lqcd_last_error(const lqcd_ctx* ctx) { return ctx ? ctx->err : "null context"; }

}  // extern "C"
