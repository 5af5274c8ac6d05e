// lqcd_slab.cu -- the C-ABI of include/lqcd_slab.h: the staggered conjugate gradient of the paper
// on a lattice cut into time-slabs, one per GPU.
// Every entry point is a thin wrapper around a *_group function that drives n slabs phase by phase;
// the one-rank-per-process calls are the n = 1 case of the same code.
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "../../include/lqcd_slab.h"
#include "slab_kernels.cuh"
#include "stag_dslash.cuh"

using namespace lqcd;

namespace {
constexpr int kStagBlock = 128;
constexpr int kVecBlock = 256;
constexpr int kReorderTile = 64;
constexpr size_t kAlign = 256;
typedef StagArgs<cplx> StagArgsD;
size_t align_up(size_t n) { return (n + kAlign - 1) / kAlign * kAlign; }
unsigned int blocks_for(size_t n, int block) { return (unsigned int)((n + block - 1) / block); }
}  // namespace

struct lqcd_slab {
    int L[4];
    int rank, nranks, T, t0, sh;
    Geom g;       // the LOCAL lattice L0 x L1 x L2 x T
    size_t nvec;  // complex numbers per local vector
    // workspace (private) byte offsets
    size_t off_gauge, off_gghost, off_r, off_p, off_t, off_sc, off_ss, off_ticket, off_partials, off_hist, ws_needed;
    size_t off_gauge_f, off_gghost_f, off_xf, off_rf, off_pf, off_tf;  // fp32 copies of the mixed-precision solver
    // mailbox (peer-visible) byte offsets
    size_t mb_word, mb_ghost, mb_needed;
    size_t max_blocks;
    int nsm;      // multiprocessors of the device the memory was bound on (148 on B200 until then)
    char* ws;
    char* mb;
    char* peer[LQCD_SLAB_MAX_RANKS];
    cudaStream_t stream;
    int device;
    bool memory_set, connected, gauge_loaded;
    bool gauge_f_ready;  // the fp32 link copies match the loaded fp64 ones
    int recon, check_every, timeout_ms, use_graph, fuse_sync;
    int acquire;       // LQCD_SLAB_OPT_ACQUIRE: -1 auto (= peers_remote), 0, 1
    bool peers_remote;  // some peer's mailbox is on another device (set by lqcd_slab_connect)
    unsigned long long seq;  // synchronisation points passed
    CgScalars* h_sc;         // pinned, 2 slots
    SlabScalars* h_ss;       // pinned
    cudaEvent_t ev[2];
    bool host_ready;
    long long launches;
    char err[320];

    cplx* gauge() const { return (cplx*)(ws + off_gauge); }
    cplx* gghost() const { return (cplx*)(ws + off_gghost); }
    cplx* r() const { return (cplx*)(ws + off_r); }
    cplx* p() const { return (cplx*)(ws + off_p); }
    cplx* t() const { return (cplx*)(ws + off_t); }
    cplxf* gauge_f() const { return (cplxf*)(ws + off_gauge_f); }
    cplxf* gghost_f() const { return (cplxf*)(ws + off_gghost_f); }
    cplxf* xf() const { return (cplxf*)(ws + off_xf); }
    cplxf* rf() const { return (cplxf*)(ws + off_rf); }
    cplxf* pf() const { return (cplxf*)(ws + off_pf); }
    cplxf* tf() const { return (cplxf*)(ws + off_tf); }
    CgScalars* sc() const { return (CgScalars*)(ws + off_sc); }
    SlabScalars* ss() const { return (SlabScalars*)(ws + off_ss); }
    double* hist() const { return (double*)(ws + off_hist); }
    ReduceScratch rs() const
    {
        ReduceScratch q;
        q.partials = (double*)(ws + off_partials);
        q.ticket = (unsigned int*)(ws + off_ticket);
        return q;
    }
    // ghost face `side` (0 = below the slab, 1 = above) of buffer `buf` in the mailbox at `base`
    cplx* ghost(char* base, int buf, int side) const
    {
        return (cplx*)(base + mb_ghost) + (size_t)(buf * 2 + side) * 3 * (size_t)sh;
    }
};

namespace {

int fail(lqcd_slab* s, int code, const char* fmt, ...)
{
    if (s) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(s->err, sizeof s->err, fmt, ap);
        va_end(ap);
    }
    return code;
}

#define SLAB_CUDA(call)                                                                                \
    do {                                                                                               \
        cudaError_t e_ = (call);                                                                       \
        if (e_ != cudaSuccess)                                                                         \
            return fail(s, LQCD_ECUDA, "%s failed: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, \
                        __LINE__);                                                                     \
    } while (0)

#define SLAB_LAUNCH_CHECK()                                                                            \
    do {                                                                                               \
        s->launches++;                                                                                 \
        cudaError_t e_ = cudaGetLastError();                                                           \
        if (e_ != cudaSuccess)                                                                         \
            return fail(s, LQCD_ECUDA, "kernel launch failed: %s (%s:%d)", cudaGetErrorString(e_),     \
                        __FILE__, __LINE__);                                                           \
    } while (0)

unsigned int vec_grid(const lqcd_slab* s)
{
    size_t b = (s->nvec + kVecBlock - 1) / kVecBlock;
    size_t cap = (size_t)s->nsm * 8;
    if (cap > 4096) cap = 4096;   // the partial-sum area has V/64 + 4096 slots
    if (b > cap) b = cap;
    if (b < 1) b = 1;
    return (unsigned int)b;
}

// Face-first walk of the slab vector kernels (slab_kernels.cuh): the face elements, one per thread, to the first
// blocks of the grid -- at most half of it.
SlabVecPlan vec_plan(const lqcd_slab* s, unsigned int grid)
{
    SlabVecPlan pl;
    pl.n = (unsigned int)s->nvec;  // 3 Vh <= 3 * 2^29
    pl.nface = 6 * (size_t)s->sh < s->nvec ? (unsigned int)(6 * (size_t)s->sh) : (unsigned int)s->nvec;
    size_t fb = ((size_t)pl.nface + kVecBlock - 1) / kVecBlock;
    if (pl.nface == pl.n) fb = grid;               // no interior (T = 2): every block owns face elements
    else if (fb > grid / 2) fb = grid / 2;
    if (fb < 1) fb = 1;
    pl.face_blocks = (int)fb;
    return pl;
}

// The n slabs of a *_group call.
struct Group {
    lqcd_slab* const* s;
    int n;
};

int group_check(const Group& G, bool need_gauge)
{
    if (!G.s || G.n < 1) return LQCD_EARG;
    for (int r = 0; r < G.n; ++r)
        if (!G.s[r]) return LQCD_EARG;
    for (int r = 0; r < G.n; ++r) {
        lqcd_slab* s = G.s[r];
        if (s->nranks != G.n || s->rank != r)
            return fail(s, LQCD_EARG, "group of %d slabs: entry %d is rank %d of %d", G.n, r, s->rank, s->nranks);
        if (!s->memory_set) return fail(s, LQCD_ESTATE, "memory not set (call lqcd_slab_set_memory)");
        if (!s->connected) return fail(s, LQCD_ESTATE, "peers not connected (call lqcd_slab_connect)");
        if (need_gauge && !s->gauge_loaded) return fail(s, LQCD_ESTATE, "gauge field not loaded (call lqcd_slab_load_gauge)");
        if (s->seq != G.s[0]->seq || s->recon != G.s[0]->recon || memcmp(s->L, G.s[0]->L, sizeof s->L))
            return fail(s, LQCD_ESTATE, "the slabs of a group must share lattice, options and call history");
    }
    return LQCD_OK;
}

// One rank alone (n = 1 of a larger job): the group is that slab; its peers are other processes.
int single_check(lqcd_slab* s, bool need_gauge)
{
    if (!s) return LQCD_EARG;
    if (!s->memory_set) return fail(s, LQCD_ESTATE, "memory not set (call lqcd_slab_set_memory)");
    if (!s->connected) return fail(s, LQCD_ESTATE, "peers not connected (call lqcd_slab_connect)");
    if (need_gauge && !s->gauge_loaded) return fail(s, LQCD_ESTATE, "gauge field not loaded (call lqcd_slab_load_gauge)");
    return LQCD_OK;
}

int use_device(lqcd_slab* s)
{
    SLAB_CUDA(cudaSetDevice(s->device));
    return LQCD_OK;
}

// ---------------------------------------------------------------- pieces of a phase
SlabPush push_next(const lqcd_slab* s)
{
    // faces stored now are read after the NEXT synchronisation point: buffer (seq + 1) & 1
    const int buf = (int)((s->seq + 1) & 1ull);
    const int R = s->nranks;
    SlabPush ph;
    ph.lo = s->ghost(s->peer[(s->rank + R - 1) % R], buf, 1);  // my first slice is the lower rank's "above"
    ph.hi = s->ghost(s->peer[(s->rank + 1) % R], buf, 0);      // my last slice is the upper rank's "below"
    ph.sh = s->sh;
    ph.Vh = s->g.Vh;
    return ph;
}

StagArgsD stag_args(const lqcd_slab* s, int parity, const cplx* in, cplx* out, bool push)
{
    StagArgsD a;
    memset(&a, 0, sizeof a);
    a.g = s->g;
    a.parity = parity;
    a.gauge = s->gauge();
    a.in = in;
    a.out = out;
    a.sc = s->sc();
    a.rs = s->rs();
    a.hist = s->hist();
    a.sl.t0 = s->t0;
    a.sl.L3g = s->L[3];
    a.sl.sh = s->sh;
    const int buf = (int)(s->seq & 1ull);  // faces of `in` arrived with the last synchronisation point
    a.sl.ghost_lo = s->ghost(s->mb, buf, 0);
    a.sl.ghost_hi = s->ghost(s->mb, buf, 1);
    a.sl.gauge_ghost = s->gghost();
    if (push) {
        const SlabPush ph = push_next(s);
        a.sl.push_lo = ph.lo;
        a.sl.push_hi = ph.hi;
    }
    a.sl.part = s->ss()->part;
    return a;
}

// Threads per block by the size of the LOCAL lattice, as stag_block_for in lqcd_api.cu: strong scaling
// shrinks the slabs, and small lattices want more, smaller blocks.
int slab_block_for(const lqcd_slab* s)
{
    const long long blocks128 = ((long long)s->g.Vh + 127) / 128;
    if (blocks128 < 2 * s->nsm) return 32;
    if (blocks128 < 8 * s->nsm) return 64;
    return 128;
}

template <int EPI, int BLOCK>
int launch_stag_block(lqcd_slab* s, const StagArgsD& a, const SlabSyncArgs* sy)
{
    const unsigned int grid = blocks_for(s->g.Vh, BLOCK);
    if (sy) {  // the synchronisation point that follows runs in the kernel's last block
        if (s->recon == 12)
            stag_dslash_slab_sync_kernel<EPI, BLOCK, 12, cplx><<<grid, BLOCK, 0, s->stream>>>(a, *sy);
        else
            stag_dslash_slab_sync_kernel<EPI, BLOCK, 18, cplx><<<grid, BLOCK, 0, s->stream>>>(a, *sy);
    } else {
        if (s->recon == 12)
            stag_dslash_slab_kernel<EPI, BLOCK, 12, cplx><<<grid, BLOCK, 0, s->stream>>>(a);
        else
            stag_dslash_slab_kernel<EPI, BLOCK, 18, cplx><<<grid, BLOCK, 0, s->stream>>>(a);
    }
    SLAB_LAUNCH_CHECK();
    return LQCD_OK;
}

template <int EPI>
int launch_stag_any(lqcd_slab* s, const StagArgsD& a, const SlabSyncArgs* sy)
{
    const int block = slab_block_for(s);
    if (block == 32) return launch_stag_block<EPI, 32>(s, a, sy);
    if (block == 64) return launch_stag_block<EPI, 64>(s, a, sy);
    return launch_stag_block<EPI, kStagBlock>(s, a, sy);
}

template <int EPI>
int launch_stag(lqcd_slab* s, const StagArgsD& a)
{
    return launch_stag_any<EPI>(s, a, nullptr);
}

// The same kernel with the synchronisation point that follows it run by its last block.
template <int EPI>
int launch_stag_sync(lqcd_slab* s, const StagArgsD& a, const SlabSyncArgs& sy)
{
    return launch_stag_any<EPI>(s, a, &sy);
}

int launch_push_faces(lqcd_slab* s, const cplx* v)
{
    const unsigned int grid = blocks_for(6 * (size_t)s->sh, kVecBlock);
    slab_push_faces_kernel<kVecBlock><<<grid < 1184 ? grid : 1184, kVecBlock, 0, s->stream>>>(v, push_next(s));
    SLAB_LAUNCH_CHECK();
    return LQCD_OK;
}

SlabSyncArgs sync_args(const lqcd_slab* s, int op, int nvals, double m2, double tol, int maxiter, double delta = 0.0)
{
    SlabSyncArgs a;
    memset(&a, 0, sizeof a);
    a.rank = s->rank;
    a.nranks = s->nranks;
    a.nvals = nvals;
    a.own.word = (unsigned long long*)(s->mb + s->mb_word);
    a.own.ghost = (cplx*)(s->mb + s->mb_ghost);
    for (int r = 0; r < s->nranks; ++r) a.peer_word[r] = (unsigned long long*)(s->peer[r] + s->mb_word);
    a.ss = s->ss();
    a.sc = s->sc();
    a.hist = s->hist();
    a.op = op;
    a.m2 = m2;
    a.tol = tol;
    a.delta = delta;
    a.maxiter = maxiter;
    a.timeout_ns = (unsigned long long)s->timeout_ms * 1000000ull;
    a.sys_fences = s->acquire >= 0 ? s->acquire : (s->peers_remote ? 1 : 0);
    return a;
}

// One synchronisation point for the whole group: every slab signals, then every slab waits and
// combines.  (With all slabs on one stream the signals therefore precede every wait: no kernel spins.)
// A group of one -- a rank driving only its own slab -- does both in one launch.
// in_producer: the producer kernel was launched with the synchronisation point in its last block
// (fused(G)); only the host's count moves.
int group_sync(const Group& G, int op, int nvals, double m2 = 0.0, double tol = 0.0, int maxiter = 0,
               bool in_producer = false, double delta = 0.0)
{
    for (int r = 0; r < G.n; ++r) G.s[r]->seq += 1;  // host copy: selects the ghost buffers; the kernels count on the device
    if (in_producer) return LQCD_OK;
    if (G.n == 1) {
        lqcd_slab* s = G.s[0];
        int rc = use_device(s);
        if (rc) return rc;
        slab_signal_wait_combine_kernel<<<1, 32, 0, s->stream>>>(sync_args(s, op, nvals, m2, tol, maxiter, delta));
        SLAB_LAUNCH_CHECK();
        return LQCD_OK;
    }
    for (int r = 0; r < G.n; ++r) {
        lqcd_slab* s = G.s[r];
        int rc = use_device(s);
        if (rc) return rc;
        slab_signal_kernel<<<1, 32, 0, s->stream>>>(sync_args(s, op, nvals, m2, tol, maxiter, delta));
        SLAB_LAUNCH_CHECK();
    }
    for (int r = 0; r < G.n; ++r) {
        lqcd_slab* s = G.s[r];
        int rc = use_device(s);
        if (rc) return rc;
        slab_wait_combine_kernel<<<1, 32, 0, s->stream>>>(sync_args(s, op, nvals, m2, tol, maxiter, delta));
        SLAB_LAUNCH_CHECK();
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

// A rank that drives only its own slab runs each synchronisation point inside the producer kernel.
// Never a group of several slabs: on one stream its producers would wait for kernels queued behind them.
bool fused(const Group& G) { return G.n == 1 && G.s[0]->fuse_sync; }

int ensure_host(lqcd_slab* s)
{
    if (s->host_ready) return LQCD_OK;
    SLAB_CUDA(cudaHostAlloc((void**)&s->h_sc, 2 * sizeof(CgScalars), cudaHostAllocDefault));
    SLAB_CUDA(cudaHostAlloc((void**)&s->h_ss, sizeof(SlabScalars), cudaHostAllocDefault));
    SLAB_CUDA(cudaEventCreateWithFlags(&s->ev[0], cudaEventDisableTiming));
    SLAB_CUDA(cudaEventCreateWithFlags(&s->ev[1], cudaEventDisableTiming));
    s->host_ready = true;
    return LQCD_OK;
}

int read_scalars(lqcd_slab* s, int slot)
{
    SLAB_CUDA(cudaMemcpyAsync(&s->h_sc[slot], s->sc(), sizeof(CgScalars), cudaMemcpyDeviceToHost, s->stream));
    SLAB_CUDA(cudaEventRecord(s->ev[slot], s->stream));
    return LQCD_OK;
}

// Drain every slab's stream and report a timed-out wait.
int group_finish(const Group& G)
{
    for (int r = 0; r < G.n; ++r) {
        lqcd_slab* s = G.s[r];
        int rc = use_device(s);
        if (rc) return rc;
        SLAB_CUDA(cudaMemcpyAsync(s->h_ss, s->ss(), sizeof(SlabScalars), cudaMemcpyDeviceToHost, s->stream));
        SLAB_CUDA(cudaStreamSynchronize(s->stream));
        if (s->h_ss->err) {
            cudaMemsetAsync(&s->ss()->err, 0, sizeof(int), s->stream);
            return fail(s, LQCD_ECOMM, "rank %d: a peer did not reach synchronisation point %llu within %d ms", s->rank,
                        s->seq, s->timeout_ms);
        }
    }
    return LQCD_OK;
}

// ---------------------------------------------------------------- operations on a group
// Faces of a caller-supplied vector: a separate small kernel, then a synchronisation point.
int group_halo_of(const Group& G, const cplx* const* v)
{
    for (int r = 0; r < G.n; ++r) {
        int rc = use_device(G.s[r]);
        if (rc) return rc;
        rc = launch_push_faces(G.s[r], v[r]);
        if (rc) return rc;
    }
    return group_sync(G, SLAB_OP_NONE, 0);
}

int group_dslash(const Group& G, int out_parity, const cplx* const* in, cplx* const* out)
{
    int rc = group_halo_of(G, in);
    if (rc) return rc;
    for (int r = 0; r < G.n; ++r) {
        rc = use_device(G.s[r]);
        if (rc) return rc;
        rc = launch_stag<SE_PLAIN>(G.s[r], stag_args(G.s[r], out_parity, in[r], out[r], false));
        if (rc) return rc;
    }
    return LQCD_OK;
}

// t = D_oe v with the faces of t pushed, then a halo-only synchronisation point: t is ready for D_eo.
int group_first_hop(const Group& G, const cplx* const* v)
{
    int rc = group_halo_of(G, v);
    if (rc) return rc;
    for (int r = 0; r < G.n; ++r) {
        rc = use_device(G.s[r]);
        if (rc) return rc;
        rc = launch_stag<SE_PLAIN>(G.s[r], stag_args(G.s[r], LQCD_ODD, v[r], G.s[r]->t(), true));
        if (rc) return rc;
    }
    return group_sync(G, SLAB_OP_NONE, 0);
}

int group_MdagM(const Group& G, double mass, const cplx* const* in, cplx* const* out)
{
    int rc = group_first_hop(G, in);
    if (rc) return rc;
    for (int r = 0; r < G.n; ++r) {
        lqcd_slab* s = G.s[r];
        rc = use_device(s);
        if (rc) return rc;
        StagArgsD a = stag_args(s, LQCD_EVEN, s->t(), out[r], false);
        a.m2 = mass * mass;
        a.p = in[r];
        rc = launch_stag<SE_MDAGM>(s, a);
        if (rc) return rc;
    }
    return LQCD_OK;
}

// One CG iteration (S1-S5) = three producer phases, each closed by a synchronisation point.
int group_iteration(const Group& G, double mass, cplx* const* x)
{
    const double m2 = mass * mass;
    const bool fz = fused(G);
    int rc;
    for (int r = 0; r < G.n; ++r) {  // S1: t = D_oe p, partial <t,t>; faces of t -> neighbours
        lqcd_slab* s = G.s[r];
        rc = use_device(s);
        if (rc) return rc;
        const StagArgsD a = stag_args(s, LQCD_ODD, s->p(), s->t(), true);
        rc = fz ? launch_stag_sync<SE_NORM>(s, a, sync_args(s, SLAB_OP_ALPHA, 1, m2, 0.0, 0)) : launch_stag<SE_NORM>(s, a);
        if (rc) return rc;
    }
    rc = group_sync(G, SLAB_OP_ALPHA, 1, m2, 0.0, 0, fz);  // S2
    if (rc) return rc;
    for (int r = 0; r < G.n; ++r) {  // S3: D_eo t fused with the x / r updates, partial <r,r>
        lqcd_slab* s = G.s[r];
        rc = use_device(s);
        if (rc) return rc;
        StagArgsD a = stag_args(s, LQCD_EVEN, s->t(), nullptr, false);
        a.m2 = m2;
        a.p = s->p();
        a.x = x[r];
        a.r = s->r();
        rc = fz ? launch_stag_sync<SE_CGUPDATE>(s, a, sync_args(s, SLAB_OP_UPDATE, 1, 0.0, 0.0, 0)) : launch_stag<SE_CGUPDATE>(s, a);
        if (rc) return rc;
    }
    rc = group_sync(G, SLAB_OP_UPDATE, 1, 0.0, 0.0, 0, fz);  // beta, exit test (S4 happens on every rank identically)
    if (rc) return rc;
    for (int r = 0; r < G.n; ++r) {  // S5: p = r + beta p, partial <p,p>; faces of p -> neighbours
        lqcd_slab* s = G.s[r];
        rc = use_device(s);
        if (rc) return rc;
        slab_cg_pupdate_kernel<kVecBlock, cplx><<<vec_grid(s), kVecBlock, 0, s->stream>>>(
            s->r(), s->p(), vec_plan(s, vec_grid(s)), push_next(s), s->sc(), s->ss(), s->rs(), sync_args(s, SLAB_OP_PP, 1, 0.0, 0.0, 0), fz ? 1 : 0);
        SLAB_LAUNCH_CHECK();
    }
    return group_sync(G, SLAB_OP_PP, 1, 0.0, 0.0, 0, fz);
}

int group_cg(const Group& G, double mass, double tol, int maxiter, const cplx* const* b, cplx* const* x, int* iters,
             double* true_residual)
{
    int rc;
    lqcd_slab* s0 = G.s[0];
    for (int r = 0; r < G.n; ++r) {  // S6
        lqcd_slab* s = G.s[r];
        rc = use_device(s);
        if (rc) return rc;
        slab_cg_init_kernel<kVecBlock><<<vec_grid(s), kVecBlock, 0, s->stream>>>(
            b[r], x[r], s->r(), s->p(), vec_plan(s, vec_grid(s)), push_next(s), s->ss(), s->rs(), sync_args(s, SLAB_OP_INIT, 1, 0.0, tol, maxiter),
            fused(G) ? 1 : 0);
        SLAB_LAUNCH_CHECK();
    }
    rc = group_sync(G, SLAB_OP_INIT, 1, 0.0, tol, maxiter, fused(G));
    if (rc) return rc;

    // Host loop as LQCD_CG_ASYNC of lqcd_cg_solve: batches of check_every iterations are enqueued
    // while the previous batch's scalars travel; after `done` every kernel of every rank is a no-op
    // (signals and waits still run, so the ranks stay in step).  The scalars are bit-identical on all
    // ranks; rank 0's copy (of this process) is the one read.
    CgScalars* h = s0->h_sc;
    int batch = s0->check_every;
    // With every slab on one stream (a rank alone, or the single-GPU group) the batch is captured once
    // and replayed as a CUDA graph: the synchronisation kernels take their number from device memory,
    // and an even count of synchronisation points per replay (3 per iteration, so an even batch)
    // leaves the ghost-buffer parity baked into the captured kernels valid for every replay.
    bool one_stream = s0->stream != nullptr;
    for (int r = 1; r < G.n; ++r)
        if (G.s[r]->stream != s0->stream || G.s[r]->device != s0->device) one_stream = false;
    GraphHolder gh;
    long long per_replay[LQCD_SLAB_MAX_RANKS] = { 0 };
    if (s0->use_graph && one_stream && maxiter > 0) {
        lqcd_slab* s = s0;
        if (batch & 1) batch += 1;  // iterations after convergence are no-ops, so this changes nothing
        unsigned long long seq0[LQCD_SLAB_MAX_RANKS];
        long long launched0[LQCD_SLAB_MAX_RANKS];
        for (int r = 0; r < G.n; ++r) {
            seq0[r] = G.s[r]->seq;
            launched0[r] = G.s[r]->launches;
        }
        SLAB_CUDA(cudaStreamBeginCapture(s0->stream, cudaStreamCaptureModeThreadLocal));
        rc = LQCD_OK;
        for (int k = 0; k < batch && !rc; ++k) rc = group_iteration(G, mass, x);
        cudaError_t ce = cudaStreamEndCapture(s0->stream, &gh.graph);
        for (int r = 0; r < G.n; ++r) {  // capturing ran nothing
            per_replay[r] = G.s[r]->launches - launched0[r];
            G.s[r]->launches = launched0[r];
            G.s[r]->seq = seq0[r];
        }
        if (rc) return rc;
        SLAB_CUDA(ce);
        SLAB_CUDA(cudaGraphInstantiate(&gh.exec, gh.graph, 0));
    }
    int slot = 0;
    bool pending[2] = { false, false };
    bool finished = false;
    long long enqueued = 0;
    while (!finished) {
        if (enqueued < (long long)maxiter) {
            if (gh.exec) {
                lqcd_slab* s = s0;
                SLAB_CUDA(cudaGraphLaunch(gh.exec, s0->stream));
                for (int r = 0; r < G.n; ++r) {
                    G.s[r]->seq += 3ull * (unsigned long long)batch;
                    G.s[r]->launches += per_replay[r];
                }
            } else {
                for (int k = 0; k < batch; ++k) {
                    rc = group_iteration(G, mass, x);
                    if (rc) return rc;
                }
            }
            enqueued += batch;
        }
        rc = use_device(s0);
        if (rc) return rc;
        rc = read_scalars(s0, slot);
        if (rc) return rc;
        pending[slot] = true;
        const int other = slot ^ 1;
        if (pending[other]) {
            lqcd_slab* s = s0;
            SLAB_CUDA(cudaEventSynchronize(s->ev[other]));
            pending[other] = false;
            if (h[other].done) finished = true;
        }
        slot = other;
    }
    rc = group_finish(G);
    if (rc) return rc;
    // One counter again.  Inside the loop the host count selects the ghost buffers (it is baked into the launches, so
    // it must advance with every enqueued iteration) and the device count tags the words (it must not be baked into a
    // replayed graph); with the synchronisation point fused into the producers, iterations enqueued after convergence
    // are complete no-ops, so the device count stops where the host count runs on.  Both are the same on every rank
    // (the host loop is deterministic, the scalars bit-identical), which is all the protocol needs; and every ghost
    // face has been consumed -- a rank passes the last real point only after its peers have signalled it, i.e. after
    // their last Dslash.  From here on the host continues from the device's number (copied by group_finish).
    for (int r = 0; r < G.n; ++r) {
        if (G.s[r]->h_ss->seq > G.s[r]->seq) return fail(G.s[r], LQCD_ESTATE, "rank %d: device passed %llu synchronisation points, host enqueued %llu",
                                                       r, G.s[r]->h_ss->seq, G.s[r]->seq);
        G.s[r]->seq = G.s[r]->h_ss->seq;
    }

    // S7: |b - A x| / |b| with a fresh A
    rc = group_first_hop(G, x);
    if (rc) return rc;
    for (int r = 0; r < G.n; ++r) {
        lqcd_slab* s = G.s[r];
        rc = use_device(s);
        if (rc) return rc;
        StagArgsD a = stag_args(s, LQCD_EVEN, s->t(), nullptr, false);
        a.m2 = mass * mass;
        a.p = x[r];
        a.b = b[r];
        rc = fused(G) ? launch_stag_sync<SE_RESIDUAL>(s, a, sync_args(s, SLAB_OP_RES2, 1, 0.0, 0.0, 0)) : launch_stag<SE_RESIDUAL>(s, a);
        if (rc) return rc;
    }
    rc = group_sync(G, SLAB_OP_RES2, 1, 0.0, 0.0, 0, fused(G));
    if (rc) return rc;
    rc = use_device(s0);
    if (rc) return rc;
    rc = read_scalars(s0, 0);
    if (rc) return rc;
    rc = group_finish(G);
    if (rc) return rc;
    *iters = h[0].iter;
    *true_residual = h[0].bb > 0.0 ? sqrt(h[0].res2 / h[0].bb) : 0.0;
    return h[0].rr_new <= h[0].thresh ? LQCD_OK : LQCD_MAXITER;
}

// ---------------------------------------------------------------- mixed precision on slabs (SURVEY.md 8(f) rows 3 + 4b)
// The solver of lqcd_cg_solve_mixed (fp32 iterations, fp64 reliable updates) on the slab
// decomposition: the fp32 vectors p and t travel as fp32 faces (half the NVLink bytes), the reliable update's x as
// fp64 faces; every sum is combined in rank order as in the fp64 slab solver.  Separate launches per
// synchronisation point (no fused tails, no graph replay): the host loop has to see `pause`.
typedef StagArgs<cplxf> StagArgsF;

SlabPushF push_next_f(const lqcd_slab* s)
{
    const SlabPush ph = push_next(s);
    SlabPushF f;
    f.lo = (cplxf*)ph.lo;  // the same ghost areas, read back as fp32 by the fp32 kernels
    f.hi = (cplxf*)ph.hi;
    f.sh = ph.sh;
    f.Vh = ph.Vh;
    return f;
}

StagArgsF stag_args_f(const lqcd_slab* s, int parity, const cplxf* in, cplxf* out, bool push)
{
    StagArgsF a;
    memset(&a, 0, sizeof a);
    a.g = s->g;
    a.parity = parity;
    a.gauge = s->gauge_f();
    a.in = in;
    a.out = out;
    a.sc = s->sc();
    a.rs = s->rs();
    a.hist = s->hist();
    a.sl.t0 = s->t0;
    a.sl.L3g = s->L[3];
    a.sl.sh = s->sh;
    const int buf = (int)(s->seq & 1ull);
    a.sl.ghost_lo = (const cplxf*)s->ghost(s->mb, buf, 0);
    a.sl.ghost_hi = (const cplxf*)s->ghost(s->mb, buf, 1);
    a.sl.gauge_ghost = s->gghost_f();
    if (push) {
        const SlabPushF ph = push_next_f(s);
        a.sl.push_lo = ph.lo;
        a.sl.push_hi = ph.hi;
    }
    a.sl.part = s->ss()->part;
    return a;
}

template <int EPI>
int launch_stag_f(lqcd_slab* s, const StagArgsF& a)
{
    const unsigned int grid = blocks_for(s->g.Vh, kStagBlock);
    if (s->recon == 12)
        stag_dslash_slab_kernel<EPI, kStagBlock, 12, cplxf><<<grid, kStagBlock, 0, s->stream>>>(a);
    else
        stag_dslash_slab_kernel<EPI, kStagBlock, 18, cplxf><<<grid, kStagBlock, 0, s->stream>>>(a);
    SLAB_LAUNCH_CHECK();
    return LQCD_OK;
}

int ensure_gauge_f(lqcd_slab* s)
{
    if (s->gauge_f_ready) return LQCD_OK;
    const size_t nc = (size_t)(s->recon / 2);
    gauge_narrow_kernel<<<s->nsm * 8, 256, 0, s->stream>>>(s->gauge(), s->gauge_f(), (size_t)s->g.V * 4 * nc);
    SLAB_LAUNCH_CHECK();
    gauge_narrow_kernel<<<64, 256, 0, s->stream>>>(s->gghost(), s->gghost_f(), 2 * nc * (size_t)s->sh);
    SLAB_LAUNCH_CHECK();
    s->gauge_f_ready = true;
    return LQCD_OK;
}

int group_pupdate_f(const Group& G)  // S5 on the fp32 copies; faces of ps -> neighbours
{
    for (int r = 0; r < G.n; ++r) {
        lqcd_slab* s = G.s[r];
        int rc = use_device(s);
        if (rc) return rc;
        slab_cg_pupdate_kernel<kVecBlock, cplxf><<<vec_grid(s), kVecBlock, 0, s->stream>>>(
            s->rf(), s->pf(), vec_plan(s, vec_grid(s)), push_next_f(s), s->sc(), s->ss(), s->rs(), sync_args(s, SLAB_OP_PP, 1, 0.0, 0.0, 0), 0);
        SLAB_LAUNCH_CHECK();
    }
    return group_sync(G, SLAB_OP_PP, 1);
}

int group_iteration_mixed(const Group& G, double mass)
{
    const double m2 = mass * mass;
    int rc;
    for (int r = 0; r < G.n; ++r) {  // S1: ts = D^_oe ps, partial <ts,ts>; fp32 faces of ts -> neighbours
        lqcd_slab* s = G.s[r];
        rc = use_device(s);
        if (rc) return rc;
        rc = launch_stag_f<SE_NORM>(s, stag_args_f(s, LQCD_ODD, s->pf(), s->tf(), true));
        if (rc) return rc;
    }
    rc = group_sync(G, SLAB_OP_ALPHA, 1, m2);  // S2
    if (rc) return rc;
    for (int r = 0; r < G.n; ++r) {  // S3 on the fp32 vectors
        lqcd_slab* s = G.s[r];
        rc = use_device(s);
        if (rc) return rc;
        StagArgsF a = stag_args_f(s, LQCD_EVEN, s->tf(), nullptr, false);
        a.m2 = m2;
        a.p = s->pf();
        a.x = s->xf();
        a.r = s->rf();
        rc = launch_stag_f<SE_CGUPDATE_MIXED>(s, a);
        if (rc) return rc;
    }
    rc = group_sync(G, SLAB_OP_UPDATE_MIXED, 1);  // beta or pause, identically on every rank
    if (rc) return rc;
    return group_pupdate_f(G);
}

// The reliable update, all fp64: x += xs, xs = 0; r = b - A x with the faces of x and of D_oe x exchanged as in
// the fp64 solver; rs = fl32(r); <r,r> combined over the ranks, beta, exit test; then the waiting fp32 p-update.
int group_reliable_update(const Group& G, double mass, const cplx* const* b, cplx* const* x)
{
    int rc;
    for (int r = 0; r < G.n; ++r) {
        lqcd_slab* s = G.s[r];
        rc = use_device(s);
        if (rc) return rc;
        mixed_accumulate_kernel<kVecBlock><<<vec_grid(s), kVecBlock, 0, s->stream>>>(x[r], s->xf(), s->nvec, s->sc(), 1);
        SLAB_LAUNCH_CHECK();
    }
    rc = group_first_hop(G, x);  // faces of x, t = D_oe x, faces of t
    if (rc) return rc;
    for (int r = 0; r < G.n; ++r) {
        lqcd_slab* s = G.s[r];
        rc = use_device(s);
        if (rc) return rc;
        StagArgsD a = stag_args(s, LQCD_EVEN, s->t(), nullptr, false);
        a.m2 = mass * mass;
        a.p = x[r];
        a.b = b[r];
        a.rf = s->rf();
        rc = launch_stag<SE_RELIABLE>(s, a);
        if (rc) return rc;
    }
    rc = group_sync(G, SLAB_OP_RELIABLE, 1);
    if (rc) return rc;
    return group_pupdate_f(G);
}

int group_cg_mixed(const Group& G, double mass, double tol, double delta, int maxiter, const cplx* const* b, cplx* const* x,
                   int* iters, int* reliable_updates, double* true_residual)
{
    int rc;
    lqcd_slab* s0 = G.s[0];
    for (int r = 0; r < G.n; ++r) {
        lqcd_slab* s = G.s[r];
        rc = use_device(s);
        if (rc) return rc;
        rc = ensure_gauge_f(s);
        if (rc) return rc;
        slab_cg_init_mixed_kernel<kVecBlock><<<vec_grid(s), kVecBlock, 0, s->stream>>>(
            b[r], x[r], s->xf(), s->rf(), s->pf(), vec_plan(s, vec_grid(s)), push_next_f(s), s->ss(), s->rs());
        SLAB_LAUNCH_CHECK();
    }
    rc = group_sync(G, SLAB_OP_INIT_MIXED, 2, 0.0, tol, maxiter, false, delta);
    if (rc) return rc;

    // Host loop as cg_run_mixed of lqcd_api.cu: batches of iterations enqueued while the previous batch's scalars
    // travel; iterations enqueued after the device paused (or finished) are no-ops on every rank -- the
    // synchronisation kernels still run, so the ranks stay in step -- and the update sequence is enqueued exactly
    // once per pause.  The scalars are bit-identical on all ranks; rank 0's copy (of this process) is read.
    CgScalars* h = s0->h_sc;
    const int batch = s0->check_every;
    int slot = 0, updates_enqueued = 0;
    bool pending[2] = { false, false };
    bool finished = maxiter <= 0;
    while (!finished) {
        for (int k = 0; k < batch; ++k) {
            rc = group_iteration_mixed(G, mass);
            if (rc) return rc;
        }
        rc = use_device(s0);
        if (rc) return rc;
        rc = read_scalars(s0, slot);
        if (rc) return rc;
        pending[slot] = true;
        const int look = slot ^ 1;
        if (pending[look]) {
            lqcd_slab* s = s0;
            SLAB_CUDA(cudaEventSynchronize(s->ev[look]));
            pending[look] = false;
            if (h[look].done) {
                finished = true;
            } else if (h[look].pause && h[look].nupd == updates_enqueued) {
                rc = group_reliable_update(G, mass, b, x);
                if (rc) return rc;
                ++updates_enqueued;
            }
        }
        slot ^= 1;
    }
    for (int r = 0; r < G.n; ++r) {  // whatever the fp32 iteration still holds goes into x
        lqcd_slab* s = G.s[r];
        rc = use_device(s);
        if (rc) return rc;
        mixed_accumulate_kernel<kVecBlock><<<vec_grid(s), kVecBlock, 0, s->stream>>>(x[r], s->xf(), s->nvec, s->sc(), 0);
        SLAB_LAUNCH_CHECK();
    }
    rc = use_device(s0);
    if (rc) return rc;
    rc = read_scalars(s0, 0);
    if (rc) return rc;
    rc = group_finish(G);
    if (rc) return rc;
    const int it = h[0].iter, nupd = h[0].nupd;
    const bool converged = h[0].bb == 0.0 || (h[0].rr_new <= h[0].thresh && !h[0].pause && nupd > 0);

    // S7: |b - A x| / |b| with a fresh fp64 A
    rc = group_first_hop(G, x);
    if (rc) return rc;
    for (int r = 0; r < G.n; ++r) {
        lqcd_slab* s = G.s[r];
        rc = use_device(s);
        if (rc) return rc;
        StagArgsD a = stag_args(s, LQCD_EVEN, s->t(), nullptr, false);
        a.m2 = mass * mass;
        a.p = x[r];
        a.b = b[r];
        rc = launch_stag<SE_RESIDUAL>(s, a);
        if (rc) return rc;
    }
    rc = group_sync(G, SLAB_OP_RES2, 1);
    if (rc) return rc;
    rc = use_device(s0);
    if (rc) return rc;
    rc = read_scalars(s0, 0);
    if (rc) return rc;
    rc = group_finish(G);
    if (rc) return rc;
    *iters = it;
    *reliable_updates = nupd;
    *true_residual = h[0].bb > 0.0 ? sqrt(h[0].res2 / h[0].bb) : 0.0;
    return converged ? LQCD_OK : LQCD_MAXITER;
}

}  // namespace

// =========================================================================== C-ABI
extern "C" {

int lqcd_slab_create(lqcd_slab** out, int L0, int L1, int L2, int L3, int rank, int nranks)
{
    if (!out) return LQCD_EARG;
    *out = nullptr;
    if (nranks < 1 || nranks > LQCD_SLAB_MAX_RANKS || rank < 0 || rank >= nranks) return LQCD_EARG;
    const int L[4] = { L0, L1, L2, L3 };
    for (int mu = 0; mu < 4; ++mu)
        if (L[mu] < 2 || (L[mu] & 1)) return LQCD_EDIM;
    if (L3 % nranks) return LQCD_EDIM;
    const int T = L3 / nranks;
    if (T < 2 || (T & 1)) return LQCD_EDIM;  // even slabs keep local parity = global parity
    const long long V = (long long)L0 * L1 * L2 * T;
    if (V > (1LL << 30)) return LQCD_EDIM;
    lqcd_slab* c = (lqcd_slab*)calloc(1, sizeof(lqcd_slab));
    if (!c) return LQCD_ENOMEM;
    memcpy(c->L, L, sizeof L);
    c->rank = rank;
    c->nranks = nranks;
    c->T = T;
    c->t0 = rank * T;
    c->g.Lh = L0 / 2;
    c->g.L1 = L1;
    c->g.L2 = L2;
    c->g.L3 = T;
    c->g.s1 = c->g.Lh;
    c->g.s2 = c->g.Lh * L1;
    c->g.s3 = c->g.Lh * L1 * L2;
    c->g.V = V;
    c->g.Vh = (int)(V / 2);
    c->sh = c->g.s3;
    c->nvec = 3 * (size_t)(V / 2);
    c->max_blocks = (size_t)V / 64 + 4096;
    c->nsm = 148;
    c->recon = 18;
    c->check_every = 8;
    c->timeout_ms = 20000;
    c->use_graph = 1;
    c->fuse_sync = nranks == 1 ? 1 : 0;  // see LQCD_SLAB_OPT_FUSE_SYNC: unvalidated across GPUs
    c->acquire = -1;

    size_t off = 0;
    const size_t vec_bytes = align_up(c->nvec * sizeof(cplx));
    c->off_gauge = off;     off += align_up((size_t)V * 36 * sizeof(cplx));
    c->off_gghost = off;    off += align_up(2 * 9 * (size_t)c->sh * sizeof(cplx));
    c->off_r = off;         off += vec_bytes;
    c->off_p = off;         off += vec_bytes;
    c->off_t = off;         off += vec_bytes;
    c->off_sc = off;        off += align_up(sizeof(CgScalars));
    c->off_ss = off;        off += align_up(sizeof(SlabScalars));
    c->off_ticket = off;    off += kAlign;
    c->off_partials = off;  off += align_up(c->max_blocks * sizeof(double));
    c->off_hist = off;      off += align_up((size_t)kHistCap * sizeof(double));
    const size_t vecf_bytes = align_up(c->nvec * sizeof(cplxf));
    c->off_gauge_f = off;   off += align_up((size_t)V * 36 * sizeof(cplxf));
    c->off_gghost_f = off;  off += align_up(2 * 9 * (size_t)c->sh * sizeof(cplxf));
    c->off_xf = off;        off += vecf_bytes;
    c->off_rf = off;        off += vecf_bytes;
    c->off_pf = off;        off += vecf_bytes;
    c->off_tf = off;        off += vecf_bytes;
    c->ws_needed = off;

    off = 0;
    c->mb_word = off;   off += align_up(2 * LQCD_SLAB_MAX_RANKS * 4 * sizeof(unsigned long long));
    c->mb_ghost = off;  off += align_up(2 * 2 * 3 * (size_t)c->sh * sizeof(cplx));
    c->mb_needed = off;
    *out = c;
    return LQCD_OK;
}

int lqcd_slab_destroy(lqcd_slab* s)
{
    if (!s) return LQCD_EARG;
    if (s->host_ready) {
        cudaFreeHost(s->h_sc);
        cudaFreeHost(s->h_ss);
        cudaEventDestroy(s->ev[0]);
        cudaEventDestroy(s->ev[1]);
    }
    free(s);
    return LQCD_OK;
}

size_t lqcd_slab_workspace_bytes(const lqcd_slab* s) { return s ? s->ws_needed : 0; }
size_t lqcd_slab_mailbox_bytes(const lqcd_slab* s) { return s ? s->mb_needed : 0; }

int lqcd_slab_set_memory(lqcd_slab* s, void* workspace_dev, size_t workspace_bytes, void* mailbox_dev, size_t mailbox_bytes,
                         void* cuda_stream)
{
    if (!s) return LQCD_EARG;
    if (!workspace_dev || !mailbox_dev) return fail(s, LQCD_EARG, "null workspace or mailbox pointer");
    if (((uintptr_t)workspace_dev) % kAlign || ((uintptr_t)mailbox_dev) % kAlign)
        return fail(s, LQCD_EARG, "workspace and mailbox must be 256-byte aligned");
    if (workspace_bytes < s->ws_needed)
        return fail(s, LQCD_ENOMEM, "workspace too small: %zu bytes given, %zu needed", workspace_bytes, s->ws_needed);
    if (mailbox_bytes < s->mb_needed)
        return fail(s, LQCD_ENOMEM, "mailbox too small: %zu bytes given, %zu needed", mailbox_bytes, s->mb_needed);
    int ndev = 0;
    SLAB_CUDA(cudaGetDeviceCount(&ndev));
    if (ndev < 1) return fail(s, LQCD_ECUDA, "no CUDA device");
    cudaPointerAttributes at;
    SLAB_CUDA(cudaPointerGetAttributes(&at, workspace_dev));
    if (at.type != cudaMemoryTypeDevice) return fail(s, LQCD_EARG, "workspace is not device memory");
    s->device = at.device;
    SLAB_CUDA(cudaSetDevice(s->device));
    int rc = ensure_host(s);
    if (rc) return rc;
    int nsm = 0;
    SLAB_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, s->device));
    if (nsm > 0) s->nsm = nsm;
    s->ws = (char*)workspace_dev;
    s->mb = (char*)mailbox_dev;
    s->stream = (cudaStream_t)cuda_stream;
    s->memory_set = true;
    s->connected = false;
    s->gauge_loaded = false;
    s->gauge_f_ready = false;
    s->seq = 0;
    SLAB_CUDA(cudaMemsetAsync(s->ws + s->off_sc, 0, align_up(sizeof(CgScalars)) + align_up(sizeof(SlabScalars)) + kAlign, s->stream));
    SLAB_CUDA(cudaMemsetAsync(s->mb, 0, s->mb_ghost, s->stream));  // the tagged words (tag 0 = no synchronisation point)
    SLAB_CUDA(cudaStreamSynchronize(s->stream));
    return LQCD_OK;
}

int lqcd_slab_connect(lqcd_slab* s, void* const* peer_mailboxes)
{
    if (!s) return LQCD_EARG;
    if (!s->memory_set) return fail(s, LQCD_ESTATE, "memory not set (call lqcd_slab_set_memory)");
    if (!peer_mailboxes) return fail(s, LQCD_EARG, "peer_mailboxes is null");
    for (int r = 0; r < s->nranks; ++r)
        if (!peer_mailboxes[r]) return fail(s, LQCD_EARG, "mailbox of rank %d is null", r);
    if (peer_mailboxes[s->rank] != (void*)s->mb) return fail(s, LQCD_EARG, "peer_mailboxes[rank] must be the own mailbox");
    // Which device holds each peer's mailbox?  One on another GPU switches the system-scope release / acquire of the
    // synchronisation points on (slab_sync.cuh).  A pointer the runtime cannot place is treated as remote.
    s->peers_remote = false;
    for (int r = 0; r < s->nranks; ++r) {
        cudaPointerAttributes at;
        const cudaError_t e = cudaPointerGetAttributes(&at, peer_mailboxes[r]);
        if (e != cudaSuccess) (void)cudaGetLastError();
        if (e != cudaSuccess || at.type != cudaMemoryTypeDevice || at.device != s->device) s->peers_remote = true;
    }
    for (int r = 0; r < s->nranks; ++r) s->peer[r] = (char*)peer_mailboxes[r];
    s->connected = true;
    return LQCD_OK;
}

int lqcd_slab_set_option(lqcd_slab* s, int option, int value)
{
    if (!s) return LQCD_EARG;
    if (option == LQCD_SLAB_OPT_RECONSTRUCT) {
        if (value != 18 && value != 12) return fail(s, LQCD_EARG, "reconstruct must be 18 or 12");
        if (value != s->recon) s->gauge_loaded = s->gauge_f_ready = false;
        s->recon = value;
        return LQCD_OK;
    }
    if (option == LQCD_SLAB_OPT_CHECK_EVERY) {
        if (value < 1 || value > 1024) return fail(s, LQCD_EARG, "check_every must be in 1..1024");
        s->check_every = value;
        return LQCD_OK;
    }
    if (option == LQCD_SLAB_OPT_TIMEOUT_MS) {
        if (value < 1 || value > 600000) return fail(s, LQCD_EARG, "timeout must be in 1..600000 ms");
        s->timeout_ms = value;
        return LQCD_OK;
    }
    if (option == LQCD_SLAB_OPT_FUSE_SYNC) {
        if (value != 0 && value != 1) return fail(s, LQCD_EARG, "fuse_sync must be 0 or 1");
        s->fuse_sync = value;
        return LQCD_OK;
    }
    if (option == LQCD_SLAB_OPT_ACQUIRE) {
        if (value < -1 || value > 1) return fail(s, LQCD_EARG, "acquire must be -1 (auto), 0 or 1");
        s->acquire = value;
        return LQCD_OK;
    }
    if (option == LQCD_SLAB_OPT_GRAPH) {
        if (value != 0 && value != 1) return fail(s, LQCD_EARG, "graph must be 0 or 1");
        s->use_graph = value;
        return LQCD_OK;
    }
    return fail(s, LQCD_EARG, "unknown option %d", option);
}

int lqcd_slab_load_gauge(lqcd_slab* s, const double* u_local_dev, const double* u3_below_dev)
{
    if (!s) return LQCD_EARG;
    if (!s->memory_set) return fail(s, LQCD_ESTATE, "memory not set (call lqcd_slab_set_memory)");
    if (!u_local_dev || !u3_below_dev) return fail(s, LQCD_EARG, "null gauge pointer");
    SLAB_CUDA(cudaSetDevice(s->device));
    const size_t V = (size_t)s->g.V;
    const unsigned int grid = blocks_for(V, kReorderTile);
    const unsigned int ggrid = blocks_for(18 * (size_t)s->sh, 256);
    if (s->recon == 12) {
        gauge_reorder_kernel<256, kReorderTile, 12, cplx><<<grid, 256, 0, s->stream>>>((const cplx*)u_local_dev, s->gauge(),
                                                                                       (size_t)s->g.Vh);
        SLAB_LAUNCH_CHECK();
        slab_ghost_links_kernel<12, cplx><<<ggrid, 256, 0, s->stream>>>((const cplx*)u3_below_dev, s->gghost(), (size_t)s->sh);
    } else {
        gauge_reorder_kernel<256, kReorderTile, 18, cplx><<<grid, 256, 0, s->stream>>>((const cplx*)u_local_dev, s->gauge(),
                                                                                       (size_t)s->g.Vh);
        SLAB_LAUNCH_CHECK();
        slab_ghost_links_kernel<18, cplx><<<ggrid, 256, 0, s->stream>>>((const cplx*)u3_below_dev, s->gghost(), (size_t)s->sh);
    }
    SLAB_LAUNCH_CHECK();
    s->gauge_loaded = true;
    s->gauge_f_ready = false;
    return LQCD_OK;
}

// ---- group calls
int lqcd_slab_dslash_group(lqcd_slab* const* slabs, int n, int out_parity, const double* const* in_dev, double* const* out_dev)
{
    const Group G = { slabs, n };
    int rc = group_check(G, true);
    if (rc) return rc;
    lqcd_slab* s = slabs[0];
    if (!in_dev || !out_dev) return fail(s, LQCD_EARG, "null pointer array");
    if (out_parity != LQCD_EVEN && out_parity != LQCD_ODD) return fail(s, LQCD_EARG, "bad parity %d", out_parity);
    for (int r = 0; r < n; ++r)
        if (!in_dev[r] || !out_dev[r] || in_dev[r] == out_dev[r]) return fail(s, LQCD_EARG, "null or aliased vector of rank %d", r);
    return group_dslash(G, out_parity, (const cplx* const*)in_dev, (cplx* const*)out_dev);
}

int lqcd_slab_apply_MdagM_group(lqcd_slab* const* slabs, int n, double mass, const double* const* in_dev, double* const* out_dev)
{
    const Group G = { slabs, n };
    int rc = group_check(G, true);
    if (rc) return rc;
    lqcd_slab* s = slabs[0];
    if (!in_dev || !out_dev) return fail(s, LQCD_EARG, "null pointer array");
    for (int r = 0; r < n; ++r)
        if (!in_dev[r] || !out_dev[r] || in_dev[r] == out_dev[r]) return fail(s, LQCD_EARG, "null or aliased vector of rank %d", r);
    return group_MdagM(G, mass, (const cplx* const*)in_dev, (cplx* const*)out_dev);
}

int lqcd_slab_cg_solve_group(lqcd_slab* const* slabs, int n, double mass, double tol, int maxiter, const double* const* b_dev,
                             double* const* x_dev, int* iters, double* true_residual)
{
    const Group G = { slabs, n };
    int rc = group_check(G, true);
    if (rc) return rc;
    lqcd_slab* s = slabs[0];
    if (!b_dev || !x_dev || !iters || !true_residual) return fail(s, LQCD_EARG, "null pointer argument");
    if (!(tol >= 0.0) || maxiter < 0) return fail(s, LQCD_EARG, "tol must be >= 0 and maxiter >= 0");
    for (int r = 0; r < n; ++r)
        if (!b_dev[r] || !x_dev[r] || b_dev[r] == x_dev[r]) return fail(s, LQCD_EARG, "null or aliased vector of rank %d", r);
    return group_cg(G, mass, tol, maxiter, (const cplx* const*)b_dev, (cplx* const*)x_dev, iters, true_residual);
}

// ---- one rank per process: the n = 1 group whose peers live elsewhere
int lqcd_slab_dslash(lqcd_slab* s, int out_parity, const double* in_dev, double* out_dev)
{
    int rc = single_check(s, true);
    if (rc) return rc;
    if (!in_dev || !out_dev || in_dev == out_dev) return fail(s, LQCD_EARG, "null or aliased vector");
    if (out_parity != LQCD_EVEN && out_parity != LQCD_ODD) return fail(s, LQCD_EARG, "bad parity %d", out_parity);
    lqcd_slab* one[1] = { s };
    const Group G = { one, 1 };
    const cplx* in[1] = { (const cplx*)in_dev };
    cplx* out[1] = { (cplx*)out_dev };
    return group_dslash(G, out_parity, in, out);
}

int lqcd_slab_apply_MdagM(lqcd_slab* s, double mass, const double* in_dev, double* out_dev)
{
    int rc = single_check(s, true);
    if (rc) return rc;
    if (!in_dev || !out_dev || in_dev == out_dev) return fail(s, LQCD_EARG, "null or aliased vector");
    lqcd_slab* one[1] = { s };
    const Group G = { one, 1 };
    const cplx* in[1] = { (const cplx*)in_dev };
    cplx* out[1] = { (cplx*)out_dev };
    return group_MdagM(G, mass, in, out);
}

int lqcd_slab_cg_solve(lqcd_slab* s, double mass, double tol, int maxiter, const double* b_dev, double* x_dev, int* iters,
                       double* true_residual)
{
    int rc = single_check(s, true);
    if (rc) return rc;
    if (!b_dev || !x_dev || !iters || !true_residual || b_dev == x_dev) return fail(s, LQCD_EARG, "null or aliased argument");
    if (!(tol >= 0.0) || maxiter < 0) return fail(s, LQCD_EARG, "tol must be >= 0 and maxiter >= 0");
    lqcd_slab* one[1] = { s };
    const Group G = { one, 1 };
    const cplx* b[1] = { (const cplx*)b_dev };
    cplx* x[1] = { (cplx*)x_dev };
    return group_cg(G, mass, tol, maxiter, b, x, iters, true_residual);
}

int lqcd_slab_cg_solve_mixed_group(lqcd_slab* const* slabs, int n, double mass, double tol, int maxiter, double delta,
                                   const double* const* b_dev, double* const* x_dev, int* iters, int* reliable_updates,
                                   double* true_residual)
{
    const Group G = { slabs, n };
    int rc = group_check(G, true);
    if (rc) return rc;
    lqcd_slab* s = slabs[0];
    if (!b_dev || !x_dev || !iters || !reliable_updates || !true_residual) return fail(s, LQCD_EARG, "null pointer argument");
    if (!(tol >= 0.0) || maxiter < 0) return fail(s, LQCD_EARG, "tol must be >= 0 and maxiter >= 0");
    if (!(delta > 0.0 && delta < 1.0)) return fail(s, LQCD_EARG, "delta must be in (0,1)");
    for (int r = 0; r < n; ++r)
        if (!b_dev[r] || !x_dev[r] || b_dev[r] == x_dev[r]) return fail(s, LQCD_EARG, "null or aliased vector of rank %d", r);
    return group_cg_mixed(G, mass, tol, delta, maxiter, (const cplx* const*)b_dev, (cplx* const*)x_dev, iters, reliable_updates,
                          true_residual);
}

int lqcd_slab_cg_solve_mixed(lqcd_slab* s, double mass, double tol, int maxiter, double delta, const double* b_dev, double* x_dev,
                             int* iters, int* reliable_updates, double* true_residual)
{
    int rc = single_check(s, true);
    if (rc) return rc;
    if (!b_dev || !x_dev || !iters || !reliable_updates || !true_residual || b_dev == x_dev)
        return fail(s, LQCD_EARG, "null or aliased argument");
    if (!(tol >= 0.0) || maxiter < 0) return fail(s, LQCD_EARG, "tol must be >= 0 and maxiter >= 0");
    if (!(delta > 0.0 && delta < 1.0)) return fail(s, LQCD_EARG, "delta must be in (0,1)");
    lqcd_slab* one[1] = { s };
    const Group G = { one, 1 };
    const cplx* b[1] = { (const cplx*)b_dev };
    cplx* x[1] = { (cplx*)x_dev };
    return group_cg_mixed(G, mass, tol, delta, maxiter, b, x, iters, reliable_updates, true_residual);
}

// ---- CUDA IPC: mailboxes across processes
int lqcd_slab_ipc_export(lqcd_slab* s, unsigned char handle[64], size_t* offset)
{
    if (!s) return LQCD_EARG;
    if (!s->memory_set) return fail(s, LQCD_ESTATE, "memory not set (call lqcd_slab_set_memory)");
    if (!handle || !offset) return fail(s, LQCD_EARG, "null pointer argument");
    static_assert(sizeof(cudaIpcMemHandle_t) == 64, "the ABI carries IPC handles as 64 bytes");
    SLAB_CUDA(cudaSetDevice(s->device));
    // the handle names the whole allocation the mailbox lies in; find its base through the driver
    typedef int (*AddressRangeFn)(unsigned long long*, size_t*, unsigned long long);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    SLAB_CUDA(cudaGetDriverEntryPoint("cuMemGetAddressRange", &fn, cudaEnableDefault, &q));
    if (!fn || q != cudaDriverEntryPointSuccess) return fail(s, LQCD_ECUDA, "cuMemGetAddressRange is not available");
    unsigned long long base = 0;
    size_t size = 0;
    const int cr = ((AddressRangeFn)fn)(&base, &size, (unsigned long long)(uintptr_t)s->mb);
    if (cr != 0) return fail(s, LQCD_ECUDA, "cuMemGetAddressRange failed with CUresult %d", cr);
    cudaIpcMemHandle_t h;
    SLAB_CUDA(cudaIpcGetMemHandle(&h, (void*)(uintptr_t)base));
    memcpy(handle, &h, 64);
    *offset = (size_t)((unsigned long long)(uintptr_t)s->mb - base);
    return LQCD_OK;
}

int lqcd_slab_ipc_open(lqcd_slab* s, const unsigned char handle[64], size_t offset, void** peer_mailbox)
{
    if (!s) return LQCD_EARG;
    if (!handle || !peer_mailbox) return fail(s, LQCD_EARG, "null pointer argument");
    if (!s->memory_set) return fail(s, LQCD_ESTATE, "memory not set (call lqcd_slab_set_memory)");
    SLAB_CUDA(cudaSetDevice(s->device));
    cudaIpcMemHandle_t h;
    memcpy(&h, handle, 64);
    void* base = nullptr;
    SLAB_CUDA(cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess));
    *peer_mailbox = (char*)base + offset;
    return LQCD_OK;
}

int lqcd_slab_ipc_close(lqcd_slab* s, void* peer_mailbox, size_t offset)
{
    if (!s) return LQCD_EARG;
    if (!peer_mailbox) return fail(s, LQCD_EARG, "null pointer argument");
    SLAB_CUDA(cudaIpcCloseMemHandle((char*)peer_mailbox - offset));
    return LQCD_OK;
}

long long lqcd_slab_sync_points(const lqcd_slab* s) { return s ? (long long)s->seq : 0; }
long long lqcd_slab_kernel_launches(const lqcd_slab* s) { return s ? s->launches : 0; }
const char* lqcd_slab_last_error(const lqcd_slab* s) { return s ? s->err : "null slab"; }

}  // extern "C"
