// slab_sync.cuh -- the cross-rank synchronisation point of the time-slab decomposition
// (include/lqcd_slab.h): mailbox layout, signal, bounded wait, rank-ordered combine.  See
// slab_kernels.cuh for the protocol.
#pragma once
#include "reduce.cuh"

namespace lqcd {

constexpr int kSlabMaxRanks = 16;

// Mailbox of one rank (device memory the peers can address).  Byte offsets are computed on the host
// by lqcd_slab_create; every rank uses the same layout for the same lattice and rank count.
//
// Sums and the "I have arrived" signal travel as TAGGED WORDS: a double goes out as two 64-bit stores, each
// (sequence number << 32) | 32 bits of the value.  A 64-bit store is single-copy atomic, so a receiver that
// sees the tag of the synchronisation point it waits for has the data that belongs to it -- no fence between
// "slot" and "flag" on the sending side and none between "flag" and "slot" on the receiving side (round 1 paid
// two system-scope fences per synchronisation point for that order).  Every synchronisation point sends at
// least the two words of value 0, so the words are also the arrival signal for the ghost faces: those were made
// visible system-wide by the blocks that stored them BEFORE they took the reduction ticket (grid_sum_block), and
// the words are only sent after the last ticket.
struct SlabMailbox {
    unsigned long long* word;  // [2][R][4]  (seq & 1, source rank, {v0 lo, v0 hi, v1 lo, v1 hi})
    cplx* ghost;               // [2][2][3][sh]  (seq & 1, lo/hi, colour, site): the neighbours' boundary slices
};

struct SlabScalars {
    double part[2];          // this rank's partial sums, written by the producer kernel
    unsigned long long seq;  // synchronisation points this rank has completed (device-resident, so a
                             // captured CUDA graph of iterations can be replayed: no host-side number
                             // is baked into the kernels)
    int err;                 // 1 = a wait timed out
    int pad;
};

enum SlabOp {
    SLAB_OP_NONE = 0,    // halo only
    SLAB_OP_INIT = 1,    // total = <b,b>: start of the CG
    SLAB_OP_ALPHA = 2,   // total = <t,t>: alpha = rr / (m^2 pp + tt)
    SLAB_OP_UPDATE = 3,  // total = <r,r> after the update: beta, exit test
    SLAB_OP_PP = 4,      // total = <p,p>
    SLAB_OP_RES2 = 5,    // total = |b - A x|^2
    // mixed-precision solver on slabs (SURVEY.md 8(f) rows 3 + 4b; the scalar steps of reduce.cuh)
    SLAB_OP_INIT_MIXED = 6,    // totals = <b,b> (fp64 source), <ps,ps> (its fp32 copy)
    SLAB_OP_UPDATE_MIXED = 7,  // total = <rs,rs> after the fp32 update: may pause for a reliable update
    SLAB_OP_RELIABLE = 8       // total = <r,r> of the fp64 residual: resumes the paused iteration
};

struct SlabSyncArgs {
    int rank, nranks;
    int nvals;                                     // partial sums carried by this point (0, 1 or 2)
    SlabMailbox own;
    unsigned long long* peer_word[kSlabMaxRanks];  // rank r's word array
    SlabScalars* ss;
    CgScalars* sc;
    double* hist;
    int op;
    double m2, tol, delta;
    int maxiter;
    unsigned long long timeout_ns;
    int sys_fences;   // 1: a peer's mailbox is on another GPU (LQCD_SLAB_OPT_ACQUIRE): release before the words, acquire after
};

__device__ __forceinline__ void st_sys_u64(unsigned long long* p, unsigned long long v)
{
    asm volatile("st.relaxed.sys.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// Polling load.  Relaxed is enough: the data IS the word (tag and payload in one single-copy-atomic 64-bit value), and
// what the arrival of the words announces -- the ghost faces -- is read by a later kernel, never by this one.
__device__ __forceinline__ unsigned long long ld_relaxed_sys_u64(const unsigned long long* p)
{
    unsigned long long v;
    asm volatile("ld.relaxed.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

__device__ __forceinline__ void fence_acq_rel_sys() { asm volatile("fence.acq_rel.sys;" ::: "memory"); }

// thread r < nranks: this rank's partial(s), tagged with the number of the synchronisation point, into rank r's
// mailbox.  The faces were stored -- and fenced at system scope -- by the producer's blocks before this runs.
// own: the partial(s) in registers (fused tail), or null = read them from `part` (left there by the producer kernel).
//
// Memory model, sender side.  The face stores were made by OTHER blocks (each fenced them at system scope before
// its ticket atomic); this thread learnt of them through the ticket chain, which is ordered at DEVICE scope only
// (__threadfence in grid_sum_block's last block).  With every mailbox on this GPU that is the same thing.  With a
// peer on another GPU the words must not become visible THERE before the faces: a system-scope fence between
// "observed the last ticket" and "store the words" makes the chain cumulative at system scope (fence + relaxed
// store = a release of everything this thread has observed).  One fence in at most 16 threads of one block.
__device__ __forceinline__ void slab_signal(const SlabSyncArgs& a, unsigned long long seq, int r, const double* own = nullptr)
{
    if (a.sys_fences) fence_acq_rel_sys();
    unsigned long long* dst = a.peer_word[r] + ((seq & 1ull) * a.nranks + a.rank) * 4;
    const unsigned long long tag = seq << 32;
    const int nv = a.nvals > 0 ? a.nvals : 1;  // a point without a sum still announces itself
    for (int k = 0; k < nv; ++k) {
        const unsigned long long bits = a.nvals > 0 ? (unsigned long long)__double_as_longlong(own ? own[k] : a.ss->part[k]) : 0ull;
        st_sys_u64(dst + 2 * k, tag | (bits & 0xffffffffull));
        st_sys_u64(dst + 2 * k + 1, tag | (bits >> 32));
    }
}

__device__ __forceinline__ unsigned long long slab_now_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// thread r < nranks waits (bounded) for rank r's words of this synchronisation point and returns rank r's
// values in val[]; false on a timeout.
__device__ __forceinline__ bool slab_wait(const SlabSyncArgs& a, unsigned long long seq, int r, double val[2])
{
    const unsigned long long* src = a.own.word + ((seq & 1ull) * a.nranks + r) * 4;
    const unsigned long long tag = (seq << 32) >> 32;
    const int nv = a.nvals > 0 ? a.nvals : 1;
    unsigned long long t0 = 0;
    val[0] = val[1] = 0.0;
    for (int k = 0; k < nv; ++k) {
        unsigned long long lo, hi;
        for (;;) {
            lo = ld_relaxed_sys_u64(src + 2 * k);
            hi = ld_relaxed_sys_u64(src + 2 * k + 1);
            if ((lo >> 32) == tag && (hi >> 32) == tag) break;
            if (t0 == 0) t0 = slab_now_ns();
            if (slab_now_ns() - t0 > a.timeout_ns) return false;
            __nanosleep(100);
        }
        val[k] = __longlong_as_double((long long)((hi << 32) | (lo & 0xffffffffull)));
    }
    // Receiver side.  The sums need no ordering (the data is the word).  The ghost faces the words announce are read
    // by the NEXT kernel of this stream; that the peer's face stores are visible to it rests, without a fence, on this
    // GPU's L2 being the point of coherence of its own memory.  With a peer on another GPU the relaxed poll is followed
    // by a system-scope fence (relaxed load + fence = acquire), which pairs with the sender's release above; the kernel
    // boundary then carries the order to the next kernel's loads.
    if (a.sys_fences) fence_acq_rel_sys();
    return true;
}

// one thread: add the ranks' values in rank order, run the scalar step, count the synchronisation point.
__device__ __forceinline__ void slab_combine(const SlabSyncArgs& a, unsigned long long seq, bool timed_out, const double (*vals)[2])
{
    a.ss->seq = seq;
    if (timed_out) {  // a peer never arrived: stop the solver instead of hanging the device
        a.ss->err = 1;
        a.sc->done = 1;
        return;
    }
    double total[2] = { 0.0, 0.0 };
    for (int q = 0; q < a.nranks; ++q)
        for (int k = 0; k < a.nvals; ++k) total[k] += vals[q][k];
    CgScalars* sc = a.sc;
    switch (a.op) {
    case SLAB_OP_INIT: {
        const double bb = total[0];
        sc->rr = bb;
        sc->rr_new = bb;
        sc->bb = bb;
        sc->pp = bb;
        sc->tt = 0.0;
        sc->alpha = 0.0;
        sc->beta = 0.0;
        sc->thresh = a.tol * a.tol * bb;
        sc->res2 = 0.0;
        sc->iter = 0;
        sc->maxiter = a.maxiter;
        sc->done = (bb == 0.0 || a.maxiter <= 0) ? 1 : 0;
        sc->pause = 0;
        sc->nupd = 0;
        a.hist[0] = bb;
        break;
    }
    case SLAB_OP_INIT_MIXED: {
        const double bb = total[0];
        sc->rr = bb;
        sc->rr_new = bb;
        sc->bb = bb;
        sc->pp = total[1];
        sc->tt = 0.0;
        sc->alpha = 0.0;
        sc->beta = 0.0;
        sc->thresh = a.tol * a.tol * bb;
        sc->res2 = 0.0;
        sc->rmax = sqrt(bb);
        sc->delta = a.delta;
        sc->iter = 0;
        sc->maxiter = a.maxiter;
        sc->done = (bb == 0.0 || a.maxiter <= 0) ? 1 : 0;
        sc->pause = 0;
        sc->nupd = 0;
        a.hist[0] = bb;
        break;
    }
    case SLAB_OP_ALPHA:
        if (sc->done | sc->pause) break;  // the producer was a no-op: `part` is stale
        sc->tt = total[0];
        sc->alpha = sc->rr / (a.m2 * sc->pp + total[0]);
        break;
    case SLAB_OP_UPDATE:
        if (sc->done) break;
        cg_after_update(sc, a.hist, total[0]);
        break;
    case SLAB_OP_UPDATE_MIXED:
        if (sc->done | sc->pause) break;
        cg_after_update_mixed(sc, a.hist, total[0]);
        break;
    case SLAB_OP_RELIABLE:
        cg_after_reliable(sc, a.hist, total[0]);
        break;
    case SLAB_OP_PP:
        if (sc->done | sc->pause) break;
        sc->pp = total[0];
        break;
    case SLAB_OP_RES2:
        sc->res2 = total[0];
        break;
    default:
        break;
    }
}

// signal + bounded wait + combine by the threads of one block (at least nranks of them): the body of every form
// of a synchronisation point.  do_signal = false: the signal was sent by an earlier launch (group calls).
// seq_done = the points this rank has completed (a.ss->seq, read by the caller); own: see slab_signal.
__device__ __forceinline__ void slab_sync_point(const SlabSyncArgs& a, bool do_signal, unsigned long long seq_done, const double* own = nullptr)
{
    __shared__ int sp_timed_out;
    __shared__ double sp_vals[kSlabMaxRanks][2];
    const unsigned long long seq = seq_done + 1;
    if (threadIdx.x == 0) sp_timed_out = 0;
    __syncthreads();
    if ((int)threadIdx.x < a.nranks) {
        if (do_signal) slab_signal(a, seq, threadIdx.x, own);
        double v[2];
        if (!slab_wait(a, seq, threadIdx.x, v)) sp_timed_out = 1;
        sp_vals[threadIdx.x][0] = v[0];
        sp_vals[threadIdx.x][1] = v[1];
    }
    __syncthreads();
    if (threadIdx.x == 0) slab_combine(a, seq, sp_timed_out != 0, sp_vals);
}

// The whole synchronisation point run by the LAST block of a producer kernel (`total` = this rank's partial sum,
// known to every thread of that block; seq_done was read while the partials were being added): what a rank that
// drives only its own slab uses instead of separate launches -- the halo exchange, the all-reduce and the scalar step
// of the CG then cost no kernel boundary at all.  Every block of the producer that stored faces has fenced them at
// system scope before taking the reduction ticket, so they are visible to a peer that sees the words.
template <int BLOCK>
__device__ __forceinline__ void slab_sync_tail(const SlabSyncArgs& a, double total, unsigned long long seq_done)
{
    const double own[2] = { total, 0.0 };
    slab_sync_point(a, true, seq_done, own);
}

}  // namespace lqcd
