// slab_sync.cuh -- the cross-rank synchronisation point of the time-slab decomposition
// (include/lqcd_slab.h): mailbox layout, signal, bounded wait, rank-ordered combine.  See
// slab_kernels.cuh for the protocol.
#pragma once
#include "reduce.cuh"

namespace lqcd {

constexpr int kSlabMaxRanks = 16;

// Mailbox of one rank (device memory the peers can address).  Byte offsets are computed on the host
// by slab_mailbox_layout(); every rank uses the same layout for the same lattice and rank count.
struct SlabMailbox {
    unsigned long long* flag;  // [R]        flag[src] = last synchronisation point src has signalled
    double* slot;              // [2][R][2]  partial sums of src at that point
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
    SLAB_OP_RES2 = 5     // total = |b - A x|^2
};

struct SlabSyncArgs {
    int rank, nranks;
    int nvals;                                     // partial sums carried by this point (0, 1 or 2)
    SlabMailbox own;
    unsigned long long* peer_flag[kSlabMaxRanks];  // rank r's flag array
    double* peer_slot[kSlabMaxRanks];              // rank r's slot array
    SlabScalars* ss;
    CgScalars* sc;
    double* hist;
    int op;
    double m2, tol;
    int maxiter;
    unsigned long long timeout_ns;
};

// thread r < nranks: this rank's partial(s) into rank r's slot, then (after a system-scope fence) the flag.
// The faces were stored by the producer kernel that precedes this one in the stream.
__device__ __forceinline__ void slab_signal(const SlabSyncArgs& a, unsigned long long seq, int r)
{
    double* dst = a.peer_slot[r] + ((seq & 1ull) * a.nranks + a.rank) * 2;
    for (int k = 0; k < a.nvals; ++k) dst[k] = a.ss->part[k];
    __threadfence_system();  // release: slots (and the producer's face stores) before the flag
    *(volatile unsigned long long*)(a.peer_flag[r] + a.rank) = seq;
}

__device__ __forceinline__ unsigned long long slab_now_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

// thread r < nranks waits (bounded) for rank r's flag; returns false on a timeout.
__device__ __forceinline__ bool slab_wait(const SlabSyncArgs& a, unsigned long long seq, int r)
{
    const volatile unsigned long long* f = a.own.flag + r;
    if (*f >= seq) return true;
    const unsigned long long t0 = slab_now_ns();
    while (*f < seq) {
        if (slab_now_ns() - t0 > a.timeout_ns) return false;
        __nanosleep(200);
    }
    return true;
}

// one thread: add the slots in rank order, run the scalar step, count the synchronisation point.
__device__ __forceinline__ void slab_combine(const SlabSyncArgs& a, unsigned long long seq, bool timed_out)
{
    a.ss->seq = seq;
    if (timed_out) {  // a peer never arrived: stop the solver instead of hanging the device
        a.ss->err = 1;
        a.sc->done = 1;
        return;
    }
    __threadfence_system();  // acquire: the flags before the slots and the ghost faces
    double total[2] = { 0.0, 0.0 };
    const volatile double* s = a.own.slot + (seq & 1ull) * a.nranks * 2;
    for (int q = 0; q < a.nranks; ++q)
        for (int k = 0; k < a.nvals; ++k) total[k] += s[q * 2 + k];
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
    case SLAB_OP_ALPHA:
        if (sc->done) break;  // the producer was a no-op: `part` is stale
        sc->tt = total[0];
        sc->alpha = sc->rr / (a.m2 * sc->pp + total[0]);
        break;
    case SLAB_OP_UPDATE:
        if (sc->done) break;
        cg_after_update(sc, a.hist, total[0]);
        break;
    case SLAB_OP_PP:
        if (sc->done) break;
        sc->pp = total[0];
        break;
    case SLAB_OP_RES2:
        sc->res2 = total[0];
        break;
    default:
        break;
    }
}

// The whole synchronisation point run by the LAST block of a producer kernel (`total` = this rank's
// partial sum, known to every thread of that block): what a rank that drives only its own slab uses
// instead of separate launches -- the halo exchange, the all-reduce and the scalar step of the CG
// then cost no kernel boundary at all.  Every block of the producer has fenced its face stores at
// system scope before taking the reduction ticket, so they are visible to a peer that sees the flag.
template <int BLOCK>
__device__ __forceinline__ void slab_sync_tail(const SlabSyncArgs& a, double total)
{
    __shared__ int tail_timed_out;
    const unsigned long long seq = a.ss->seq + 1;
    if (threadIdx.x == 0) {
        tail_timed_out = 0;
        a.ss->part[0] = total;
    }
    __syncthreads();
    if ((int)threadIdx.x < a.nranks) {
        slab_signal(a, seq, threadIdx.x);
        if (!slab_wait(a, seq, threadIdx.x)) tail_timed_out = 1;
    }
    __syncthreads();
    if (threadIdx.x == 0) slab_combine(a, seq, tail_timed_out != 0);
}

}  // namespace lqcd
