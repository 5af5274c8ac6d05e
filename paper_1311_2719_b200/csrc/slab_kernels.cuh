// slab_kernels.cuh -- kernels of the time-slab decomposition (
// include/lqcd_slab.h) that are not Dslash: the vector kernels with the face stores fused in,
// and the two tiny kernels of a cross-rank synchronisation point.
//
// A synchronisation point, number `seq` (1, 2, 3, ... since lqcd_slab_connect, the same on every rank
// because every rank makes the same sequence of calls):
//   producer kernel   writes its vector, stores the two boundary time-slices of that vector into the
//                     neighbour ranks' ghost faces (buffer seq & 1) through peer memory, and leaves
//                     this rank's partial sum(s) in `part`;
//   slab_signal       thread r: copies `part` into rank r's slot [seq & 1][me], fences at system scope,
//                     then stores flag[me] = seq in rank r's mailbox;
//   slab_wait_combine thread r: waits (bounded) until flag[r] >= seq in the own mailbox; then one
//                     thread adds the slots in RANK ORDER -- every rank adds the same numbers in the
//                     same order, so all ranks hold bit-identical scalars and take the same exit
//                     decision -- and runs the scalar step of the CG.
// Buffers alternate with seq & 1: a rank can be at most one synchronisation point ahead of a peer
// that has not read its faces/slots yet, never two (it needs that peer's next signal to go on).
// The paper instead gathers the WHOLE vector through the host every iteration.
#pragma once
#include "cg_kernels.cuh"

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
    double part[2];  // this rank's partial sums, written by the producer kernel
    int err;         // 1 = a wait timed out
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
    unsigned long long seq;
    int nvals;                                  // partial sums carried by this point (0, 1 or 2)
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

static __global__ void slab_signal_kernel(const SlabSyncArgs a)
{
    const int r = threadIdx.x;
    if (r >= a.nranks) return;
    double* dst = a.peer_slot[r] + ((a.seq & 1ull) * a.nranks + a.rank) * 2;
    for (int k = 0; k < a.nvals; ++k) dst[k] = a.ss->part[k];
    __threadfence_system();
    *(volatile unsigned long long*)(a.peer_flag[r] + a.rank) = a.seq;
}

__device__ __forceinline__ unsigned long long slab_now_ns()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}

static __global__ void slab_wait_combine_kernel(const SlabSyncArgs a)
{
    __shared__ int timed_out;
    const int r = threadIdx.x;
    if (r == 0) timed_out = 0;
    __syncthreads();
    if (r < a.nranks) {
        const volatile unsigned long long* f = a.own.flag + r;
        if (*f < a.seq) {
            const unsigned long long t0 = slab_now_ns();
            while (*f < a.seq) {
                if (slab_now_ns() - t0 > a.timeout_ns) {
                    timed_out = 1;
                    break;
                }
                __nanosleep(200);
            }
        }
    }
    __syncthreads();
    if (r != 0) return;
    if (timed_out) {  // a peer never arrived: stop the solver instead of hanging the device
        a.ss->err = 1;
        a.sc->done = 1;
        return;
    }
    __threadfence_system();
    double total[2] = { 0.0, 0.0 };
    const volatile double* s = a.own.slot + (a.seq & 1ull) * a.nranks * 2;
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

// Where the two boundary time-slices of a slab vector go: element (c, e) of local slice 0 into the
// lower neighbour's ghost_hi, of local slice T-1 into the upper neighbour's ghost_lo.
struct SlabPush {
    cplx* lo;
    cplx* hi;
    int sh;       // sites of one parity in a time-slice
    int Vh;       // local sites of one parity
};

__device__ __forceinline__ void slab_push_elem(const SlabPush& ph, size_t i, cplx v)
{
    const size_t c = i / (size_t)ph.Vh;
    const size_t e = i - c * (size_t)ph.Vh;
    if (e < (size_t)ph.sh) ph.lo[c * ph.sh + e] = v;
    if (e >= (size_t)(ph.Vh - ph.sh)) ph.hi[c * ph.sh + (e - (size_t)(ph.Vh - ph.sh))] = v;
}

// Faces of a vector that no kernel of ours produced (a caller's input, or x before the final check).
template <int BLOCK>
__global__ void __launch_bounds__(BLOCK) slab_push_faces_kernel(const cplx* __restrict__ v, SlabPush ph)
{
    // elements (c, e) with e in the first or the last slice: 2 * 3 * sh of them
    const size_t n = 6 * (size_t)ph.sh;
    for (size_t j = (size_t)blockIdx.x * BLOCK + threadIdx.x; j < n; j += (size_t)gridDim.x * BLOCK) {
        const size_t face = j / (3 * (size_t)ph.sh);
        const size_t k = j - face * 3 * (size_t)ph.sh;
        const size_t c = k / ph.sh, f = k - c * ph.sh;
        if (face == 0)
            ph.lo[c * ph.sh + f] = v[c * (size_t)ph.Vh + f];
        else
            ph.hi[c * ph.sh + f] = v[c * (size_t)ph.Vh + (size_t)(ph.Vh - ph.sh) + f];
    }
}

// S6 on a slab: p = r = b, x = 0, partial <b,b>; the faces of p go to the neighbours.
template <int BLOCK>
__global__ void __launch_bounds__(BLOCK) slab_cg_init_kernel(const cplx* __restrict__ b, cplx* __restrict__ x,
                                                             cplx* __restrict__ r, cplx* __restrict__ p, size_t n,
                                                             SlabPush ph, SlabScalars* ss, ReduceScratch rs)
{
    double local = 0.0;
    for (size_t i = (size_t)blockIdx.x * BLOCK + threadIdx.x; i < n; i += (size_t)gridDim.x * BLOCK) {
        const cplx v = b[i];
        r[i] = v;
        p[i] = v;
        x[i] = cmake(0.0, 0.0);
        slab_push_elem(ph, i, v);
        local += cnorm2(v);
    }
    grid_sum<BLOCK>(local, rs, [ss](double bb) { ss->part[0] = bb; });
}

// S5 on a slab: p = r + beta p, partial <p,p>; the faces of the new p go to the neighbours.
template <int BLOCK>
__global__ void __launch_bounds__(BLOCK) slab_cg_pupdate_kernel(const cplx* __restrict__ r, cplx* __restrict__ p, size_t n,
                                                                SlabPush ph, const CgScalars* sc, SlabScalars* ss,
                                                                ReduceScratch rs)
{
    if (sc->done) return;
    const double beta = sc->beta;
    double local = 0.0;
    for (size_t i = (size_t)blockIdx.x * BLOCK + threadIdx.x; i < n; i += (size_t)gridDim.x * BLOCK) {
        const cplx rv = r[i];
        cplx pv = p[i];
        pv.x = fma(beta, pv.x, rv.x);
        pv.y = fma(beta, pv.y, rv.y);
        p[i] = pv;
        slab_push_elem(ph, i, pv);
        local += cnorm2(pv);
    }
    grid_sum<BLOCK>(local, rs, [ss](double pp) { ss->part[0] = pp; });
}

// U_3 of the time-slice below the slab: canonical [parity][sh][3][3] -> [parity][NC][sh].
template <int RECON>
__global__ void slab_ghost_links_kernel(const cplx* __restrict__ u3, cplx* __restrict__ soa, size_t sh)
{
    constexpr int NC = RECON / 2;
    const size_t n = 2 * sh * NC;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const size_t parity = i / (sh * NC);
        const size_t rest = i - parity * sh * NC;
        const size_t k = rest / sh, f = rest - k * sh;
        soa[i] = u3[(parity * sh + f) * 9 + k];
    }
}

}  // namespace lqcd
