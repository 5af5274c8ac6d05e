// slab_kernels.cuh -- kernels of the time-slab decomposition (
// include/lqcd_slab.h) that are not Dslash: the vector kernels with the face stores fused in,
// and the stand-alone kernels of a cross-rank synchronisation point (slab_sync.cuh has its pieces).
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
//   A rank that drives only its own slab runs signal + wait + combine in the LAST BLOCK of the producer
//   kernel (slab_sync_tail; no extra launch), or as one launch after producers that have no sum; a group
//   of slabs on one stream launches all signals, then all waits, so that no kernel ever spins.
// Buffers alternate with seq & 1: a rank can be at most one synchronisation point ahead of a peer
// that has not read its faces/slots yet, never two (it needs that peer's next signal to go on).
// The paper instead gathers the WHOLE vector through the host every iteration.
#pragma once
#include "cg_kernels.cuh"
#include "slab_sync.cuh"

namespace lqcd {

static __global__ void slab_signal_kernel(const SlabSyncArgs a)
{
    if ((int)threadIdx.x < a.nranks) slab_signal(a, a.ss->seq + 1, threadIdx.x);
}

static __global__ void slab_wait_combine_kernel(const SlabSyncArgs a)
{
    __shared__ int timed_out;
    const unsigned long long seq = a.ss->seq + 1;
    if (threadIdx.x == 0) timed_out = 0;
    __syncthreads();
    if ((int)threadIdx.x < a.nranks && !slab_wait(a, seq, threadIdx.x)) timed_out = 1;
    __syncthreads();
    if (threadIdx.x == 0) slab_combine(a, seq, timed_out != 0);
}

// Both in one launch: what a rank that drives only its own slab enqueues (one process per GPU).
// Never used by a group of several slabs on one stream, where every signal must precede every wait.
static __global__ void slab_signal_wait_combine_kernel(const SlabSyncArgs a)
{
    __shared__ int timed_out;
    const unsigned long long seq = a.ss->seq + 1;
    if (threadIdx.x == 0) timed_out = 0;
    __syncthreads();
    if ((int)threadIdx.x < a.nranks) {
        slab_signal(a, seq, threadIdx.x);
        if (!slab_wait(a, seq, threadIdx.x)) timed_out = 1;
    }
    __syncthreads();
    if (threadIdx.x == 0) slab_combine(a, seq, timed_out != 0);
}


// Where the two boundary time-slices of a slab vector go: element (c, e) of local slice 0 into the
// lower neighbour's ghost_hi, of local slice T-1 into the upper neighbour's ghost_lo.
struct SlabPush {
    cplx* lo;
    cplx* hi;
    int sh;       // sites of one parity in a time-slice
    int Vh;       // local sites of one parity
};

__device__ __forceinline__ bool slab_push_elem(const SlabPush& ph, size_t i, cplx v)
{
    const size_t c = i / (size_t)ph.Vh;
    const size_t e = i - c * (size_t)ph.Vh;
    const bool lo = e < (size_t)ph.sh, hi = e >= (size_t)(ph.Vh - ph.sh);
    if (lo) ph.lo[c * ph.sh + e] = v;
    if (hi) ph.hi[c * ph.sh + (e - (size_t)(ph.Vh - ph.sh))] = v;
    return lo || hi;
}

// The vector kernels give every block one contiguous run of elements (not a grid-stride walk), so only
// the few blocks whose run meets a boundary time-slice store into a neighbour's memory -- and only
// those pay for a system-scope fence.
__device__ __forceinline__ void slab_block_range(size_t n, size_t& i0, size_t& i1)
{
    const size_t per = (n + gridDim.x - 1) / gridDim.x;
    i0 = (size_t)blockIdx.x * per;
    i1 = i0 + per < n ? i0 + per : n;
    if (i0 > n) i0 = n;
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
                                                             SlabPush ph, SlabScalars* ss, ReduceScratch rs,
                                                             const SlabSyncArgs sy, int fused)
{
    double local = 0.0;
    bool wrote_peer = false;
    size_t i0, i1;
    slab_block_range(n, i0, i1);
    for (size_t i = i0 + threadIdx.x; i < i1; i += BLOCK) {
        const cplx v = b[i];
        r[i] = v;
        p[i] = v;
        x[i] = cmake(0.0, 0.0);
        wrote_peer |= slab_push_elem(ph, i, v);
        local += cnorm2(v);
    }
    if (fused)
        grid_sum_block<BLOCK>(local, wrote_peer, rs, [&sy](double bb) { slab_sync_tail<BLOCK>(sy, bb); });
    else
        grid_sum<BLOCK>(local, rs, [ss](double bb) { ss->part[0] = bb; });
}

// S5 on a slab: p = r + beta p, partial <p,p>; the faces of the new p go to the neighbours.
template <int BLOCK>
__global__ void __launch_bounds__(BLOCK) slab_cg_pupdate_kernel(const cplx* __restrict__ r, cplx* __restrict__ p, size_t n,
                                                                SlabPush ph, const CgScalars* sc, SlabScalars* ss,
                                                                ReduceScratch rs, const SlabSyncArgs sy, int fused)
{
    if (sc->done) return;
    const double beta = sc->beta;
    double local = 0.0;
    bool wrote_peer = false;
    size_t i0, i1;
    slab_block_range(n, i0, i1);
    for (size_t i = i0 + threadIdx.x; i < i1; i += BLOCK) {
        const cplx rv = r[i];
        cplx pv = p[i];
        pv.x = fma(beta, pv.x, rv.x);
        pv.y = fma(beta, pv.y, rv.y);
        p[i] = pv;
        wrote_peer |= slab_push_elem(ph, i, pv);
        local += cnorm2(pv);
    }
    if (fused)
        grid_sum_block<BLOCK>(local, wrote_peer, rs, [&sy](double pp) { slab_sync_tail<BLOCK>(sy, pp); });
    else
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
