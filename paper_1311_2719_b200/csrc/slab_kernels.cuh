// slab_kernels.cuh -- kernels of the time-slab decomposition (
// include/lqcd_slab.h) that are not Dslash: the vector kernels with the face stores fused in,
// and the stand-alone kernels of a cross-rank synchronisation point (slab_sync.cuh has its pieces).
//
// A synchronisation point, number `seq` (1, 2, 3, ... since lqcd_slab_connect, the same on every rank
// because every rank makes the same sequence of calls):
//   producer kernel   writes its vector, stores the two boundary time-slices of that vector into the
//                     neighbour ranks' ghost faces (buffer seq & 1) through peer memory, and leaves
//                     this rank's partial sum(s) in `part`;
//   slab_signal       thread r: stores `part`, as 64-bit words tagged with seq, into rank r's mailbox
//                     [seq & 1][me] (slab_sync.cuh: the tag makes a separate flag and its fences unnecessary);
//   slab_wait_combine thread r: waits (bounded) for rank r's words of this seq in the own mailbox; then one
//                     thread adds the values in RANK ORDER -- every rank adds the same numbers in the
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

static __global__ void slab_wait_combine_kernel(const SlabSyncArgs a) { slab_sync_point(a, false, a.ss->seq); }

// Both in one launch: what a rank that drives only its own slab enqueues (one process per GPU).
// Never used by a group of several slabs on one stream, where every signal must precede every wait.
static __global__ void slab_signal_wait_combine_kernel(const SlabSyncArgs a) { slab_sync_point(a, true, a.ss->seq); }


// Where the two boundary time-slices of a slab vector go: element (c, e) of local slice 0 into the
// lower neighbour's ghost_hi, of local slice T-1 into the upper neighbour's ghost_lo.
template <class C>
struct SlabPushT {
    C* lo;
    C* hi;
    int sh;       // sites of one parity in a time-slice
    int Vh;       // local sites of one parity
};
typedef SlabPushT<cplx> SlabPush;    // fp64 vectors
typedef SlabPushT<cplxf> SlabPushF;  // fp32 vectors of the mixed-precision solver (the same ghost areas, half used)

// The vector kernels walk the n = 3 Vh elements in a FACE-FIRST order: virtual index v < 6 sh is an element of one
// of the two boundary time-slices (face f = v / sh: colour f / 2, first or last slice), the rest is the interior.
// The first `face_blocks` blocks of the grid own the face elements, one per thread where the grid allows: they store
// into a neighbour's memory, must fence at system scope before they take the reduction ticket, and -- having a
// fraction of the work of an interior block -- do so while the interior blocks are still streaming (round 1: the
// fence sat on the kernel's tail, 28.6 us against 14.4 us for the same p-update without faces).
struct SlabVecPlan {
    unsigned int n, nface;  // elements, face elements (6 sh, or n if the slab has no interior); n = 3 Vh < 2^31
    int face_blocks;        // blocks [0, face_blocks) own the face elements, the others the interior
};

// The walk of one block: v = v0 + threadIdx.x, v0 + threadIdx.x + step, ... < v1 -- a grid-stride walk inside the
// block's group (faces or interior), so that at any moment the blocks of a group stream neighbouring addresses (one
// contiguous run per block, as in round 1, cost 8 us of the 23 us p-update at 32^4 in DRAM locality).
__device__ __forceinline__ void slab_vec_range(const SlabVecPlan& pl, int block, unsigned int& v0, unsigned int& v1, unsigned int& step)
{
    if (gridDim.x == 1) {  // a single block walks everything, faces first
        v0 = 0;
        v1 = pl.n;
        step = block;
    } else if ((int)blockIdx.x < pl.face_blocks) {
        v0 = blockIdx.x * block;
        v1 = pl.nface;
        step = pl.face_blocks * block;
    } else {
        v0 = pl.nface + (blockIdx.x - pl.face_blocks) * block;
        v1 = pl.n;
        step = (gridDim.x - pl.face_blocks) * block;
    }
}

// virtual index -> element index i = c Vh + e, and where (if anywhere) the element goes in the neighbours' ghosts.
// 32-bit arithmetic throughout: with 64-bit divisions this index computation, not memory, bounded the kernel
// (7 elements x 2 divisions per thread: 8 of the 23 us of the p-update at 32^4).
template <class C>
__device__ __forceinline__ unsigned int slab_vec_elem(const SlabPushT<C>& ph, const SlabVecPlan& pl, unsigned int v, C*& peer_dst)
{
    const unsigned int sh = (unsigned int)ph.sh, Vh = (unsigned int)ph.Vh;
    peer_dst = nullptr;
    if (v < pl.nface) {
        if (Vh == 2 * sh) {  // T = 2: every site lies on a face, plain order; slice 0 -> lo, slice 1 -> hi
            const unsigned int c = v / Vh, e = v - c * Vh;
            peer_dst = e < sh ? ph.lo + (size_t)(c * sh + e) : ph.hi + (size_t)(c * sh + (e - sh));
            return v;
        }
        const unsigned int f = v / sh, k = v - f * sh, c = f >> 1;
        if (f & 1) {
            peer_dst = ph.hi + (size_t)(c * sh + k);
            return c * Vh + (Vh - sh) + k;
        }
        peer_dst = ph.lo + (size_t)(c * sh + k);
        return c * Vh + k;
    }
    const unsigned int w = v - pl.nface, per = Vh - 2 * sh;
    const unsigned int c = w / per;
    return c * Vh + sh + (w - c * per);
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
                                                             cplx* __restrict__ r, cplx* __restrict__ p, SlabVecPlan pl,
                                                             SlabPush ph, SlabScalars* ss, ReduceScratch rs,
                                                             const SlabSyncArgs sy, int fused)
{
    double local = 0.0;
    bool wrote_peer = false;
    unsigned int v0, v1, step;
    slab_vec_range(pl, BLOCK, v0, v1, step);
    for (unsigned int v = v0 + threadIdx.x; v < v1; v += step) {
        cplx* dst;
        const size_t i = slab_vec_elem(ph, pl, v, dst);
        const cplx val = b[i];
        r[i] = val;
        p[i] = val;
        x[i] = cmake(0.0, 0.0);
        if (dst) {
            *dst = val;
            wrote_peer = true;
        }
        local += cnorm2(val);
    }
    if (fused)
        grid_sum_block<BLOCK>(local, wrote_peer, rs, [&sy]() { return sy.ss->seq; },
                              [&sy](double bb, unsigned long long sq) { slab_sync_tail<BLOCK>(sy, bb, sq); });
    else
        grid_sum<BLOCK>(local, rs, [ss](double bb) { ss->part[0] = bb; });
}

// S5 on a slab: p = r + beta p, partial <p,p>; the faces of the new p go to the neighbours.  C = cplx, or cplxf for
// the fp32 inner iteration of the mixed-precision solver (evaluated in fp64, rounded on store, the norm taken of
// the stored value: as cg_pupdate_kernel).
template <int BLOCK, class C>
__global__ void __launch_bounds__(BLOCK) slab_cg_pupdate_kernel(const C* __restrict__ r, C* __restrict__ p, SlabVecPlan pl,
                                                                SlabPushT<C> ph, const CgScalars* sc, SlabScalars* ss,
                                                                ReduceScratch rs, const SlabSyncArgs sy, int fused)
{
    if (sc->done | sc->pause) return;
    const double beta = sc->beta;
    double local = 0.0;
    bool wrote_peer = false;
    unsigned int v0, v1, step;
    slab_vec_range(pl, BLOCK, v0, v1, step);
    for (unsigned int v = v0 + threadIdx.x; v < v1; v += step) {
        C* dst;
        const size_t i = slab_vec_elem(ph, pl, v, dst);
        const double2 rv = to_d(r[i]);
        double2 pv = to_d(p[i]);
        pv.x = fma(beta, pv.x, rv.x);
        pv.y = fma(beta, pv.y, rv.y);
        const C ps = to_cplx(pv, (C*)0);
        p[i] = ps;
        if (dst) {
            *dst = ps;
            wrote_peer = true;
        }
        local += cnorm2(ps);
    }
    if (fused)
        grid_sum_block<BLOCK>(local, wrote_peer, rs, [&sy]() { return sy.ss->seq; },
                              [&sy](double pp, unsigned long long sq) { slab_sync_tail<BLOCK>(sy, pp, sq); });
    else
        grid_sum<BLOCK>(local, rs, [ss](double pp) { ss->part[0] = pp; });
}

// S6 of the mixed-precision solver on a slab (cg_init_mixed_kernel): x = 0 (fp64), xs = 0, rs = ps = fl32(b), partial
// <b,b> from the fp64 source and <ps,ps> from its fp32 copy; the faces of ps go to the neighbours.
template <int BLOCK>
__global__ void __launch_bounds__(BLOCK) slab_cg_init_mixed_kernel(const cplx* __restrict__ b, cplx* __restrict__ x,
                                                                   cplxf* __restrict__ xs, cplxf* __restrict__ rs_,
                                                                   cplxf* __restrict__ ps, SlabVecPlan pl, SlabPushF ph,
                                                                   SlabScalars* ss, ReduceScratch rs)
{
    double local[2] = { 0.0, 0.0 };
    unsigned int v0, v1, step;
    slab_vec_range(pl, BLOCK, v0, v1, step);
    for (unsigned int v = v0 + threadIdx.x; v < v1; v += step) {
        cplxf* dst;
        const size_t i = slab_vec_elem(ph, pl, v, dst);
        const cplx val = b[i];
        const cplxf vf = make_float2((float)val.x, (float)val.y);
        x[i] = cmake(0.0, 0.0);
        xs[i] = make_float2(0.f, 0.f);
        rs_[i] = vf;
        ps[i] = vf;
        if (dst) *dst = vf;
        local[0] += cnorm2(val);
        local[1] += cnorm2(vf);
    }
    grid_sum_n<BLOCK, 2>(local, rs, [ss](const double (&tot)[2]) {
        ss->part[0] = tot[0];
        ss->part[1] = tot[1];
    });
}

// U_3 of the time-slice below the slab: canonical [parity][sh][3][3] -> [parity][NC][sh].
template <int RECON, class C>
__global__ void slab_ghost_links_kernel(const cplx* __restrict__ u3, C* __restrict__ soa, size_t sh)
{
    constexpr int NC = RECON / 2;
    const size_t n = 2 * sh * NC;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const size_t parity = i / (sh * NC);
        const size_t rest = i - parity * sh * NC;
        const size_t k = rest / sh, f = rest - k * sh;
        soa[i] = to_cplx(u3[(parity * sh + f) * 9 + k], (C*)0);
    }
}

}  // namespace lqcd
