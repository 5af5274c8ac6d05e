// reduce.cuh -- deterministic grid-wide sums without a host round trip.
//
// The paper reduces <r,r>, <ap,ap>, <p,p> with OpenACC reduction(+) clauses (PAPER.md:68-74,
// :85, :90) and keeps alpha/beta on the device.  Here every kernel that
// produces a vector also produces its norm: warp shuffles -> shared memory -> one partial per
// block -> the last block to finish (ticket counter) adds the partials in a fixed order and
// runs a small "finalise" functor that updates the CG scalars in device memory.  No floating
// point atomics: the result does not depend on block scheduling, so iteration counts are
// reproducible run to run.
#pragma once
#include "device_common.cuh"

namespace lqcd {

// CG scalars, device resident (the paper's alpha, betan, betad, alphan, alphad, nitcg).
struct CgScalars {
    double rr;        // <r,r> of the current residual (betad/alphan)
    double rr_new;    // <r,r> after the update (betan)
    double bb;        // <b,b>
    double pp;        // <p,p>
    double tt;        // <t,t>, t = D_oe p (staggered) or M p (Wilson)
    double alpha;     // rr / <p,Ap>
    double beta;      // rr_new / rr
    double thresh;    // tol^2 * bb
    double res2;      // |b - A x|^2 of the final check
    double aux;       // second sum of the two-sum kernels (|b|^2 of the full-system residual)
    double rmax;      // mixed precision: largest |r| since the last reliable update
    double delta;     // mixed precision: reliable-update threshold
    int iter;         // completed iterations
    int done;         // 1 once converged (or b = 0): later iterations become no-ops
    int maxiter;
    int pause;        // mixed precision: 1 = a reliable update is due; the fp32 iteration kernels are
                      // no-ops until the update sequence has run (it clears the flag)
    int nupd;         // mixed precision: reliable updates completed
    int xdue;         // Wilson solvers: 1 = the x += alpha p of the last iteration is still to be done by the
                      // vector kernel that follows the update of r (cg_xpupdate_kernel clears it)
    int pad[2];
};
static_assert(sizeof(CgScalars) == 128, "CgScalars is copied to the host as one 128-byte block");

struct ReduceScratch {
    double* partials;      // one per block
    unsigned int* ticket;  // zero between kernels
};

static constexpr int kHistCap = 65536;

// Scalar bookkeeping after x += alpha p, r -= alpha Ap (run by one thread of the last block):
// iteration count, history, beta = betan/betad and betad = betan, exit flag
// (relative rule, reading A6).
__device__ __forceinline__ void cg_after_update(CgScalars* sc, double* hist, double rr_new)
{
    const int it = sc->iter + 1;
    sc->iter = it;
    sc->rr_new = rr_new;
    if (it < kHistCap) hist[it] = rr_new;
    sc->beta = rr_new / sc->rr;
    sc->rr = rr_new;
    if (rr_new <= sc->thresh || it >= sc->maxiter) sc->done = 1;
}

// Mixed precision: after the fp32 update of xs and rs.  The reliable update
// is due when the iterated residual has fallen by `delta` below the largest one since the last
// update, or claims convergence; then the iteration pauses (beta and the p-update wait for the
// fp64 residual).  Otherwise as cg_after_update, except that convergence is never declared here.
__device__ __forceinline__ void cg_after_update_mixed(CgScalars* sc, double* hist, double rr_new)
{
    const int it = sc->iter + 1;
    sc->iter = it;
    sc->rr_new = rr_new;
    if (it < kHistCap) hist[it] = rr_new;
    const double rn = sqrt(rr_new);
    const bool update = rn < sc->delta * sc->rmax || rr_new <= sc->thresh;
    if (rn > sc->rmax) sc->rmax = rn;
    if (update) {
        sc->pause = 1;
    } else {
        sc->beta = rr_new / sc->rr;
        sc->rr = rr_new;
        if (it >= sc->maxiter) sc->done = 1;
    }
}

// After the fp64 residual r = b - A x of a reliable update: |r|^2 replaces the iterated value,
// convergence is decided on it, and the paused iteration resumes with beta from it.
__device__ __forceinline__ void cg_after_reliable(CgScalars* sc, double* hist, double rr_true)
{
    const int it = sc->iter;
    sc->rr_new = rr_true;
    if (it < kHistCap) hist[it] = rr_true;
    sc->rmax = sqrt(rr_true);
    sc->nupd += 1;
    sc->pause = 0;
    if (rr_true <= sc->thresh) {
        sc->done = 1;
    } else {
        sc->beta = rr_true / sc->rr;
        sc->rr = rr_true;
        if (it >= sc->maxiter) sc->done = 1;
    }
}

template <int BLOCK>
__device__ __forceinline__ double block_sum(double v)
{
    __shared__ double warp_part[BLOCK / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    __syncthreads();  // protect warp_part against a previous call
    if (lane == 0) warp_part[w] = v;
    __syncthreads();
    double s = 0.0;
    if (w == 0) {
        s = lane < BLOCK / 32 ? warp_part[lane] : 0.0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    }
    return s;  // valid in warp 0
}

// Every thread of every block calls this once with its local contribution.  `fin(total)` runs in
// thread 0 of the last block only.
template <int BLOCK, class Finalise>
__device__ __forceinline__ void grid_sum(double local, const ReduceScratch& rs, Finalise fin)
{
    __shared__ bool is_last;
    double s = block_sum<BLOCK>(local);
    if (threadIdx.x == 0) {
        rs.partials[blockIdx.x] = s;
        __threadfence();
        unsigned int t = atomicAdd(rs.ticket, 1u);
        is_last = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (is_last) {
        __threadfence();
        double acc = 0.0;
        for (unsigned int i = threadIdx.x; i < gridDim.x; i += BLOCK) acc += __ldcg(rs.partials + i);
        double total = block_sum<BLOCK>(acc);
        if (threadIdx.x == 0) {
            *rs.ticket = 0u;
            fin(total);
        }
    }
}

// As grid_sum, but `fin(total)` is called by EVERY thread of the last block (total broadcast): for
// finalisers that talk to other GPUs (slab_sync_tail).  `wrote_peer`: this thread stored into another
// GPU's memory; a block in which any thread did fences at SYSTEM scope before it takes the ticket
// (membar.sys in every block costs ~20 us on a 4096-block kernel, so only those blocks pay it).
template <int BLOCK, class Early, class Finalise>
__device__ __forceinline__ void grid_sum_block(double local, bool wrote_peer, const ReduceScratch& rs, Early early, Finalise fin)
{
    __shared__ bool is_last_b;
    __shared__ double total_b;
    const int any_peer = __syncthreads_or(wrote_peer ? 1 : 0);
    double s = block_sum<BLOCK>(local);
    if (threadIdx.x == 0) {
        rs.partials[blockIdx.x] = s;
        if (any_peer)
            __threadfence_system();
        else
            __threadfence();
        unsigned int t = atomicAdd(rs.ticket, 1u);
        is_last_b = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (is_last_b) {
        __threadfence();
        // what the finaliser will need from memory is asked for now, so that it arrives while the partials are added
        const auto e = early();
        double acc = 0.0;
        for (unsigned int i = threadIdx.x; i < gridDim.x; i += BLOCK) acc += __ldcg(rs.partials + i);
        double total = block_sum<BLOCK>(acc);
        if (threadIdx.x == 0) {
            *rs.ticket = 0u;
            total_b = total;
        }
        __syncthreads();
        fin(total_b, e);
    }
}

// The same for N sums at once (partials laid out [N][gridDim.x]); `fin(total[N])`.
template <int BLOCK, int N, class Finalise>
__device__ __forceinline__ void grid_sum_n(const double (&local)[N], const ReduceScratch& rs, Finalise fin)
{
    __shared__ bool is_last_n;
    double s[N];
#pragma unroll
    for (int k = 0; k < N; ++k) s[k] = block_sum<BLOCK>(local[k]);
    if (threadIdx.x == 0) {
#pragma unroll
        for (int k = 0; k < N; ++k) rs.partials[(size_t)k * gridDim.x + blockIdx.x] = s[k];
        __threadfence();
        unsigned int t = atomicAdd(rs.ticket, 1u);
        is_last_n = (t == gridDim.x - 1);
    }
    __syncthreads();
    if (is_last_n) {
        __threadfence();
        double total[N];
#pragma unroll
        for (int k = 0; k < N; ++k) {
            double acc = 0.0;
            for (unsigned int i = threadIdx.x; i < gridDim.x; i += BLOCK) acc += __ldcg(rs.partials + (size_t)k * gridDim.x + i);
            total[k] = block_sum<BLOCK>(acc);
        }
        if (threadIdx.x == 0) {
            *rs.ticket = 0u;
            fin(total);
        }
    }
}

}  // namespace lqcd
