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
    double aux;       // scratch sum for the stand-alone norm kernel
    int iter;         // completed iterations
    int done;         // 1 once converged (or b = 0): later iterations become no-ops
    int maxiter;
    int pad;
};

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
