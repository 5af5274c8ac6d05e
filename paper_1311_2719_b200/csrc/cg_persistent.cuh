// cg_persistent.cuh -- the whole iteration loop of the staggered conjugate gradient (SURVEY.md 8(a) rows
// S1-S5; the paper's "do nx=1,niterc" loop) as ONE cooperative kernel.
//
// "The entire conjugate gradient routine runs on the GPU".  On lattices whose whole
// working set sits in the L2 (4^4, 16^4: BASELINE.json configs 1, 2) an iteration of the three-kernel
// solver is bounded by its three kernel boundaries, not by bytes: 17-26 us per iteration of which at most
// 12 us are hopping terms, even replayed from a CUDA graph.  Here the three phases of an iteration are
// separated by a grid-wide barrier inside one launch (a kernel synchronising with itself: co-residency of
// all its blocks is guaranteed by the cooperative launch), and the loop runs until the exit rule fires or
// `niter` iterations have been done.  No scalar goes to the host inside the loop; alpha, beta and the exit
// flag are evaluated redundantly -- and bit-identically -- by every block from the per-block partial sums.
//
// Arithmetic and summation order are EXACTLY those of the three-kernel path with 32-thread blocks
// (stag_dslash_kernel<SE_NORM, 32>, <SE_CGUPDATE, 32>, cg_pupdate_kernel<256>; 32 threads is what that path
// uses on the small lattices this kernel is for): one WARP of a 256-thread physical block is one "virtual
// block" of the hopping terms, the whole physical block one 256-element block of the p-update; they leave
// the same partial sums and add them in the same order.  The iterates are therefore bit-identical to
// lqcd_cg_solve's other modes at LQCD_OPT_STAG_BLOCK = 32 (tested), whatever the number of physical blocks.
// One physical block per SM at most (255 registers: every load of a hopping term is issued before its first
// use), at most 148 blocks in a barrier; lattices of up to 8 virtual blocks run in ONE block, where the
// barrier is __syncthreads and the links stay in L1 from iteration to iteration.
#pragma once
#include "stag_dslash.cuh"

namespace lqcd {

struct PersistArgs {
    Geom g;
    const cplx* gauge;   // [2][4][RECON/2][Vh]
    cplx* p;             // [3][Vh] even sites
    cplx* t;             // [3][Vh] odd sites (scratch)
    cplx* x;
    cplx* r;
    double m2;
    CgScalars* sc;
    double* hist;
    double* partials;    // 3 arrays: [nvb] Dslash-1, [nvb] Dslash-2, [vgrid] p-update
    unsigned int* bar;   // grid barrier: arrivals since the launch (the host zeroes it before every launch)
    int nvb;             // virtual blocks of the hopping terms: ceil(Vh / 32)
    int vgrid;           // virtual blocks of the p-update (256 elements each, strided like cg_pupdate_kernel)
    int niter;           // iterations this launch may run
};

// Link loads of the loop: ordinary L1-allocating loads -- a block re-reads the same links every iteration.  B200, CG ms
// at cfg 1 / cfg 2 (20 solves, two runs each): streaming (.cs, what the three-kernel path uses) 2.00 / 2.20-2.22,
// L2 only (.cg) 2.27 / 2.14, default 2.00 / 2.14-2.16 (profiles/r03_bench.md).
constexpr int kPersistLinks = LP_DEFAULT;
constexpr int kPersistBlock = 256;   // threads of a physical block = 8 virtual blocks of the hopping terms at a time
constexpr int kPersistSmemPartials = 2048;

// All blocks of the (cooperative) grid; `epoch` counts this block's barriers since the launch.  One release
// increment per block, then an acquire poll until all gridDim.x blocks of this epoch have arrived: stores made
// by any block before the barrier are visible to every block after it (to plain or .cg loads -- never the
// read-only path for data written inside this kernel).  A single block needs no more than __syncthreads.
__device__ __forceinline__ void grid_barrier(unsigned int* bar, unsigned int& epoch)
{
    __syncthreads();
    if (gridDim.x == 1) return;
    epoch += 1;
    if (threadIdx.x == 0) {
        const unsigned int target = epoch * gridDim.x;
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(bar) : "memory");
        unsigned int seen;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(bar) : "memory");
        } while (seen < target);
    }
    __syncthreads();
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// grid_sum<32>'s final step (reduce.cuh) run by every block: lane l adds partials l, l+32, ... in that order,
// then the 32 sums meet in the same xor shuffles.  The total is returned to every thread.
__device__ __forceinline__ double total_of_partials32(const double* partials, int n)
{
    __shared__ double sp[kPersistSmemPartials];
    __shared__ double total_s;
    const int lane = threadIdx.x & 31;
    if (n <= kPersistSmemPartials) {
        for (int i = threadIdx.x; i < n; i += kPersistBlock) sp[i] = __ldcg(partials + i);
        __syncthreads();
        if (threadIdx.x < 32) {
            double acc = 0.0;
            for (int i = lane; i < n; i += 32) acc += sp[i];
            acc = warp_sum(acc);
            if (lane == 0) total_s = acc;
        }
    } else if (threadIdx.x < 32) {
        double acc = 0.0;
        for (int i = lane; i < n; i += 32) acc += __ldcg(partials + i);
        acc = warp_sum(acc);
        if (lane == 0) total_s = acc;
    }
    __syncthreads();
    const double total = total_s;
    __syncthreads();  // total_s and sp are reused by the next call
    return total;
}

// block_sum<256> (reduce.cuh) by the 256 threads of a physical block; the sum is returned to every thread.
__device__ __forceinline__ double block_sum256_all(double v)
{
    __shared__ double total_b;
    const double s = block_sum<kPersistBlock>(v);
    if (threadIdx.x == 0) total_b = s;
    __syncthreads();
    const double total = total_b;
    __syncthreads();
    return total;
}

template <int RECON>
__global__ void __launch_bounds__(kPersistBlock, 1) stag_cg_persistent_kernel(const PersistArgs a)
{
    const size_t Vh = (size_t)a.g.Vh;
    const size_t nvec = 3 * Vh;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    constexpr int kWarps = kPersistBlock / 32;
    double* const part1 = a.partials;
    double* const part2 = a.partials + a.nvb;
    double* const part3 = a.partials + 2 * (size_t)a.nvb;
    unsigned int epoch = 0;

    // the CG scalars live in registers, identical in every thread of every block
    CgScalars* sc = a.sc;
    int it = sc->iter;
    const int maxiter = sc->maxiter;
    const double thresh = sc->thresh;
    double rr = sc->rr, pp = sc->pp, rr_new = sc->rr_new, tt = sc->tt, alpha = sc->alpha, beta = sc->beta;
    bool done = sc->done != 0;

    StagArgs<cplx> d1;  // t_o = D_oe p_e
    d1.g = a.g;
    d1.parity = 1;
    d1.gauge = a.gauge;
    d1.in = a.p;
    StagArgs<cplx> d2;  // D_eo t_o
    d2.g = a.g;
    d2.parity = 0;
    d2.gauge = a.gauge;
    d2.in = a.t;

    for (int k = 0; k < a.niter && !done; ++k) {
        // ---- S1: t = D_oe p; one warp = one 32-site virtual block, its |t|^2 as stag_dslash_kernel<SE_NORM, 32> leaves it
        for (int vb = blockIdx.x * kWarps + warp; vb < a.nvb; vb += gridDim.x * kWarps) {
            const int e = vb * 32 + lane;
            double local = 0.0;
            if (e < a.g.Vh) {
                cplx acc[3] = { czero<cplx>(), czero<cplx>(), czero<cplx>() };
                const Site s = decode_site(a.g, 1, e);
                stag_hop<0, RECON, false, cplx, VL_PLAIN, kPersistLinks>(d1, s, acc);
                stag_hop<1, RECON, false, cplx, VL_PLAIN, kPersistLinks>(d1, s, acc);
                stag_hop<2, RECON, false, cplx, VL_PLAIN, kPersistLinks>(d1, s, acc);
                stag_hop<3, RECON, false, cplx, VL_PLAIN, kPersistLinks>(d1, s, acc);
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    st_vec(a.t + c * Vh + e, acc[c]);
                    local += cnorm2(acc[c]);
                }
            }
            local = warp_sum(local);
            if (lane == 0) part1[vb] = local;
        }
        grid_barrier(a.bar, epoch);
        // ---- S2: alpha = rr / <p,Ap>, <p,Ap> from norms only
        tt = total_of_partials32(part1, a.nvb);
        alpha = rr / (a.m2 * pp + tt);

        // ---- S3: Ap = m^2 p - D_eo t (never stored); x += alpha p; r -= alpha Ap; partial |r|^2
        for (int vb = blockIdx.x * kWarps + warp; vb < a.nvb; vb += gridDim.x * kWarps) {
            const int e = vb * 32 + lane;
            double local = 0.0;
            if (e < a.g.Vh) {
                cplx acc[3] = { czero<cplx>(), czero<cplx>(), czero<cplx>() };
                const Site s = decode_site(a.g, 0, e);
                stag_hop<0, RECON, false, cplx, VL_PLAIN, kPersistLinks>(d2, s, acc);
                stag_hop<1, RECON, false, cplx, VL_PLAIN, kPersistLinks>(d2, s, acc);
                stag_hop<2, RECON, false, cplx, VL_PLAIN, kPersistLinks>(d2, s, acc);
                stag_hop<3, RECON, false, cplx, VL_PLAIN, kPersistLinks>(d2, s, acc);
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const size_t i = c * Vh + e;
                    const double2 pv = a.p[i], q = acc[c];
                    double2 xv = a.x[i], rv = a.r[i];
                    const double2 ap = cmake(fma(a.m2, pv.x, -q.x), fma(a.m2, pv.y, -q.y));
                    xv.x = fma(alpha, pv.x, xv.x);   // x = x + alpha p
                    xv.y = fma(alpha, pv.y, xv.y);
                    rv.x = fma(-alpha, ap.x, rv.x);  // r = r - alpha atap
                    rv.y = fma(-alpha, ap.y, rv.y);
                    a.x[i] = xv;
                    a.r[i] = rv;
                    local += cnorm2(rv);             // betan = <r,r>
                }
            }
            local = warp_sum(local);
            if (lane == 0) part2[vb] = local;
        }
        grid_barrier(a.bar, epoch);
        // ---- S4: beta, exit test (cg_after_update), on the device
        rr_new = total_of_partials32(part2, a.nvb);
        it += 1;
        if (blockIdx.x == 0 && threadIdx.x == 0 && it < kHistCap) a.hist[it] = rr_new;
        beta = rr_new / rr;
        rr = rr_new;
        if (rr_new <= thresh || it >= maxiter) done = true;
        if (done) break;

        // ---- S5: p = r + beta p, |p|^2: a physical block is one 256-thread block of cg_pupdate_kernel<256> at a time
        const size_t stride = (size_t)a.vgrid * kPersistBlock;
        for (int vb = blockIdx.x; vb < a.vgrid; vb += gridDim.x) {
            double local = 0.0;
            for (size_t j = (size_t)vb * kPersistBlock + threadIdx.x; j < nvec; j += stride) {
                const double2 rv = a.r[j];
                double2 pv = a.p[j];
                pv.x = fma(beta, pv.x, rv.x);
                pv.y = fma(beta, pv.y, rv.y);
                a.p[j] = pv;
                local += cnorm2(pv);
            }
            const double s_ = block_sum<kPersistBlock>(local);
            if (threadIdx.x == 0) part3[vb] = s_;
        }
        grid_barrier(a.bar, epoch);
        {
            double acc = 0.0;
            for (int i = threadIdx.x; i < a.vgrid; i += kPersistBlock) acc += __ldcg(part3 + i);
            pp = block_sum256_all(acc);
        }
    }

    if (blockIdx.x == 0 && threadIdx.x == 0) {
        sc->iter = it;
        sc->rr = rr;
        sc->rr_new = rr_new;
        sc->pp = pp;
        sc->tt = tt;
        sc->alpha = alpha;
        sc->beta = beta;
        sc->done = done ? 1 : 0;
    }
}

}  // namespace lqcd
