// cg_kernels.cuh -- the CG vector kernels, the one-off gauge
// reordering (S0) and the neighbour-table builder.
#pragma once
#include "reduce.cuh"

namespace lqcd {

// Which elements of the arrays make up a CG vector: n elements in runs of `inner`, the runs `stride`
// apart.  Contiguous vectors: inner = stride = n.  The even half of a full-lattice Wilson vector
// [12][V] (even-odd preconditioned solver): n = 12 Vh, inner = Vh, stride = V.
struct VecLayout {
    size_t n, inner, stride;
    __device__ __forceinline__ size_t at(size_t j) const
    {
        if (inner == n) return j;
        const size_t k = j / inner;
        return k * stride + (j - k * inner);
    }
};

// S6: p = r = b, x = 0, betan = <r,r> in one pass; also bb, pp and the CG
// bookkeeping.
template <int BLOCK>
__global__ void __launch_bounds__(BLOCK) cg_init_kernel(const cplx* __restrict__ b, cplx* __restrict__ x,
                                                        cplx* __restrict__ r, cplx* __restrict__ p, VecLayout lay,
                                                        CgScalars* sc, ReduceScratch rs, double* hist, double tol,
                                                        int maxiter)
{
    double local = 0.0;
    for (size_t j = (size_t)blockIdx.x * BLOCK + threadIdx.x; j < lay.n; j += (size_t)gridDim.x * BLOCK) {
        const size_t i = lay.at(j);
        const cplx v = b[i];
        r[i] = v;
        p[i] = v;
        x[i] = cmake(0.0, 0.0);
        local += cnorm2(v);
    }
    grid_sum<BLOCK>(local, rs, [sc, hist, tol, maxiter](double bb) {
        sc->rr = bb;
        sc->rr_new = bb;
        sc->bb = bb;
        sc->pp = bb;
        sc->tt = 0.0;
        sc->alpha = 0.0;
        sc->beta = 0.0;
        sc->thresh = tol * tol * bb;
        sc->res2 = 0.0;
        sc->iter = 0;
        sc->maxiter = maxiter;
        sc->done = (bb == 0.0 || maxiter <= 0) ? 1 : 0;  // b = 0: x = 0, iters = 0 (reading A11)
        sc->pause = 0;
        sc->nupd = 0;
        sc->xdue = 0;
        hist[0] = bb;
    });
}

// S6 of the mixed-precision solver: x = 0 (fp64), xs = 0, rs = ps = fl32(b),
// rr = bb = <b,b> from the fp64 source, pp = <ps,ps> from the fp32 copy, rmax = |b|.
template <int BLOCK>
__global__ void __launch_bounds__(BLOCK) cg_init_mixed_kernel(const cplx* __restrict__ b, cplx* __restrict__ x,
                                                              cplxf* __restrict__ xs, cplxf* __restrict__ rs,
                                                              cplxf* __restrict__ ps, size_t n, CgScalars* sc,
                                                              ReduceScratch rs_, double* hist, double tol, double delta,
                                                              int maxiter)
{
    double local[2] = { 0.0, 0.0 };
    for (size_t i = (size_t)blockIdx.x * BLOCK + threadIdx.x; i < n; i += (size_t)gridDim.x * BLOCK) {
        const cplx v = b[i];
        const cplxf vf = make_float2((float)v.x, (float)v.y);
        x[i] = cmake(0.0, 0.0);
        xs[i] = make_float2(0.f, 0.f);
        rs[i] = vf;
        ps[i] = vf;
        local[0] += cnorm2(v);
        local[1] += cnorm2(vf);
    }
    grid_sum_n<BLOCK, 2>(local, rs_, [sc, hist, tol, delta, maxiter](const double (&tot)[2]) {
        const double bb = tot[0];
        sc->rr = bb;
        sc->rr_new = bb;
        sc->bb = bb;
        sc->pp = tot[1];
        sc->tt = 0.0;
        sc->alpha = 0.0;
        sc->beta = 0.0;
        sc->thresh = tol * tol * bb;
        sc->res2 = 0.0;
        sc->rmax = sqrt(bb);
        sc->delta = delta;
        sc->iter = 0;
        sc->maxiter = maxiter;
        sc->done = (bb == 0.0 || maxiter <= 0) ? 1 : 0;
        sc->pause = 0;
        sc->nupd = 0;
        hist[0] = bb;
    });
}

// Reliable update, first step: x += xs (fp64), xs = 0.  `only_if_paused` = 1 inside the iteration
// (a stale launch must not touch anything); 0 for the final accumulation after the loop has ended.
template <int BLOCK>
__global__ void __launch_bounds__(BLOCK) mixed_accumulate_kernel(cplx* __restrict__ x, cplxf* __restrict__ xs, size_t n,
                                                                 const CgScalars* sc, int only_if_paused)
{
    if (only_if_paused && !sc->pause) return;
    for (size_t i = (size_t)blockIdx.x * BLOCK + threadIdx.x; i < n; i += (size_t)gridDim.x * BLOCK) {
        const cplxf d = xs[i];
        cplx v = x[i];
        v.x += (double)d.x;
        v.y += (double)d.y;
        x[i] = v;
        xs[i] = make_float2(0.f, 0.f);
    }
}

// fp64 structure-of-arrays links -> fp32 copy of the same layout (built once per loaded gauge field).
static __global__ void gauge_narrow_kernel(const cplx* __restrict__ g64, cplxf* __restrict__ g32, size_t n)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const cplx v = g64[i];
        g32[i] = make_float2((float)v.x, (float)v.y);
    }
}

// S5 (PAPER.md:96 gives beta; the p-update itself fell off the truncated listing, reading A7):
// p = r + beta p, pp = <p,p>.
// C = cplx (the fp64 path) or cplxf (the fp32 inner iteration: evaluated in fp64, rounded on store,
// the norm taken of the stored value).
template <int BLOCK, class C>
__global__ void __launch_bounds__(BLOCK) cg_pupdate_kernel(const C* __restrict__ r, C* __restrict__ p, VecLayout lay,
                                                           CgScalars* sc, ReduceScratch rs)
{
    if (sc->done | sc->pause) return;
    const double beta = sc->beta;
    double local = 0.0;
    for (size_t j = (size_t)blockIdx.x * BLOCK + threadIdx.x; j < lay.n; j += (size_t)gridDim.x * BLOCK) {
        const size_t i = lay.at(j);
        const double2 rv = to_d(r[i]);
        double2 pv = to_d(p[i]);
        pv.x = fma(beta, pv.x, rv.x);
        pv.y = fma(beta, pv.y, rv.y);
        const C ps = to_cplx(pv, (C*)0);
        p[i] = ps;
        local += cnorm2(ps);
    }
    grid_sum<BLOCK>(local, rs, [sc](double pp) { sc->pp = pp; });
}

// The vector kernel of a Wilson CG iteration: x += alpha p (the second half of S3, moved here
// because this kernel reads p anyway -- the Dslash kernel that updates r then never touches p or x), then S5:
// p = r + beta p, pp = <p,p> unless the exit rule has fired.  `xdue` makes a pre-enqueued launch after
// convergence a no-op without losing the x update of the converging iteration.
template <int BLOCK>
__global__ void __launch_bounds__(BLOCK) cg_xpupdate_kernel(const cplx* __restrict__ r, cplx* __restrict__ p, cplx* __restrict__ x,
                                                            VecLayout lay, CgScalars* sc, ReduceScratch rs)
{
    if (!sc->xdue) return;
    const double alpha = sc->alpha, beta = sc->beta;
    const bool done = sc->done != 0;
    double local = 0.0;
    for (size_t j = (size_t)blockIdx.x * BLOCK + threadIdx.x; j < lay.n; j += (size_t)gridDim.x * BLOCK) {
        const size_t i = lay.at(j);
        double2 pv = p[i];
        double2 xv = x[i];
        xv.x = fma(alpha, pv.x, xv.x);   // x = x + alpha p
        xv.y = fma(alpha, pv.y, xv.y);
        st_stream(x + i, xv);
        if (!done) {
            const double2 rv = r[i];
            pv.x = fma(beta, pv.x, rv.x);
            pv.y = fma(beta, pv.y, rv.y);
            p[i] = pv;
            local += cnorm2(pv);
        }
    }
    grid_sum<BLOCK>(local, rs, [sc, done](double pp) {
        if (!done) sc->pp = pp;
        sc->xdue = 0;
    });
}

// S0: canonical u[g][mu][3][3] (array of structures, 576 B per site, fp64) ->
// [parity][mu][RECON/2][Vh] in the storage type C (structure of arrays; two rows only for
// RECON = 12).  A block stages TILE sites through shared memory so both the global read and the
// global write are contiguous.
template <int BLOCK, int TILE, int RECON, class C>
__global__ void __launch_bounds__(BLOCK) gauge_reorder_kernel(const cplx* __restrict__ u, C* __restrict__ soa,
                                                              size_t Vh)
{
    constexpr int NC = RECON / 2;
    __shared__ cplx tile[TILE * 36 + 1];
    const size_t V = 2 * Vh;
    const size_t g0 = (size_t)blockIdx.x * TILE;
    const size_t nsite = g0 + TILE <= V ? TILE : V - g0;
    for (size_t i = threadIdx.x; i < nsite * 36; i += BLOCK) tile[i] = u[g0 * 36 + i];
    __syncthreads();
    for (size_t i = threadIdx.x; i < nsite * 4 * NC; i += BLOCK) {
        const size_t j = i / nsite;  // mu*NC + k
        const size_t s = i - j * nsite;
        const size_t mu = j / NC, k = j - mu * NC;
        const size_t g = g0 + s;
        const size_t parity = g >= Vh ? 1 : 0;
        const size_t e = g - parity * Vh;
        soa[(parity * 4 * NC + j) * Vh + e] = to_cplx(tile[s * 36 + mu * 9 + k], (C*)0);
    }
}

// The paper's iup / idn as g-indices, from the same nbr_fwd / nbr_bwd the
// Dslash kernels use, plus lex2eo[s] = g.
static __global__ void tables_kernel(Geom g, int32_t* __restrict__ iup, int32_t* __restrict__ idn,
                              int32_t* __restrict__ lex2eo)
{
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= g.V) return;
    const int parity = idx >= g.Vh ? 1 : 0;
    const int e = (int)(idx - (long long)parity * g.Vh);
    const Site s = decode_site(g, parity, e);
    const long long other = (long long)(1 - parity) * g.Vh;
    iup[0 * g.V + idx] = (int32_t)(other + nbr_fwd<0>(g, s));
    iup[1 * g.V + idx] = (int32_t)(other + nbr_fwd<1>(g, s));
    iup[2 * g.V + idx] = (int32_t)(other + nbr_fwd<2>(g, s));
    iup[3 * g.V + idx] = (int32_t)(other + nbr_fwd<3>(g, s));
    idn[0 * g.V + idx] = (int32_t)(other + nbr_bwd<0>(g, s));
    idn[1 * g.V + idx] = (int32_t)(other + nbr_bwd<1>(g, s));
    idn[2 * g.V + idx] = (int32_t)(other + nbr_bwd<2>(g, s));
    idn[3 * g.V + idx] = (int32_t)(other + nbr_bwd<3>(g, s));
    const long long L0 = 2LL * g.Lh;
    const long long x0 = 2LL * s.xh + s.r;
    const long long lex = x0 + L0 * (s.x1 + (long long)g.L1 * (s.x2 + (long long)g.L2 * s.x3));
    lex2eo[lex] = (int32_t)idx;
}

}  // namespace lqcd
