// stag_dslash.cuh -- staggered hopping term with fused CG epilogues.
//
//   (D chi)(x) = 1/2 sum_mu eta_mu(x) [ b+ U_mu(x) chi(x+mu^) - b- U_mu(x-mu^)^+ chi(x-mu^) ]
//
// This is the paper's fmv / fmtv pair: fmv = D_oe, fmtv = the second hop that
// "accumulates into atap which was pre-set to p".  One thread per output site;
// consecutive threads own consecutive half-lattice indices e, and every array is
// structure-of-arrays with the site index fastest, so each warp-wide 128-bit load is one
// contiguous 512-byte run (the paper's p(l,ic) layout, extended to the links).
// Neighbour indices, staggered phases and the antiperiodic time boundary are computed in
// registers; the iup/idn tables are never read on the hot path.
//
// HBM traffic per output site: 8 links x 144 B (streamed once, evict-first) + 48 B input vector
// (each element is gathered by 8 sites but read from DRAM once: L1/L2 hits) + 48 B output
// = 1248 B, the figure the roofline is quoted on.
#pragma once
#include "reduce.cuh"

namespace lqcd {

enum StagEpilogue {
    SE_PLAIN = 0,     // out = D in                                            (lqcd_dslash)
    SE_NORM = 1,      // out = D in, tt = |out|^2, alpha = rr/(m^2 pp + tt)     (S1 + S2)
    SE_MDAGM = 2,     // out = m^2 p - D in                                     (lqcd_apply_MdagM, 2nd hop)
    SE_CGUPDATE = 3,  // Ap = m^2 p - D in; x += alpha p; r -= alpha Ap; |r|^2  (S3), Ap never stored
    SE_RESIDUAL = 4   // |b - (m^2 p - D in)|^2                                 (S7), nothing stored
};

struct StagArgs {
    Geom g;
    int parity;         // parity of the output sites
    const cplx* gauge;  // [2][4][9][Vh]
    const cplx* in;     // [3][Vh] on parity 1-parity
    cplx* out;          // [3][Vh]
    const cplx* p;      // epilogue operand on the output parity (p, or x for SE_RESIDUAL)
    cplx* x;
    cplx* r;
    const cplx* b;
    double m2;
    CgScalars* sc;
    ReduceScratch rs;
    double* hist;
};

template <int MU>
__device__ __forceinline__ void stag_hop(const StagArgs& a, const Site& s, cplx acc[3])
{
    const size_t Vh = (size_t)a.g.Vh;
    double eta;
    if (MU == 0) eta = 0.5;
    else if (MU == 1) eta = s.r ? -0.5 : 0.5;
    else if (MU == 2) eta = ((s.r + s.x1) & 1) ? -0.5 : 0.5;
    else eta = ((s.r + s.x1 + s.x2) & 1) ? -0.5 : 0.5;

    const int ef = nbr_fwd<MU>(a.g, s);
    const int eb = nbr_bwd<MU>(a.g, s);
    const cplx* Uf = a.gauge + (size_t)((a.parity * 4 + MU) * 9) * Vh + s.e;
    const cplx* Ub = a.gauge + (size_t)(((1 - a.parity) * 4 + MU) * 9) * Vh + eb;

    cplx U[9], W[9], vf[3], vb[3];
#pragma unroll
    for (int k = 0; k < 9; ++k) U[k] = ld_stream(Uf + k * Vh);
#pragma unroll
    for (int c = 0; c < 3; ++c) vf[c] = ld_keep(a.in + c * Vh + ef);
#pragma unroll
    for (int k = 0; k < 9; ++k) W[k] = ld_stream(Ub + k * Vh);
#pragma unroll
    for (int c = 0; c < 3; ++c) vb[c] = ld_keep(a.in + c * Vh + eb);

    const double sf = eta * bc_fwd<MU>(a.g, s);
    const double sb = -eta * bc_bwd<MU>(a.g, s);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        vf[c] = cscale(sf, vf[c]);
        vb[c] = cscale(sb, vb[c]);
    }
#pragma unroll
    for (int r = 0; r < 3; ++r) {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            cfma(acc[r], U[r * 3 + c], vf[c]);       // U_mu(x) chi(x+mu)
            cfma_conj(acc[r], W[c * 3 + r], vb[c]);  // U_mu(x-mu)^+ chi(x-mu)
        }
    }
}

template <int EPI, int BLOCK>
__global__ void __launch_bounds__(BLOCK) stag_dslash_kernel(const StagArgs a)
{
    if (EPI == SE_NORM || EPI == SE_CGUPDATE) {
        if (a.sc->done) return;  // converged earlier: this (pre-enqueued) iteration is a no-op
    }
    const int e = blockIdx.x * BLOCK + threadIdx.x;
    const bool active = e < a.g.Vh;
    const size_t Vh = (size_t)a.g.Vh;
    cplx acc[3] = { cmake(0, 0), cmake(0, 0), cmake(0, 0) };
    if (active) {
        const Site s = decode_site(a.g, a.parity, e);
        stag_hop<0>(a, s, acc);
        stag_hop<1>(a, s, acc);
        stag_hop<2>(a, s, acc);
        stag_hop<3>(a, s, acc);
    }
    if (EPI == SE_PLAIN) {
        if (active) {
#pragma unroll
            for (int c = 0; c < 3; ++c) st_vec(a.out + c * Vh + e, acc[c]);
        }
    } else if (EPI == SE_MDAGM) {
        if (active) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const cplx pv = a.p[c * Vh + e];
                st_vec(a.out + c * Vh + e, cmake(fma(a.m2, pv.x, -acc[c].x), fma(a.m2, pv.y, -acc[c].y)));
            }
        }
    } else if (EPI == SE_NORM) {
        double local = 0.0;
        if (active) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                st_vec(a.out + c * Vh + e, acc[c]);
                local += cnorm2(acc[c]);
            }
        }
        CgScalars* sc = a.sc;
        const double m2 = a.m2;
        grid_sum<BLOCK>(local, a.rs, [sc, m2](double tt) {
            sc->tt = tt;
            sc->alpha = sc->rr / (m2 * sc->pp + tt);  // <p,Ap> from norms only
        });
    } else if (EPI == SE_CGUPDATE) {
        double local = 0.0;
        if (active) {
            const double alpha = a.sc->alpha;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const size_t i = c * Vh + e;
                const cplx pv = a.p[i];
                cplx xv = a.x[i], rv = a.r[i];
                const cplx ap = cmake(fma(a.m2, pv.x, -acc[c].x), fma(a.m2, pv.y, -acc[c].y));
                xv.x = fma(alpha, pv.x, xv.x);   // x = x + alpha p
                xv.y = fma(alpha, pv.y, xv.y);
                rv.x = fma(-alpha, ap.x, rv.x);  // r = r - alpha atap
                rv.y = fma(-alpha, ap.y, rv.y);
                a.x[i] = xv;
                a.r[i] = rv;
                local += cnorm2(rv);             // betan = <r,r>
            }
        }
        CgScalars* sc = a.sc;
        double* hist = a.hist;
        grid_sum<BLOCK>(local, a.rs, [sc, hist](double rr_new) {
            const int it = sc->iter + 1;
            sc->iter = it;
            sc->rr_new = rr_new;
            if (it < kHistCap) hist[it] = rr_new;
            sc->beta = rr_new / sc->rr;  // beta = betan/betad; betad = betan
            sc->rr = rr_new;
            if (rr_new <= sc->thresh || it >= sc->maxiter) sc->done = 1;
        });
    } else {  // SE_RESIDUAL
        double local = 0.0;
        if (active) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const size_t i = c * Vh + e;
                const cplx xv = a.p[i], bv = a.b[i];
                const double re = bv.x - fma(a.m2, xv.x, -acc[c].x);
                const double im = bv.y - fma(a.m2, xv.y, -acc[c].y);
                local += fma(re, re, im * im);
            }
        }
        CgScalars* sc = a.sc;
        grid_sum<BLOCK>(local, a.rs, [sc](double res2) { sc->res2 = res2; });
    }
}

}  // namespace lqcd
