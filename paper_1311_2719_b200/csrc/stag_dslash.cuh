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
#include "slab_sync.cuh"

namespace lqcd {

enum StagEpilogue {
    SE_PLAIN = 0,     // out = D in                                            (lqcd_dslash)
    SE_NORM = 1,      // out = D in, tt = |out|^2, alpha = rr/(m^2 pp + tt)     (S1 + S2)
    SE_MDAGM = 2,     // out = m^2 p - D in                                     (lqcd_apply_MdagM, 2nd hop)
    SE_CGUPDATE = 3,  // Ap = m^2 p - D in; x += alpha p; r -= alpha Ap; |r|^2  (S3), Ap never stored
    SE_RESIDUAL = 4,  // |b - (m^2 p - D in)|^2                                 (S7), nothing stored
    // full-system solve M x = b, M = m + D; `m2` carries the mass m here
    SE_PREP = 5,      // out = m p - D in              source preparation  b' = m b_e - D_eo b_o
    SE_RECON = 6,     // out = (p - D in)/m            reconstruction      x_o = (b_o - D_oe x_e)/m
    SE_RESIDUAL_M = 7, // |b - (m p + D in)|^2 and |b|^2 of one parity, set (flag = 0) or added (flag = 1)
    // mixed-precision CG with reliable updates
    SE_CGUPDATE_MIXED = 8,  // SE_CGUPDATE on the fp32 vectors; the scalar step may pause for a reliable update
    SE_RELIABLE = 9         // fp64: r = b - (m^2 p - D in), rf = fl32(r), |r|^2; resumes the paused iteration
};

// Time-slab decomposition (include/lqcd_slab.h).  The Geom of a slab is
// that of its local L0 x L1 x L2 x T lattice; hops in time that leave the slab read the neighbour
// rank's boundary time-slice from a ghost face ([3][sh], sh = sites of one parity in a time-slice)
// that the neighbour's producing kernel stored there through peer memory, and the backward hop at
// the first local slice reads U_3 of the slice below from a ghost copy ([parity][NC][sh]).
template <class C>
struct SlabArgs {
    int t0, L3g, sh;       // first global time-slice of the slab, global time extent, half-slice sites
    const C* ghost_lo;     // input vector on time-slice t0-1 (global, periodic), parity of `in`
    const C* ghost_hi;     // input vector on time-slice t0+T
    const C* gauge_ghost;  // U_3 on time-slice t0-1
    C* push_lo;            // where the slab below (rank-1) keeps its ghost_hi: receives `out` on local slice 0
    C* push_hi;            // where the slab above (rank+1) keeps its ghost_lo: receives `out` on local slice T-1
    double* part;          // this rank's partial sums (the cross-rank combine kernel adds them in rank order)
};

template <class C>
struct StagArgs {
    Geom g;
    int parity;      // parity of the output sites
    const C* gauge;  // [2][4][RECON/2][Vh]
    const C* in;     // [3][Vh] on parity 1-parity
    C* out;          // [3][Vh]
    const C* p;      // epilogue operand on the output parity (p, or x for SE_RESIDUAL)
    C* x;
    C* r;
    const C* b;
    cplxf* rf;       // SE_RELIABLE: the fp32 residual the inner iteration continues from
    double m2;
    int flag;
    CgScalars* sc;
    ReduceScratch rs;
    double* hist;
    SlabArgs<C> sl;  // used by the SLAB instantiations only
};

// LINKS: cache policy of the link loads of the undivided lattice (device_common.cuh LinkPolicy).
template <int MU, int RECON, bool SLAB, class C, int VL = VL_NC, int LINKS = LP_STREAM>
__device__ __forceinline__ void stag_hop(const StagArgs<C>& a, const Site& s, C acc[3])
{
    constexpr int NC = RECON / 2;
    const size_t Vh = (size_t)a.g.Vh;
    const double eta = half_eta<MU>(s);
    const C* Uf = a.gauge + (size_t)((a.parity * 4 + MU) * NC) * Vh + s.e;
    C U[9], W[9], vf[3], vb[3];
    double sf, sb;
    if (SLAB && MU == 3) {
        // Time hops of a slab: no wrap inside the slab; the two boundary slices read the ghost faces the
        // neighbour ranks stored through peer memory.  One code path: base pointer and colour stride are
        // selected, then the loads are those of the undivided kernel.  L2 loads (ld.cg) throughout --
        // never the read-only path for peer-written data; the t+-1 neighbours are sh sites away, in
        // other blocks, so L1 would not have helped.
        const bool top = s.x3 + 1 == a.g.L3, bottom = s.x3 == 0;
        const size_t sh = (size_t)a.sl.sh;
        const C* vfp = top ? a.sl.ghost_hi + (s.e - (a.g.L3 - 1) * a.g.s3) : a.in + (s.e + a.g.s3);
        const size_t vfs = top ? sh : Vh;
        const C* vbp = bottom ? a.sl.ghost_lo + s.e : a.in + (s.e - a.g.s3);
        const C* Ub = bottom ? a.sl.gauge_ghost + (size_t)((1 - a.parity) * NC) * sh + s.e
                             : a.gauge + (size_t)(((1 - a.parity) * 4 + MU) * NC) * Vh + (s.e - a.g.s3);
        const size_t vbs = bottom ? sh : Vh;
        load_link<RECON>(Uf, Vh, U);
#pragma unroll
        for (int c = 0; c < 3; ++c) vf[c] = __ldcg(vfp + c * vfs);
        load_link<RECON>(Ub, vbs, W);
#pragma unroll
        for (int c = 0; c < 3; ++c) vb[c] = __ldcg(vbp + c * vbs);
        // antiperiodic boundary of the GLOBAL lattice (reading A4)
        sf = (a.sl.t0 + s.x3 + 1 == a.sl.L3g) ? -eta : eta;
        sb = (a.sl.t0 + s.x3 == 0) ? eta : -eta;
    } else {
        const int ef = nbr_fwd<MU>(a.g, s);
        const int eb = nbr_bwd<MU>(a.g, s);
        const C* Ub = a.gauge + (size_t)(((1 - a.parity) * 4 + MU) * NC) * Vh + eb;
        load_link<RECON, C, LINKS>(Uf, Vh, U);
#pragma unroll
        for (int c = 0; c < 3; ++c) vf[c] = ld_vec<VL>(a.in + c * Vh + ef);
        load_link<RECON, C, LINKS>(Ub, Vh, W);
#pragma unroll
        for (int c = 0; c < 3; ++c) vb[c] = ld_vec<VL>(a.in + c * Vh + eb);
        sf = eta * bc_fwd<MU>(a.g, s);
        sb = -eta * bc_bwd<MU>(a.g, s);
    }
    reconstruct_link<RECON>(U);
    reconstruct_link<RECON>(W);

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

// Epilogue arithmetic is done in fp64 whatever the storage type C (free for fp64, a handful of
// converts per site for the fp32 inner iterations of the mixed-precision solver).
// Minimum resident blocks per SM (measured on B200 at 32^4, profiles/):
// all nine entries: the plain Dslash runs at 93-94 us whatever the bound (252 registers at 1, 72 at
// 7), but the kernels with a CG epilogue gain from occupancy because the epilogue's loads of p, r, x
// are issued after the hops: 247 us per CG iteration at 1-2 blocks/SM, 239 at 4-5, 235 at 7.
// Two-row links: without a bound ptxas keeps both links of a hop and their rebuilt rows live
// (128-138 registers, 3 blocks/SM: 6.2 TB/s); 4 blocks/SM caps it at 128 and measured best
// (65.4 us = 6.9 TB/s; 5 -> 68 us, 6+ spills -> 100+ us).
#ifndef LQCD_STAG_MINB18
#define LQCD_STAG_MINB18 7
#endif
#ifndef LQCD_STAG_MINB12
#define LQCD_STAG_MINB12 4
#endif
#ifndef LQCD_STAG_MINB18F
#define LQCD_STAG_MINB18F 8
#endif
#ifndef LQCD_STAG_MINB12F
#define LQCD_STAG_MINB12F 8
#endif
template <int RECON, class C> struct StagMinBlocks { static constexpr int value = RECON == 12 ? LQCD_STAG_MINB12 : LQCD_STAG_MINB18; };
template <int RECON> struct StagMinBlocks<RECON, cplxf> { static constexpr int value = RECON == 12 ? LQCD_STAG_MINB12F : LQCD_STAG_MINB18F; };

// Slab kernels that produce a vector the next Dslash will read (SE_PLAIN, SE_NORM) also store its
// two boundary time-slices into the neighbour ranks' ghost faces: the halo exchange is part of the
// producing kernel (stores through peer memory over NVLink), not a separate pack + send.
template <class C>
__device__ __forceinline__ void slab_push(const StagArgs<C>& a, int x3, int e, const C v[3])
{
    const size_t sh = (size_t)a.sl.sh;
    if (a.sl.push_lo == nullptr) return;  // the vector produced is not the input of a later Dslash
    if (x3 == 0) {
#pragma unroll
        for (int c = 0; c < 3; ++c) a.sl.push_lo[c * sh + e] = v[c];
    }
    if (x3 + 1 == a.g.L3) {
        const int f = e - (a.g.L3 - 1) * a.g.s3;
#pragma unroll
        for (int c = 0; c < 3; ++c) a.sl.push_hi[c * sh + f] = v[c];
    }
}

// `sy` (slab kernels only): non-null = this kernel's LAST block also runs the synchronisation point
// that follows it (slab_sync_tail); null = the host launches the synchronisation kernels.
template <int EPI, int BLOCK, int RECON, bool SLAB, class C>
__device__ __forceinline__ void stag_dslash_body(const StagArgs<C>& a, const SlabSyncArgs* sy = nullptr)
{
    if (EPI == SE_NORM || EPI == SE_CGUPDATE || EPI == SE_CGUPDATE_MIXED) {
        // converged earlier, or waiting for a reliable update: this (pre-enqueued) iteration is a no-op
        if (a.sc->done | a.sc->pause) return;
    }
    int e = blockIdx.x * BLOCK + threadIdx.x;
    const bool active = e < a.g.Vh;
    if (SLAB) {
        // Slab kernels walk the sites starting at the LAST time-slice (then slice 0, 1, ...): the blocks that store
        // faces into a neighbour's memory -- and pay a system-scope fence for it before they take the reduction
        // ticket -- are then the first to run instead of the last, and their fences are off the kernel's tail.
        e += a.g.Vh - a.sl.sh;
        if (e >= a.g.Vh) e -= a.g.Vh;
    }
    const size_t Vh = (size_t)a.g.Vh;
    C acc[3] = { czero<C>(), czero<C>(), czero<C>() };
    int x3 = 0;
    if (active) {
        const Site s = decode_site(a.g, a.parity, e);
        x3 = s.x3;
        stag_hop<0, RECON, SLAB>(a, s, acc);
        stag_hop<1, RECON, SLAB>(a, s, acc);
        stag_hop<2, RECON, SLAB>(a, s, acc);
        stag_hop<3, RECON, SLAB>(a, s, acc);
    }
    bool wrote_peer = false;
    if (SLAB && (EPI == SE_PLAIN || EPI == SE_NORM)) {
        if (active) {
            slab_push(a, x3, e, acc);
            wrote_peer = a.sl.push_lo != nullptr && (x3 == 0 || x3 + 1 == a.g.L3);
        }
    }
    if (SLAB && EPI != SE_PLAIN && EPI != SE_MDAGM) {
        // Slab epilogues with a sum: the same per-site arithmetic as below, but the total over this
        // rank's sites is only a partial; the scalar step runs in the cross-rank combine kernel.
        double local = 0.0;
        if (active) {
            if (EPI == SE_NORM) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    st_vec(a.out + c * Vh + e, acc[c]);
                    local += cnorm2(acc[c]);
                }
            } else if (EPI == SE_RELIABLE) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const size_t i = c * Vh + e;
                    const double2 xv = to_d(a.p[i]), bv = to_d(a.b[i]), q = to_d(acc[c]);
                    const double2 rv = cmake(bv.x - fma(a.m2, xv.x, -q.x), bv.y - fma(a.m2, xv.y, -q.y));
                    a.rf[i] = make_float2((float)rv.x, (float)rv.y);
                    local += cnorm2(rv);
                }
            } else if (EPI == SE_CGUPDATE || EPI == SE_CGUPDATE_MIXED) {
                const double alpha = a.sc->alpha;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const size_t i = c * Vh + e;
                    const double2 pv = to_d(a.p[i]), q = to_d(acc[c]);
                    double2 xv = to_d(a.x[i]), rv = to_d(a.r[i]);
                    const double2 ap = cmake(fma(a.m2, pv.x, -q.x), fma(a.m2, pv.y, -q.y));
                    xv.x = fma(alpha, pv.x, xv.x);
                    xv.y = fma(alpha, pv.y, xv.y);
                    rv.x = fma(-alpha, ap.x, rv.x);
                    rv.y = fma(-alpha, ap.y, rv.y);
                    const C rs_ = to_cplx(rv, (C*)0);
                    a.x[i] = to_cplx(xv, (C*)0);
                    a.r[i] = rs_;
                    local += cnorm2(rs_);
                }
            } else {  // SE_RESIDUAL
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const size_t i = c * Vh + e;
                    const double2 xv = to_d(a.p[i]), bv = to_d(a.b[i]), q = to_d(acc[c]);
                    const double re = bv.x - fma(a.m2, xv.x, -q.x);
                    const double im = bv.y - fma(a.m2, xv.y, -q.y);
                    local += fma(re, re, im * im);
                }
            }
        }
        if (sy != nullptr) {
            grid_sum_block<BLOCK>(local, wrote_peer, a.rs, [sy]() { return sy->ss->seq; },
                                  [sy](double v, unsigned long long sq) { slab_sync_tail<BLOCK>(*sy, v, sq); });
        } else {
            double* part = a.sl.part;
            grid_sum<BLOCK>(local, a.rs, [part](double v) { part[0] = v; });
        }
        return;
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
                const double2 pv = to_d(a.p[c * Vh + e]), q = to_d(acc[c]);
                st_vec(a.out + c * Vh + e, to_cplx(cmake(fma(a.m2, pv.x, -q.x), fma(a.m2, pv.y, -q.y)), (C*)0));
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
    } else if (EPI == SE_CGUPDATE || EPI == SE_CGUPDATE_MIXED) {
        double local = 0.0;
        if (active) {
            const double alpha = a.sc->alpha;
            // all nine operands are loaded before the first store: p, x and r may alias as far as the compiler
            // can tell, so a load placed after a store waits for it (three serial round trips, colour by colour)
            C p3[3], x3[3], r3[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const size_t i = c * Vh + e;
                p3[c] = a.p[i];
                x3[c] = a.x[i];
                r3[c] = a.r[i];
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const size_t i = c * Vh + e;
                const double2 pv = to_d(p3[c]), q = to_d(acc[c]);
                double2 xv = to_d(x3[c]), rv = to_d(r3[c]);
                const double2 ap = cmake(fma(a.m2, pv.x, -q.x), fma(a.m2, pv.y, -q.y));
                xv.x = fma(alpha, pv.x, xv.x);   // x = x + alpha p
                xv.y = fma(alpha, pv.y, xv.y);
                rv.x = fma(-alpha, ap.x, rv.x);  // r = r - alpha atap
                rv.y = fma(-alpha, ap.y, rv.y);
                const C rs_ = to_cplx(rv, (C*)0);
                a.x[i] = to_cplx(xv, (C*)0);
                a.r[i] = rs_;
                local += cnorm2(rs_);            // betan = <r,r>
            }
        }
        CgScalars* sc = a.sc;
        double* hist = a.hist;
        if (EPI == SE_CGUPDATE)
            grid_sum<BLOCK>(local, a.rs, [sc, hist](double rr_new) { cg_after_update(sc, hist, rr_new); });
        else
            grid_sum<BLOCK>(local, a.rs, [sc, hist](double rr_new) { cg_after_update_mixed(sc, hist, rr_new); });
    } else if (EPI == SE_RELIABLE) {
        double local = 0.0;
        if (active) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const size_t i = c * Vh + e;
                const double2 xv = to_d(a.p[i]), bv = to_d(a.b[i]), q = to_d(acc[c]);
                const double2 rv = cmake(bv.x - fma(a.m2, xv.x, -q.x), bv.y - fma(a.m2, xv.y, -q.y));
                a.rf[i] = make_float2((float)rv.x, (float)rv.y);
                local += cnorm2(rv);
            }
        }
        CgScalars* sc = a.sc;
        double* hist = a.hist;
        grid_sum<BLOCK>(local, a.rs, [sc, hist](double rr_true) { cg_after_reliable(sc, hist, rr_true); });
    } else if (EPI == SE_PREP || EPI == SE_RECON) {
        if (active) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double2 pv = to_d(a.p[c * Vh + e]), q = to_d(acc[c]);
                const double2 o = EPI == SE_PREP ? cmake(fma(a.m2, pv.x, -q.x), fma(a.m2, pv.y, -q.y))
                                                 : cmake((pv.x - q.x) / a.m2, (pv.y - q.y) / a.m2);
                st_vec(a.out + c * Vh + e, to_cplx(o, (C*)0));
            }
        }
    } else if (EPI == SE_RESIDUAL_M) {
        double local[2] = { 0.0, 0.0 };
        if (active) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const size_t i = c * Vh + e;
                const double2 xv = to_d(a.p[i]), bv = to_d(a.b[i]), q = to_d(acc[c]);
                const double re = bv.x - fma(a.m2, xv.x, q.x);
                const double im = bv.y - fma(a.m2, xv.y, q.y);
                local[0] += fma(re, re, im * im);
                local[1] += cnorm2(bv);
            }
        }
        CgScalars* sc = a.sc;
        const int add = a.flag;
        grid_sum_n<BLOCK, 2>(local, a.rs, [sc, add](const double (&tot)[2]) {
            sc->res2 = add ? sc->res2 + tot[0] : tot[0];
            sc->aux = add ? sc->aux + tot[1] : tot[1];
        });
    } else {  // SE_RESIDUAL
        double local = 0.0;
        if (active) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const size_t i = c * Vh + e;
                const double2 xv = to_d(a.p[i]), bv = to_d(a.b[i]), q = to_d(acc[c]);
                const double re = bv.x - fma(a.m2, xv.x, -q.x);
                const double im = bv.y - fma(a.m2, xv.y, -q.y);
                local += fma(re, re, im * im);
            }
        }
        CgScalars* sc = a.sc;
        grid_sum<BLOCK>(local, a.rs, [sc](double res2) { sc->res2 = res2; });
    }
}

template <int EPI, int BLOCK, int RECON, class C>
__global__ void __launch_bounds__(BLOCK, StagMinBlocks<RECON, C>::value) stag_dslash_kernel(const StagArgs<C> a)
{
    stag_dslash_body<EPI, BLOCK, RECON, false>(a);
}

// The same hopping term on one rank's time-slab (fp64; SE_PLAIN, SE_NORM, SE_MDAGM, SE_CGUPDATE, SE_RESIDUAL).
template <int EPI, int BLOCK, int RECON, class C>
__global__ void __launch_bounds__(BLOCK, StagMinBlocks<RECON, C>::value) stag_dslash_slab_kernel(const StagArgs<C> a)
{
    stag_dslash_body<EPI, BLOCK, RECON, true>(a);
}

// ... with the synchronisation point that follows it run by its last block (one rank per process).
template <int EPI, int BLOCK, int RECON, class C>
__global__ void __launch_bounds__(BLOCK, StagMinBlocks<RECON, C>::value)
stag_dslash_slab_sync_kernel(const StagArgs<C> a, const SlabSyncArgs sy)
{
    stag_dslash_body<EPI, BLOCK, RECON, true>(a, &sy);
}

}  // namespace lqcd
