// wilson_dslash.cuh -- Wilson hopping term with fused CG epilogues.
//
//   (D_W psi)(x) = sum_mu [ (1-gamma_mu) b+ U_mu(x) psi(x+mu^) + (1+gamma_mu) b- U_mu(x-mu^)^+ psi(x-mu^) ]
//   M = 1 - kappa D_W,   M^+ = gamma5 M gamma5 = 1 - kappa D_W^+,  D_W^+ = the same sum with the
//   projector signs exchanged (gamma5 gamma_mu gamma5 = -gamma_mu).
//
// The paper only mentions its Wilson program; the operator is BASELINE.json
// config 4's (DeGrand-Rossi basis).  In that basis every gamma_mu couples the upper spin pair
// (0,1) to the lower pair (2,3) with entries among +-1, +-i:  (gamma psi)_s = i^K_s psi_{pi(s)}.
// Hence (1 -+ gamma) psi has two independent spin components h_s = psi_s -+ i^K_s psi_pi(s),
// s = 0,1, and its lower components are -+ conj(i^K_s) h_s at spin pi(s): only two SU(3)
// matrix-vector products per hop instead of four.
//
// One thread per output site; full-lattice structure-of-arrays vectors v[spin][c][g].
#pragma once
#include "reduce.cuh"

// Minimum resident blocks per SM.  Left alone ptxas takes 132-148 registers (3 blocks of 128 threads per
// SM); capped at 128 registers a fourth block fits and the CG on 16^3 x 32 runs 16 % faster (sweep on
// B200, cfg 4, us per iteration at 1..6 blocks: 145.2 145.0 146.0 122.2 141.7 160.5; profiles/r01_bench.md).
#ifndef LQCD_WILSON_MINB
#define LQCD_WILSON_MINB 4
#endif
// Components per batch of the epilogue's loads (all loads of a batch precede its first store): one vector
// (M, M + norm) and two vectors (the update of r) per component.
#ifndef LQCD_WILSON_EPI_BATCH_M
#define LQCD_WILSON_EPI_BATCH_M 6
#endif
#ifndef LQCD_WILSON_EPI_BATCH_U
#define LQCD_WILSON_EPI_BATCH_U 6
#endif

namespace lqcd {

enum WilsonEpilogue {
    WE_PLAIN = 0,     // out = D in on one parity                               (lqcd_dslash)
    WE_M = 1,         // out = in - kappa D in, full lattice
    WE_M_NORM = 2,    // the same + tt = |out|^2, alpha = rr/tt                 (S1, S2: <p,Ap> = |Mp|^2)
    WE_CGUPDATE = 3,  // Ap = in - kappa D^+ in; r -= alpha Ap; |r|^2   (S3; its x += alpha p: cg_xpupdate_kernel)
    WE_RESIDUAL = 4,  // |b - (in - kappa D^+ in)|^2                            (S7)
    // One-parity kernels of the even-odd (Schur) preconditioned solver, SURVEY.md 8(f) row 4.  `p` is the
    // site-diagonal operand on the output parity, `kappa` carries the coefficient c of  d = p + c * (D in):
    // c = -kappa^2 for Mhat = 1 - kappa^2 D_eo D_oe, c = +kappa for the source preparation and the
    // reconstruction, c = -kappa for the rows of M itself.
    WE_EO_XPAY = 5,       // out = d
    WE_EO_XPAY_NORM = 6,  // out = d, tt = |d|^2, alpha = rr/tt                 (<p, Mhat^+ Mhat p> = |Mhat p|^2)
    WE_EO_CGUPDATE = 7,   // Ap = d; r -= alpha Ap; |r|^2                       (x += alpha q: cg_xpupdate_kernel)
    WE_EO_RESIDUAL = 8    // |b - d|^2 and |b|^2 of one parity, set (flag = 0) or added (flag = 1)
};
__host__ __device__ constexpr bool wilson_one_parity(int epi) { return epi == WE_PLAIN || epi >= WE_EO_XPAY; }

struct WilsonArgs {
    Geom g;
    int parity;         // WE_PLAIN: output parity.  Other epilogues cover both parities.
    const cplx* gauge;  // [2][4][RECON/2][Vh]
    const cplx* in;     // [4][3][V]
    cplx* out;          // [4][3][V]
    const cplx* p;
    cplx* x;
    cplx* r;
    const cplx* b;
    double kappa;
    int flag;
    CgScalars* sc;
    ReduceScratch rs;
    double* hist;
};

// gamma_mu in the DeGrand-Rossi basis: (gamma psi)_s = i^K psi_PI for the upper rows s = 0, 1.
template <int MU> struct GammaDR;
template <> struct GammaDR<0> { static constexpr int PI0 = 3, K0 = 1, PI1 = 2, K1 = 1; };  // rows (0,0,0,i), (0,0,i,0)
template <> struct GammaDR<1> { static constexpr int PI0 = 3, K0 = 2, PI1 = 2, K1 = 0; };  // rows (0,0,0,-1), (0,0,1,0)
template <> struct GammaDR<2> { static constexpr int PI0 = 2, K0 = 1, PI1 = 3, K1 = 3; };  // rows (0,0,i,0), (0,0,0,-i)
template <> struct GammaDR<3> { static constexpr int PI0 = 2, K0 = 0, PI1 = 3, K1 = 0; };  // rows (0,0,1,0), (0,0,0,1)

// One hop.  PLUS = false: projector (1 - gamma_mu); PLUS = true: (1 + gamma_mu).
// ADJ = false: multiply by U (forward link at x); ADJ = true: by U^+ (link at x - mu^).
template <int MU, bool PLUS, bool ADJ>
__device__ __forceinline__ void wilson_hop_math(const cplx U[9], const cplx psi[4][3], double sign, cplx acc[4][3])
{
    typedef GammaDR<MU> G;
    // h_s = psi_s -+ i^K psi_pi(s)
    constexpr int KH0 = PLUS ? G::K0 : (G::K0 + 2) & 3;
    constexpr int KH1 = PLUS ? G::K1 : (G::K1 + 2) & 3;
    // lower components: -+ conj(i^K) (U h)_s at spin pi(s)
    constexpr int KL0 = PLUS ? (4 - G::K0) & 3 : (6 - G::K0) & 3;
    constexpr int KL1 = PLUS ? (4 - G::K1) & 3 : (6 - G::K1) & 3;
    cplx h0[3], h1[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        h0[c] = cscale(sign, cadd(psi[0][c], mul_i_pow<KH0>(psi[G::PI0][c])));
        h1[c] = cscale(sign, cadd(psi[1][c], mul_i_pow<KH1>(psi[G::PI1][c])));
    }
#pragma unroll
    for (int r = 0; r < 3; ++r) {
        cplx u0 = czero<cplx>(), u1 = czero<cplx>();
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            if (ADJ) {
                cfma_conj(u0, U[c * 3 + r], h0[c]);
                cfma_conj(u1, U[c * 3 + r], h1[c]);
            } else {
                cfma(u0, U[r * 3 + c], h0[c]);
                cfma(u1, U[r * 3 + c], h1[c]);
            }
        }
        acc[0][r] = cadd(acc[0][r], u0);
        acc[1][r] = cadd(acc[1][r], u1);
        acc[G::PI0][r] = cadd(acc[G::PI0][r], mul_i_pow<KL0>(u0));
        acc[G::PI1][r] = cadd(acc[G::PI1][r], mul_i_pow<KL1>(u1));
    }
}

// VL: how the spinor is loaded (device_common.cuh).  The one-parity kernels are also launched with in == out
// (the even-odd solver keeps an intermediate in the other half of the same array: reads go to one parity, writes
// to the other, never to a shared 128-byte line) -- legal for ordinary loads, not for the read-only path, whose
// contract is that the kernel writes nothing it reads through it: they take VL_PLAIN and no __restrict__.
template <int MU, bool PLUS, bool ADJ, int RECON, int LINKS, int VL>
__device__ __forceinline__ void wilson_hop(const cplx* __restrict__ link, size_t Vh, const cplx* src,
                                           size_t V, double sign, cplx acc[4][3])
{
    cplx U[9], psi[4][3];
    load_link<RECON, cplx, LINKS>(link, Vh, U);
#pragma unroll
    for (int s = 0; s < 4; ++s)
#pragma unroll
        for (int c = 0; c < 3; ++c) psi[s][c] = ld_vec<VL>(src + (size_t)(s * 3 + c) * V);
    reconstruct_link<RECON>(U);
    wilson_hop_math<MU, PLUS, ADJ>(U, psi, sign, acc);
}

template <int MU, bool DAGGER, int RECON, int LINKS, int VL>
__device__ __forceinline__ void wilson_dir(const WilsonArgs& a, const Site& s, int parity, cplx acc[4][3])
{
    const size_t Vh = (size_t)a.g.Vh, V = (size_t)a.g.V;
    const int ef = nbr_fwd<MU>(a.g, s);
    const int eb = nbr_bwd<MU>(a.g, s);
    const size_t other = (size_t)(1 - parity) * Vh;
    const cplx* Uf = a.gauge + (size_t)((parity * 4 + MU) * (RECON / 2)) * Vh + s.e;
    const cplx* Ub = a.gauge + (size_t)(((1 - parity) * 4 + MU) * (RECON / 2)) * Vh + eb;
    // D: forward (1-gamma), backward (1+gamma);  D^+: forward (1+gamma), backward (1-gamma)
    wilson_hop<MU, DAGGER, false, RECON, LINKS, VL>(Uf, Vh, a.in + other + ef, V, bc_fwd<MU>(a.g, s), acc);
    wilson_hop<MU, !DAGGER, true, RECON, LINKS, VL>(Ub, Vh, a.in + other + eb, V, bc_bwd<MU>(a.g, s), acc);
}

// Which site a thread owns.  One-parity kernels cover the Vh sites of a.parity.  The full-lattice kernels
// alternate the parities block by block (block 2k: tile k of the even sites, block 2k+1: tile k of the odd
// sites), so that U_mu(x) is read as the forward link of x and as the backward link of x+mu^ within a short
// time: with links loaded through L2 (LP_L2) the second use hits, and a full-lattice operator moves 576
// instead of 1152 bytes of links per site from HBM (ncu at 16^3 x 32: 100.7 MB read by the M kernel =
// 75.5 MB of links + 25.2 MB of p, against 160 MB with the parities one after the other and evict-first links).
template <int EPI, int BLOCK>
__device__ __forceinline__ bool wilson_thread_site(const WilsonArgs& a, int& parity, int& e)
{
    if (wilson_one_parity(EPI)) {
        parity = a.parity;
        e = blockIdx.x * BLOCK + threadIdx.x;
    } else {
        parity = blockIdx.x & 1;
        e = (blockIdx.x >> 1) * BLOCK + threadIdx.x;
    }
    return e < a.g.Vh;
}
__host__ __device__ constexpr bool wilson_full_lattice(int epi) { return !wilson_one_parity(epi); }

// Everything after the eight hops: the site-diagonal term, the fused CG updates and the grid-wide sums.
template <int EPI, int BLOCK>
__device__ __forceinline__ void wilson_epilogue(const WilsonArgs& a, bool active, size_t gsite, cplx acc[4][3])
{
    const size_t V = (size_t)a.g.V;
    if (EPI == WE_PLAIN) {
        if (active) {
#pragma unroll
            for (int k = 0; k < 12; ++k) st_vec(a.out + (size_t)k * V + gsite, acc[k / 3][k % 3]);
        }
        return;
    }
    if (EPI >= WE_EO_XPAY) {
        // one-parity forms: d = p + c * acc (operands loaded in batches before the stores, as below)
        double local[2] = { 0.0, 0.0 };
        if (active) {
            if (EPI == WE_EO_CGUPDATE) {
                // r -= alpha Ap, |r|^2; x += alpha q is done by cg_xpupdate_kernel (q = the search direction it updates)
                const double alpha = a.sc->alpha;
                constexpr int NB = LQCD_WILSON_EPI_BATCH_U;
#pragma unroll
                for (int h = 0; h < 12 / NB; ++h) {
                    cplx c0[NB], rv[NB];
#pragma unroll
                    for (int j = 0; j < NB; ++j) {
                        const size_t i = (size_t)(h * NB + j) * V + gsite;
                        c0[j] = a.p[i];
                        rv[j] = a.r[i];
                    }
#pragma unroll
                    for (int j = 0; j < NB; ++j) {
                        const int k = h * NB + j;
                        const cplx d = cmake(fma(a.kappa, acc[k / 3][k % 3].x, c0[j].x), fma(a.kappa, acc[k / 3][k % 3].y, c0[j].y));
                        rv[j].x = fma(-alpha, d.x, rv[j].x);
                        rv[j].y = fma(-alpha, d.y, rv[j].y);
                        a.r[(size_t)k * V + gsite] = rv[j];
                        local[0] += cnorm2(rv[j]);
                    }
                }
            } else {
                cplx c0[12];
#pragma unroll
                for (int k = 0; k < 12; ++k) c0[k] = a.p[(size_t)k * V + gsite];
#pragma unroll
                for (int k = 0; k < 12; ++k) {
                    const size_t i = (size_t)k * V + gsite;
                    const cplx d = cmake(fma(a.kappa, acc[k / 3][k % 3].x, c0[k].x), fma(a.kappa, acc[k / 3][k % 3].y, c0[k].y));
                    if (EPI == WE_EO_XPAY || EPI == WE_EO_XPAY_NORM) {
                        st_vec(a.out + i, d);
                        if (EPI == WE_EO_XPAY_NORM) local[0] += cnorm2(d);
                    } else {  // WE_EO_RESIDUAL
                        const cplx bv = a.b[i];
                        const double re = bv.x - d.x, im = bv.y - d.y;
                        local[0] += fma(re, re, im * im);
                        local[1] += cnorm2(bv);
                    }
                }
            }
        }
        CgScalars* sc = a.sc;
        if (EPI == WE_EO_XPAY_NORM) {
            grid_sum<BLOCK>(local[0], a.rs, [sc](double tt) {
                sc->tt = tt;
                sc->alpha = sc->rr / tt;
            });
        } else if (EPI == WE_EO_CGUPDATE) {
            double* hist = a.hist;
            grid_sum<BLOCK>(local[0], a.rs, [sc, hist](double rr_new) {
                cg_after_update(sc, hist, rr_new);
                sc->xdue = 1;
            });
        } else if (EPI == WE_EO_RESIDUAL) {
            const int add = a.flag;
            grid_sum_n<BLOCK, 2>(local, a.rs, [sc, add](const double (&tot)[2]) {
                sc->res2 = add ? sc->res2 + tot[0] : tot[0];
                sc->aux = add ? sc->aux + tot[1] : tot[1];
            });
        }
        return;
    }
    // M-type: m = in(x) - kappa * acc.  The operands of a batch are all loaded before the first store of that
    // batch: `in`, `out`, `r` may alias as far as the compiler can tell, so a load placed after a store waits
    // for it -- component by component that was twelve serial round trips to L2 per thread (ncu, round 2).
    double local = 0.0;
    if (EPI == WE_M || EPI == WE_M_NORM) {
        if (active) {
            constexpr int NB = LQCD_WILSON_EPI_BATCH_M;
#pragma unroll
            for (int h = 0; h < 12 / NB; ++h) {
                cplx c0[NB];
#pragma unroll
                for (int j = 0; j < NB; ++j) c0[j] = a.in[(size_t)(h * NB + j) * V + gsite];
#pragma unroll
                for (int j = 0; j < NB; ++j) {
                    const int k = h * NB + j;
                    const cplx m = cmake(fma(-a.kappa, acc[k / 3][k % 3].x, c0[j].x), fma(-a.kappa, acc[k / 3][k % 3].y, c0[j].y));
                    st_vec(a.out + (size_t)k * V + gsite, m);
                    if (EPI == WE_M_NORM) local += cnorm2(m);
                }
            }
        }
    } else if (EPI == WE_CGUPDATE) {
        // r -= alpha Ap, |r|^2.  x += alpha p is done by the vector kernel that follows (cg_xpupdate_kernel): it reads p
        // anyway, so the search direction is not read here at all (192 B per site less than in round 1).
        if (active) {
            const double alpha = a.sc->alpha;
            constexpr int NB = LQCD_WILSON_EPI_BATCH_U;
#pragma unroll
            for (int h = 0; h < 12 / NB; ++h) {
                cplx c0[NB], rv[NB];
#pragma unroll
                for (int j = 0; j < NB; ++j) {
                    const size_t i = (size_t)(h * NB + j) * V + gsite;
                    c0[j] = a.in[i];
                    rv[j] = a.r[i];
                }
#pragma unroll
                for (int j = 0; j < NB; ++j) {
                    const int k = h * NB + j;
                    const cplx m = cmake(fma(-a.kappa, acc[k / 3][k % 3].x, c0[j].x), fma(-a.kappa, acc[k / 3][k % 3].y, c0[j].y));
                    rv[j].x = fma(-alpha, m.x, rv[j].x);
                    rv[j].y = fma(-alpha, m.y, rv[j].y);
                    a.r[(size_t)k * V + gsite] = rv[j];
                    local += cnorm2(rv[j]);
                }
            }
        }
    } else {  // WE_RESIDUAL
        if (active) {
            cplx c0[12];
#pragma unroll
            for (int k = 0; k < 12; ++k) c0[k] = a.in[(size_t)k * V + gsite];
#pragma unroll
            for (int k = 0; k < 12; ++k) {
                const cplx m = cmake(fma(-a.kappa, acc[k / 3][k % 3].x, c0[k].x), fma(-a.kappa, acc[k / 3][k % 3].y, c0[k].y));
                const cplx bv = a.b[(size_t)k * V + gsite];
                const double re = bv.x - m.x, im = bv.y - m.y;
                local += fma(re, re, im * im);
            }
        }
    }
    CgScalars* sc = a.sc;
    if (EPI == WE_M_NORM) {
        grid_sum<BLOCK>(local, a.rs, [sc](double tt) {
            sc->tt = tt;
            sc->alpha = sc->rr / tt;  // <p, M^+M p> = |M p|^2
        });
    } else if (EPI == WE_CGUPDATE) {
        double* hist = a.hist;
        grid_sum<BLOCK>(local, a.rs, [sc, hist](double rr_new) {
            cg_after_update(sc, hist, rr_new);
            sc->xdue = 1;  // the x += alpha p of this iteration is still to be done
        });
    } else if (EPI == WE_RESIDUAL) {
        grid_sum<BLOCK>(local, a.rs, [sc](double res2) { sc->res2 = res2; });
    }
}

// LINKS: cache policy of the link loads (device_common.cuh).  Full-lattice kernels always LP_L2 (see
// wilson_thread_site); one-parity kernels read every link once per launch: LP_STREAM unless the whole field is
// small enough to stay in L2 from one launch to the next.
template <int EPI, bool DAGGER, int BLOCK, int RECON, int LINKS>
__global__ void __launch_bounds__(BLOCK, LQCD_WILSON_MINB) wilson_dslash_kernel(const WilsonArgs a)
{
    if (EPI == WE_M_NORM || EPI == WE_CGUPDATE || EPI == WE_EO_XPAY_NORM || EPI == WE_EO_CGUPDATE) {
        if (a.sc->done) return;
    }
    int parity, e;
    const bool active = wilson_thread_site<EPI, BLOCK>(a, parity, e);
    const size_t gsite = (size_t)parity * (size_t)a.g.Vh + (size_t)e;

    cplx acc[4][3];
#pragma unroll
    for (int s = 0; s < 4; ++s)
#pragma unroll
        for (int c = 0; c < 3; ++c) acc[s][c] = czero<cplx>();
    constexpr int VL = wilson_one_parity(EPI) ? VL_PLAIN : VL_NC;
    if (active) {
        const Site st = decode_site(a.g, parity, e);
        wilson_dir<0, DAGGER, RECON, LINKS, VL>(a, st, parity, acc);
        wilson_dir<1, DAGGER, RECON, LINKS, VL>(a, st, parity, acc);
        wilson_dir<2, DAGGER, RECON, LINKS, VL>(a, st, parity, acc);
        wilson_dir<3, DAGGER, RECON, LINKS, VL>(a, st, parity, acc);
    }
    wilson_epilogue<EPI, BLOCK>(a, active, gsite, acc);
}

}  // namespace lqcd
