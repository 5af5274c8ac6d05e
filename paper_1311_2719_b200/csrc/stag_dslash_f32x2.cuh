// stag_dslash_f32x2.cuh -- the fp32 staggered hopping term of the mixed-precision solver
// with TWO neighbouring sites per thread and 128-bit loads.
//
// Why: with one site per thread an fp32 complex number is a 64-bit load, a warp-wide request carries
// 256 bytes, and the kernel stalls at 56-58 % of the DRAM peak whatever the occupancy (profiles/:
// the number of requests in flight per SM is the limit, not their bytes).  A thread that owns the
// sites e = 2j and 2j+1 of a row reads (re, im, re, im) of both with one 128-bit load: the same bytes
// in half the requests.  For mu >= 1 the neighbours of the pair are again an aligned pair; for
// mu = 0 the neighbour pair is shifted by one site in one of the two directions (which one depends
// on the row's x0 parity), so those loads -- 1 hop in 8 -- stay 64-bit.
//
// Needs L0 % 4 == 0 (pairs must not straddle rows); other lattices keep the one-site kernel.
// Per-site arithmetic and its order are those of stag_hop (stag_dslash.cuh): the two kernels give
// bit-identical vectors; only the grouping of the partial sums differs.
#pragma once
#include "stag_dslash.cuh"

namespace lqcd {

__device__ __forceinline__ float4 ld_stream4(const float2* p)
{
    float4 v;
    asm volatile("ld.global.cs.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ float4 ld_keep4(const float2* p) { return __ldg((const float4*)p); }
__device__ __forceinline__ void split(float4 q, float2& a, float2& b)
{
    a = make_float2(q.x, q.y);
    b = make_float2(q.z, q.w);
}
__device__ __forceinline__ float4 join(float2 a, float2 b) { return make_float4(a.x, a.y, b.x, b.y); }

template <int MU, int RECON>
__device__ __forceinline__ void stag_hop2(const StagArgs<cplxf>& a, const Site& s, cplxf acc[2][3])
{
    constexpr int NC = RECON / 2;
    const size_t Vh = (size_t)a.g.Vh;
    const double eta = half_eta<MU>(s);  // the same for both sites of the pair (same row)
    const cplxf* Uf = a.gauge + (size_t)((a.parity * 4 + MU) * NC) * Vh + s.e;
    const cplxf* Ubase = a.gauge + (size_t)(((1 - a.parity) * 4 + MU) * NC) * Vh;
    cplxf U[2][9], W[2][9], vf[2][3], vb[2][3];
#pragma unroll
    for (int k = 0; k < NC; ++k) split(ld_stream4(Uf + k * Vh), U[0][k], U[1][k]);
    if (MU == 0) {
        // x0 = 2 xh + r: the forward neighbour of a site has half-index e (r = 0) or e + 1 (r = 1), the
        // backward one e - 1 (r = 0) or e (r = 1), wrapping inside the row
        const int ef0 = s.r ? s.e + 1 : s.e;
        const int ef1 = s.r ? (s.xh + 2 == a.g.Lh ? s.e + 2 - a.g.Lh : s.e + 2) : s.e + 1;
        const int eb0 = s.r ? s.e : (s.xh == 0 ? s.e + a.g.Lh - 1 : s.e - 1);
        const int eb1 = s.r ? s.e + 1 : s.e;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            vf[0][c] = ld_keep(a.in + c * Vh + ef0);
            vf[1][c] = ld_keep(a.in + c * Vh + ef1);
        }
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            W[0][k] = ld_stream(Ubase + k * Vh + eb0);
            W[1][k] = ld_stream(Ubase + k * Vh + eb1);
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            vb[0][c] = ld_keep(a.in + c * Vh + eb0);
            vb[1][c] = ld_keep(a.in + c * Vh + eb1);
        }
    } else {
        const int ef = nbr_fwd<MU>(a.g, s);  // even: strides and wraps are multiples of Lh, and Lh is even
        const int eb = nbr_bwd<MU>(a.g, s);
#pragma unroll
        for (int c = 0; c < 3; ++c) split(ld_keep4(a.in + c * Vh + ef), vf[0][c], vf[1][c]);
#pragma unroll
        for (int k = 0; k < NC; ++k) split(ld_stream4(Ubase + k * Vh + eb), W[0][k], W[1][k]);
#pragma unroll
        for (int c = 0; c < 3; ++c) split(ld_keep4(a.in + c * Vh + eb), vb[0][c], vb[1][c]);
    }
    const double sf = eta * bc_fwd<MU>(a.g, s);
    const double sb = -eta * bc_bwd<MU>(a.g, s);
#pragma unroll
    for (int i = 0; i < 2; ++i) {
        reconstruct_link<RECON>(U[i]);
        reconstruct_link<RECON>(W[i]);
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            vf[i][c] = cscale(sf, vf[i][c]);
            vb[i][c] = cscale(sb, vb[i][c]);
        }
#pragma unroll
        for (int r = 0; r < 3; ++r) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                cfma(acc[i][r], U[i][r * 3 + c], vf[i][c]);
                cfma_conj(acc[i][r], W[i][c * 3 + r], vb[i][c]);
            }
        }
    }
}

#ifndef LQCD_STAG_MINB_F32X2
#define LQCD_STAG_MINB_F32X2 4
#endif

// EPI = SE_NORM (S1 + S2) or SE_CGUPDATE_MIXED (S3 of the fp32 inner iteration).
template <int EPI, int BLOCK, int RECON>
__global__ void __launch_bounds__(BLOCK, LQCD_STAG_MINB_F32X2) stag_dslash_f32x2_kernel(const StagArgs<cplxf> a)
{
    static_assert(EPI == SE_NORM || EPI == SE_CGUPDATE_MIXED, "only the two kernels of the fp32 iteration");
    if (a.sc->done | a.sc->pause) return;
    const int e = 2 * (blockIdx.x * BLOCK + threadIdx.x);
    const bool active = e < a.g.Vh;
    const size_t Vh = (size_t)a.g.Vh;
    cplxf acc[2][3];
#pragma unroll
    for (int i = 0; i < 2; ++i)
#pragma unroll
        for (int c = 0; c < 3; ++c) acc[i][c] = czero<cplxf>();
    if (active) {
        const Site s = decode_site(a.g, a.parity, e);
        stag_hop2<0, RECON>(a, s, acc);
        stag_hop2<1, RECON>(a, s, acc);
        stag_hop2<2, RECON>(a, s, acc);
        stag_hop2<3, RECON>(a, s, acc);
    }
    double local = 0.0;
    if (EPI == SE_NORM) {
        if (active) {
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                *(float4*)(a.out + c * Vh + e) = join(acc[0][c], acc[1][c]);
                local += cnorm2(acc[0][c]);
                local += cnorm2(acc[1][c]);
            }
        }
        CgScalars* sc = a.sc;
        const double m2 = a.m2;
        grid_sum<BLOCK>(local, a.rs, [sc, m2](double tt) {
            sc->tt = tt;
            sc->alpha = sc->rr / (m2 * sc->pp + tt);  // <p,Ap> from norms only
        });
    } else {
        if (active) {
            const double alpha = a.sc->alpha;
            // all operands loaded before the first store (see SE_CGUPDATE in stag_dslash.cuh)
            float4 pq[3], xq[3], rq[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const size_t i = c * Vh + e;
                pq[c] = *(const float4*)(a.p + i);
                xq[c] = *(const float4*)(a.x + i);
                rq[c] = *(const float4*)(a.r + i);
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const size_t i = c * Vh + e;
                cplxf p2[2], x2[2], r2[2];
                split(pq[c], p2[0], p2[1]);
                split(xq[c], x2[0], x2[1]);
                split(rq[c], r2[0], r2[1]);
#pragma unroll
                for (int k = 0; k < 2; ++k) {
                    const double2 pv = to_d(p2[k]), q = to_d(acc[k][c]);
                    double2 xv = to_d(x2[k]), rv = to_d(r2[k]);
                    const double2 ap = cmake(fma(a.m2, pv.x, -q.x), fma(a.m2, pv.y, -q.y));
                    xv.x = fma(alpha, pv.x, xv.x);   // x = x + alpha p
                    xv.y = fma(alpha, pv.y, xv.y);
                    rv.x = fma(-alpha, ap.x, rv.x);  // r = r - alpha atap
                    rv.y = fma(-alpha, ap.y, rv.y);
                    x2[k] = to_cplx(xv, (cplxf*)0);
                    r2[k] = to_cplx(rv, (cplxf*)0);
                    local += cnorm2(r2[k]);          // betan = <r,r>
                }
                *(float4*)(a.x + i) = join(x2[0], x2[1]);
                *(float4*)(a.r + i) = join(r2[0], r2[1]);
            }
        }
        CgScalars* sc = a.sc;
        double* hist = a.hist;
        grid_sum<BLOCK>(local, a.rs, [sc, hist](double rr_new) { cg_after_update_mixed(sc, hist, rr_new); });
    }
}

// S5 of the fp32 iteration with 128-bit accesses: p = r + beta p on pairs of complex numbers (n even).
template <int BLOCK>
__global__ void __launch_bounds__(BLOCK) cg_pupdate_f32x2_kernel(const cplxf* __restrict__ r, cplxf* __restrict__ p, size_t n,
                                                                 CgScalars* sc, ReduceScratch rs)
{
    if (sc->done | sc->pause) return;
    const double beta = sc->beta;
    double local = 0.0;
    const size_t n2 = n / 2;
    for (size_t j = (size_t)blockIdx.x * BLOCK + threadIdx.x; j < n2; j += (size_t)gridDim.x * BLOCK) {
        cplxf r2[2], p2[2];
        split(*(const float4*)(r + 2 * j), r2[0], r2[1]);
        split(*(const float4*)(p + 2 * j), p2[0], p2[1]);
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            const double2 rv = to_d(r2[k]);
            double2 pv = to_d(p2[k]);
            pv.x = fma(beta, pv.x, rv.x);
            pv.y = fma(beta, pv.y, rv.y);
            p2[k] = to_cplx(pv, (cplxf*)0);
            local += cnorm2(p2[k]);
        }
        *(float4*)(p + 2 * j) = join(p2[0], p2[1]);
    }
    grid_sum<BLOCK>(local, rs, [sc](double pp) { sc->pp = pp; });
}

}  // namespace lqcd
