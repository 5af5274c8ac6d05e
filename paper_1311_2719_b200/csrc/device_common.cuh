// device_common.cuh -- lattice geometry, complex arithmetic, link loading (with the optional
// two-row reconstruction) and cache-hinted loads shared by the Dslash kernels.
// Index convention: include/lqcd.h.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace lqcd {

// One complex number = one vector load/store: 128 bits in fp64, 64 bits in fp32 (the fp32
// types serve the inner iterations of the mixed-precision solver only).
template <class T> struct CplxOf;
template <> struct CplxOf<double> { typedef double2 type; };
template <> struct CplxOf<float> { typedef float2 type; };
typedef double2 cplx;   // fp64 complex, the precision of the path (reading A5)
typedef float2 cplxf;

// Half-lattice geometry.  A site of parity p is addressed by e = xh + Lh*(x1 + L1*(x2 + L2*x3)),
// xh = x0 >> 1, x0 = 2*xh + ((x1+x2+x3+p) & 1).
struct Geom {
    int Lh, L1, L2, L3;  // Lh = L0/2
    int s1, s2, s3;      // half-index strides of directions 1,2,3: Lh, Lh*L1, Lh*L1*L2
    int Vh;              // sites per parity
    long long V;         // all sites
};

struct Site {
    int e, xh, x1, x2, x3;
    int r;  // x0 & 1 = (x1+x2+x3+parity) & 1: constant along a row of the half lattice
};

__device__ __forceinline__ Site decode_site(const Geom& g, int parity, int e)
{
    Site s;
    s.e = e;
    int t = e / g.Lh;
    s.xh = e - t * g.Lh;
    int t2 = t / g.L1;
    s.x1 = t - t2 * g.L1;
    s.x3 = t2 / g.L2;
    s.x2 = t2 - s.x3 * g.L2;
    s.r = (s.x1 + s.x2 + s.x3 + parity) & 1;
    return s;
}

// Half-index (in the opposite parity) of the neighbour x + mu^ / x - mu^, periodic wrap.
template <int MU>
__device__ __forceinline__ int nbr_fwd(const Geom& g, const Site& s)
{
    if (MU == 0) return s.r ? (s.xh + 1 == g.Lh ? s.e - (g.Lh - 1) : s.e + 1) : s.e;
    if (MU == 1) return s.x1 + 1 == g.L1 ? s.e - (g.L1 - 1) * g.s1 : s.e + g.s1;
    if (MU == 2) return s.x2 + 1 == g.L2 ? s.e - (g.L2 - 1) * g.s2 : s.e + g.s2;
    return s.x3 + 1 == g.L3 ? s.e - (g.L3 - 1) * g.s3 : s.e + g.s3;
}
template <int MU>
__device__ __forceinline__ int nbr_bwd(const Geom& g, const Site& s)
{
    if (MU == 0) return s.r ? s.e : (s.xh == 0 ? s.e + (g.Lh - 1) : s.e - 1);
    if (MU == 1) return s.x1 == 0 ? s.e + (g.L1 - 1) * g.s1 : s.e - g.s1;
    if (MU == 2) return s.x2 == 0 ? s.e + (g.L2 - 1) * g.s2 : s.e - g.s2;
    return s.x3 == 0 ? s.e + (g.L3 - 1) * g.s3 : s.e - g.s3;
}

// Antiperiodic time boundary: -1 on the hop that crosses x3 = L3-1 <-> 0.
template <int MU>
__device__ __forceinline__ double bc_fwd(const Geom& g, const Site& s)
{
    return (MU == 3 && s.x3 + 1 == g.L3) ? -1.0 : 1.0;
}
template <int MU>
__device__ __forceinline__ double bc_bwd(const Geom& g, const Site& s)
{
    return (MU == 3 && s.x3 == 0) ? -1.0 : 1.0;
}

// Staggered phase eta_mu(x) / 2 (reading A3) from the decoded site.
template <int MU>
__device__ __forceinline__ double half_eta(const Site& s)
{
    if (MU == 0) return 0.5;
    if (MU == 1) return s.r ? -0.5 : 0.5;
    if (MU == 2) return ((s.r + s.x1) & 1) ? -0.5 : 0.5;
    return ((s.r + s.x1 + s.x2) & 1) ? -0.5 : 0.5;
}

// ------------------------------------------------------------------ loads / stores
// Links are read exactly once per Dslash and the field (0.6-6 GB) does not fit the 126 MB L2:
// stream them (evict-first, no L1 allocation) so they do not push the vectors out.
__device__ __forceinline__ double2 ld_stream(const double2* p)
{
    double2 v;
    asm volatile("ld.global.cs.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
__device__ __forceinline__ float2 ld_stream(const float2* p)
{
    float2 v;
    asm volatile("ld.global.cs.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}
// Link loads by cache policy.  LP_STREAM: as above (fields larger than L2).  LP_L2: through L2 with normal
// eviction and no L1 allocation -- for fields that FIT in L2 and are read by both parities of a full-lattice
// operator (each link is the forward link of x and the backward link of x+mu^), so the second use and every
// later iteration hits L2.  LP_DEFAULT: ordinary loads that also allocate in L1 -- for the one-kernel CG loop
// (cg_persistent.cuh), whose links are re-read by the same block every iteration.  (An evict-last L2 policy
// and a persisting-L2 window were measured and dropped: DESIGN.md.)
enum LinkPolicy { LP_STREAM = 0, LP_L2 = 1, LP_DEFAULT = 2 };
template <int POLICY>
__device__ __forceinline__ double2 ld_link(const double2* p)
{
    double2 v;
    if (POLICY == LP_L2)
        asm volatile("ld.global.cg.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    else if (POLICY == LP_DEFAULT)
        asm volatile("ld.global.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    else
        asm volatile("ld.global.cs.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
template <int POLICY>
__device__ __forceinline__ float2 ld_link(const float2* p)
{
    float2 v;
    if (POLICY == LP_L2)
        asm volatile("ld.global.cg.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    else if (POLICY == LP_DEFAULT)
        asm volatile("ld.global.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    else
        asm volatile("ld.global.cs.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}
// Vectors are re-read by up to 8 neighbouring sites: read-only path, keep in L1/L2.
__device__ __forceinline__ double2 ld_keep(const double2* p) { return __ldg(p); }
__device__ __forceinline__ float2 ld_keep(const float2* p) { return __ldg(p); }
// Vector loads by coherence need.  VL_NC: the read-only (non-coherent) path -- only for data no block of the
// running kernel writes.  VL_PLAIN: ordinary L1-allocating loads, for kernels that read what other blocks of
// the SAME launch wrote before a grid-wide barrier (cg_persistent.cuh; the barrier's fences invalidate L1).
enum VecLoad { VL_NC = 0, VL_PLAIN = 1 };
template <int VL, class C>
__device__ __forceinline__ C ld_vec(const C* p)
{
    if (VL == VL_PLAIN) return *p;
    return __ldg(p);
}
template <class C>
__device__ __forceinline__ void st_vec(C* p, C v) { *p = v; }
// x is read and written exactly once per CG iteration: stream it past the caches.
__device__ __forceinline__ void st_stream(double2* p, double2 v)
{
    asm volatile("st.global.cs.v2.f64 [%0], {%1, %2};" ::"l"(p), "d"(v.x), "d"(v.y) : "memory");
}
__device__ __forceinline__ void st_stream(float2* p, float2 v)
{
    asm volatile("st.global.cs.v2.f32 [%0], {%1, %2};" ::"l"(p), "f"(v.x), "f"(v.y) : "memory");
}

// ------------------------------------------------------------------ complex helpers
__device__ __forceinline__ double2 cmake(double re, double im) { return make_double2(re, im); }
__device__ __forceinline__ float2 cmake(float re, float im) { return make_float2(re, im); }
template <class C> __device__ __forceinline__ C czero() { C z; z.x = 0; z.y = 0; return z; }
template <class C> __device__ __forceinline__ C cadd(C a, C b) { return cmake(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ double2 cscale(double s, double2 a) { return cmake(s * a.x, s * a.y); }
__device__ __forceinline__ float2 cscale(double s, float2 a) { return cmake((float)s * a.x, (float)s * a.y); }
// |a|^2, always returned (and summed by the caller) in fp64
__device__ __forceinline__ double cnorm2(double2 a) { return fma(a.x, a.x, a.y * a.y); }
__device__ __forceinline__ double cnorm2(float2 a) { return (double)a.x * (double)a.x + (double)a.y * (double)a.y; }
// acc += a * b
template <class C>
__device__ __forceinline__ void cfma(C& acc, C a, C b)
{
    acc.x = fma(a.x, b.x, acc.x);
    acc.x = fma(-a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y);
    acc.y = fma(a.y, b.x, acc.y);
}
// acc += conj(a) * b
template <class C>
__device__ __forceinline__ void cfma_conj(C& acc, C a, C b)
{
    acc.x = fma(a.x, b.x, acc.x);
    acc.x = fma(a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y);
    acc.y = fma(-a.y, b.x, acc.y);
}
// conj(a*b - c*d)
template <class C>
__device__ __forceinline__ C conj_cross(C a, C b, C c, C d)
{
    C r;
    r.x = fma(a.x, b.x, -(a.y * b.y));
    r.x = fma(-c.x, d.x, r.x);
    r.x = fma(c.y, d.y, r.x);
    r.y = fma(c.x, d.y, c.y * d.x);
    r.y = fma(-a.x, b.y, r.y);
    r.y = fma(-a.y, b.x, r.y);
    return r;
}
// multiplication by i^K
template <int K, class C>
__device__ __forceinline__ C mul_i_pow(C a)
{
    if (K == 0) return a;
    if (K == 1) return cmake(-a.y, a.x);
    if (K == 2) return cmake(-a.x, -a.y);
    return cmake(a.y, -a.x);
}
// fp64 <-> working precision
__device__ __forceinline__ double2 to_d(double2 a) { return a; }
__device__ __forceinline__ double2 to_d(float2 a) { return make_double2((double)a.x, (double)a.y); }
__device__ __forceinline__ double2 to_cplx(double2 a, double2*) { return a; }
__device__ __forceinline__ float2 to_cplx(double2 a, float2*) { return make_float2((float)a.x, (float)a.y); }

// ------------------------------------------------------------------ links
// Internal gauge layout: [parity][mu][NC][Vh] with NC = RECON/2 stored complex numbers per link.
// RECON = 18: all nine entries.  RECON = 12: the first two rows; the third row of an SU(3) matrix
// is the conjugated cross product of the first two ("two-column link compression",
// SURVEY.md 8(f) row 1): 96 instead of 144 bytes per link from HBM for 42 extra flops.
template <int RECON, class C, int POLICY = LP_STREAM>
__device__ __forceinline__ void load_link(const C* __restrict__ p, size_t Vh, C U[9])
{
    constexpr int NC = RECON / 2;
#pragma unroll
    for (int k = 0; k < NC; ++k) U[k] = ld_link<POLICY>(p + k * Vh);
}
// Kept apart from load_link so that a hop can issue all its loads before the first dependent flop.
template <int RECON, class C>
__device__ __forceinline__ void reconstruct_link(C U[9])
{
    if (RECON == 12) {
        U[6] = conj_cross(U[1], U[5], U[2], U[4]);
        U[7] = conj_cross(U[2], U[3], U[0], U[5]);
        U[8] = conj_cross(U[0], U[4], U[1], U[3]);
    }
}

}  // namespace lqcd
