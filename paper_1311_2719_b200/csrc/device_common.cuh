// device_common.cuh -- lattice geometry, complex arithmetic and cache-hinted loads shared by
// the Dslash kernels.  Index convention: include/lqcd.h.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace lqcd {

typedef double2 cplx;  // (re, im): one 128-bit load/store per complex number

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

// ------------------------------------------------------------------ loads / stores
// Links are read exactly once per Dslash and the field (0.6-6 GB) does not fit the 126 MB L2:
// stream them (evict-first, no L1 allocation) so they do not push the vectors out.
__device__ __forceinline__ cplx ld_stream(const cplx* p)
{
    cplx v;
    asm volatile("ld.global.cs.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
    return v;
}
// Vectors are re-read by up to 8 neighbouring sites: read-only path, keep in L1/L2.
__device__ __forceinline__ cplx ld_keep(const cplx* p) { return __ldg(p); }
__device__ __forceinline__ void st_vec(cplx* p, cplx v) { *p = v; }

// ------------------------------------------------------------------ complex helpers
__device__ __forceinline__ cplx cmake(double re, double im) { return make_double2(re, im); }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return cmake(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return cmake(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cscale(double s, cplx a) { return cmake(s * a.x, s * a.y); }
__device__ __forceinline__ double cnorm2(cplx a) { return fma(a.x, a.x, a.y * a.y); }
// acc += a * b
__device__ __forceinline__ void cfma(cplx& acc, cplx a, cplx b)
{
    acc.x = fma(a.x, b.x, acc.x);
    acc.x = fma(-a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y);
    acc.y = fma(a.y, b.x, acc.y);
}
// acc += conj(a) * b
__device__ __forceinline__ void cfma_conj(cplx& acc, cplx a, cplx b)
{
    acc.x = fma(a.x, b.x, acc.x);
    acc.x = fma(a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y);
    acc.y = fma(-a.y, b.x, acc.y);
}
// multiplication by i^K
template <int K>
__device__ __forceinline__ cplx mul_i_pow(cplx a)
{
    if (K == 0) return a;
    if (K == 1) return cmake(-a.y, a.x);
    if (K == 2) return cmake(-a.x, -a.y);
    return cmake(a.y, -a.x);
}

}  // namespace lqcd
