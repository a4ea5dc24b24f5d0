// hr_common.cuh — geometry, device layout and small arithmetic helpers shared by the CUDA kernels
// of libhr_dslash.  Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <type_traits>

#include "../../include/hr_dslash.h"

namespace hr {

// ------------------------------------------------------------------ geometry
// Device layout.  A lattice site x = (x0,x1,x2,x3) has parity p = (x0+x1+x2+x3)&1,
// row = (x0*L1 + x1)*L2 + x2 and pair index h = x3/2; every row holds L3h = L3/2 sites of each parity.
// All fields are parity-split and blocked by row:
//   16-byte-chunk fields (spinor, compressed fund links, clover blocks):
//        chunk c of site (row,h) sits at 16-byte index (row*NCH + c)*L3h + h  of its parity half
//   adjoint links: 9 real planes per row,  real index (row*9 + k)*L3h + h
// so one x3-row of one field is a single contiguous run of NCH*L3h*16 bytes.
struct Geo {
    int L0, L1, L2, L3h;
    int R;    // rows = L0*L1*L2
    int Vh;   // sites per parity = R*L3h
    int s0;   // row stride of x0 = L1*L2
    int s1;   // row stride of x1 = L2
};

inline bool geom_ok(const hr_geom* g) {
    if (!g) return false;
    for (int m = 0; m < 4; ++m)
        if (g->L[m] < 2 || (g->L[m] & 1)) return false;
    double v = (double)g->L[0] * g->L[1] * g->L[2] * g->L[3];
    if (v > 2.0e9) return false;  // 32-bit site indices
    if (g->rep != HR_REP_FUND && g->rep != HR_REP_ADJ && g->rep != HR_REP_SU3) return false;
    if (g->rep == HR_REP_SU3 && g->link_storage == HR_LINKS_ONTHEFLY) return false;   // complex 3 x 3 links: all three rows, or the first two
    if (g->prec != HR_PREC_F64 && g->prec != HR_PREC_F32) return false;
    if (g->link_storage != HR_LINKS_FULL && g->link_storage != HR_LINKS_COMPRESSED && g->link_storage != HR_LINKS_ONTHEFLY) return false;
    if (g->link_storage == HR_LINKS_ONTHEFLY && g->rep != HR_REP_ADJ) return false;
    if (g->kernel < HR_KERNEL_AUTO || g->kernel > HR_KERNEL_TILED) return false;
    return true;
}

inline Geo make_geo(const hr_geom* g) {
    Geo o;
    o.L0 = g->L[0]; o.L1 = g->L[1]; o.L2 = g->L[2]; o.L3h = g->L[3] / 2;
    o.R = o.L0 * o.L1 * o.L2;
    o.Vh = o.R * o.L3h;
    o.s0 = o.L1 * o.L2;
    o.s1 = o.L2;
    return o;
}

inline size_t real_bytes(int prec) { return prec == HR_PREC_F64 ? 8 : 4; }
inline int ncolour(int rep) { return rep == HR_REP_FUND ? 2 : 3; }
// 16-byte chunks per spinor / compressed fundamental link / clover site (two blocks)
inline int spinor_chunks(int rep, int prec) { return 8 * ncolour(rep) * (int)real_bytes(prec) / 16; }
inline int link_chunks(int prec) { return 4 * (int)real_bytes(prec) / 16; }
inline int clover_chunks(int prec, int rep = HR_REP_FUND) { const int d = 2 * ncolour(rep); return 2 * d * d * (int)real_bytes(prec) / 16; }

// ------------------------------------------------------------------ complex numbers in registers
template <typename T>
struct cplx {
    T re, im;
};
template <typename T> __device__ __forceinline__ cplx<T> mk(T a, T b) { cplx<T> r; r.re = a; r.im = b; return r; }
template <typename T> __device__ __forceinline__ cplx<T> operator+(cplx<T> a, cplx<T> b) { return mk<T>(a.re + b.re, a.im + b.im); }
template <typename T> __device__ __forceinline__ cplx<T> operator-(cplx<T> a, cplx<T> b) { return mk<T>(a.re - b.re, a.im - b.im); }
template <typename T> __device__ __forceinline__ cplx<T> operator-(cplx<T> a) { return mk<T>(-a.re, -a.im); }
template <typename T> __device__ __forceinline__ cplx<T> operator*(cplx<T> a, cplx<T> b) {
    return mk<T>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re);
}
template <typename T> __device__ __forceinline__ cplx<T> operator*(T s, cplx<T> a) { return mk<T>(s * a.re, s * a.im); }
template <typename T> __device__ __forceinline__ cplx<T> conj(cplx<T> a) { return mk<T>(a.re, -a.im); }
// i*a and -i*a
template <typename T> __device__ __forceinline__ cplx<T> timesI(cplx<T> a) { return mk<T>(-a.im, a.re); }
template <typename T> __device__ __forceinline__ cplx<T> timesMinusI(cplx<T> a) { return mk<T>(a.im, -a.re); }
// acc += a*b ; acc += conj(a)*b
template <typename T> __device__ __forceinline__ void cmad(cplx<T>& acc, cplx<T> a, cplx<T> b) {
    acc.re = fma(a.re, b.re, acc.re); acc.re = fma(-a.im, b.im, acc.re);
    acc.im = fma(a.re, b.im, acc.im); acc.im = fma(a.im, b.re, acc.im);
}
template <typename T> __device__ __forceinline__ void cmadc(cplx<T>& acc, cplx<T> a, cplx<T> b) {
    acc.re = fma(a.re, b.re, acc.re); acc.re = fma(a.im, b.im, acc.re);
    acc.im = fma(a.re, b.im, acc.im); acc.im = fma(-a.im, b.re, acc.im);
}

// ------------------------------------------------------------------ 16-byte chunk access
template <typename T> struct Chunk;
template <> struct Chunk<double> { typedef double2 type; };
template <> struct Chunk<float> { typedef float4 type; };

// cache behaviour of a global access: spinors are re-read by neighbouring sites and should
// stay in L1/L2; links, clover blocks and outputs are touched once per kernel and are streamed.
enum { LD_KEEP = 0, LD_STREAM = 1, LD_NOALLOC = 2 };

template <int POLICY> __device__ __forceinline__ double2 ldg16(const double2* p) {
    if (POLICY == LD_STREAM) return __ldcs(p);
    if (POLICY == LD_NOALLOC) {
        double2 v;
        asm("ld.global.nc.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "l"(p));
        return v;
    }
    return __ldg(p);
}
template <int POLICY> __device__ __forceinline__ float4 ldg16(const float4* p) {
    if (POLICY == LD_STREAM) return __ldcs(p);
    if (POLICY == LD_NOALLOC) {
        float4 v;
        asm("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
        return v;
    }
    return __ldg(p);
}
template <int POLICY> __device__ __forceinline__ double ldg_real(const double* p) {
    if (POLICY != LD_KEEP) return __ldcs(p);
    return __ldg(p);
}
template <int POLICY> __device__ __forceinline__ float ldg_real(const float* p) {
    if (POLICY != LD_KEEP) return __ldcs(p);
    return __ldg(p);
}
// outputs are written once and not read again by the same kernel: streaming stores (plain stores measured 2-25 % slower,
// profiles/r01_tiled_variants.md)
__device__ __forceinline__ void stg16_stream(double2* p, double2 v) { __stcs(p, v); }
__device__ __forceinline__ void stg16_stream(float4* p, float4 v) { __stcs(p, v); }

__device__ __forceinline__ void chunk_to_reals(double2 v, double* e) { e[0] = v.x; e[1] = v.y; }
__device__ __forceinline__ void chunk_to_reals(float4 v, float* e) { e[0] = v.x; e[1] = v.y; e[2] = v.z; e[3] = v.w; }
__device__ __forceinline__ double2 reals_to_chunk(const double* e) { return make_double2(e[0], e[1]); }
__device__ __forceinline__ float4 reals_to_chunk(const float* e) { return make_float4(e[0], e[1], e[2], e[3]); }

// NC complex numbers of one site <-> NCH chunks at stride L3h (chunk index (row*NCH + c)*L3h + h)
template <typename T, int NC> struct SiteIO;
template <int NC> struct SiteIO<double, NC> {
    static constexpr int NCH = NC;
    template <int POLICY>
    static __device__ __forceinline__ void load(cplx<double>* s, const void* base, size_t first, int stride) {
        const double2* p = reinterpret_cast<const double2*>(base) + first;
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            double2 v = ldg16<POLICY>(p + (size_t)c * stride);
            s[c] = mk<double>(v.x, v.y);
        }
    }
    static __device__ __forceinline__ void store(void* base, size_t first, int stride, const cplx<double>* s) {
        double2* p = reinterpret_cast<double2*>(base) + first;
#pragma unroll
        for (int c = 0; c < NC; ++c) stg16_stream(p + (size_t)c * stride, make_double2(s[c].re, s[c].im));
    }
};
template <int NC> struct SiteIO<float, NC> {
    static_assert(NC % 2 == 0, "fp32 chunks hold two complex numbers");
    static constexpr int NCH = NC / 2;
    template <int POLICY>
    static __device__ __forceinline__ void load(cplx<float>* s, const void* base, size_t first, int stride) {
        const float4* p = reinterpret_cast<const float4*>(base) + first;
#pragma unroll
        for (int c = 0; c < NC / 2; ++c) {
            float4 v = ldg16<POLICY>(p + (size_t)c * stride);
            s[2 * c] = mk<float>(v.x, v.y);
            s[2 * c + 1] = mk<float>(v.z, v.w);
        }
    }
    static __device__ __forceinline__ void store(void* base, size_t first, int stride, const cplx<float>* s) {
        float4* p = reinterpret_cast<float4*>(base) + first;
#pragma unroll
        for (int c = 0; c < NC / 2; ++c)
            stg16_stream(p + (size_t)c * stride, make_float4(s[2 * c].re, s[2 * c].im, s[2 * c + 1].re, s[2 * c + 1].im));
    }
};

// ------------------------------------------------------------------ links in registers
// fundamental, compressed: first row (alpha, beta) of U = [[alpha, beta], [-conj(beta), conj(alpha)]]
// (exact for SU(2)).  adjoint: real 3x3.
template <typename T, int N> struct Link;
template <typename T> struct Link<T, 2> { cplx<T> a, b; };
template <typename T> struct Link<T, 3> { T r[9]; };
// complex 3 x 3 (HR_REP_SU3): row-major, m[3*row + col]
template <typename T> struct LinkC3 { cplx<T> m[9]; };

// chunk index of link (parity half `par`, direction mu, row, h): the gauge field is [par][mu][row][chunk][h]
template <typename T, int POLICY>
__device__ __forceinline__ void load_link(Link<T, 2>& u, const void* gauge, const Geo& g, int par, int mu, int row, int h) {
    cplx<T> ab[2];
    constexpr int LCH = SiteIO<T, 2>::NCH;
    size_t first = ((size_t)(par * 4 + mu) * g.R + row) * (LCH * g.L3h) + h;
    SiteIO<T, 2>::template load<POLICY>(ab, gauge, first, g.L3h);
    u.a = ab[0];
    u.b = ab[1];
}
template <typename T, int POLICY>
__device__ __forceinline__ void load_link(Link<T, 3>& u, const void* gauge, const Geo& g, int par, int mu, int row, int h) {
    const T* p = reinterpret_cast<const T*>(gauge) + ((size_t)(par * 4 + mu) * g.R + row) * (9 * g.L3h) + h;
#pragma unroll
    for (int k = 0; k < 9; ++k) u.r[k] = ldg_real<POLICY>(p + (size_t)k * g.L3h);
}

// ONFLY: the gauge field handed to the kernel is the fundamental one; an adjoint link is rebuilt in registers,
//   R_ab = (a0^2 - |a|^2) delta_ab + 2 a_a a_b + 2 a0 eps_abc a_c,   U = a0 + i a.sigma  (alpha = a0 + i a3, beta = a2 + i a1)
// — the closed form of R^{ab} = 1/2 tr(sigma_a U sigma_b U^dag) also used by represent_kernel.
template <typename T, int POLICY, bool ONFLY>
__device__ __forceinline__ void load_link_rep(Link<T, 2>& u, const void* gauge, const Geo& g, int par, int mu, int row, int h) {
    load_link<T, POLICY>(u, gauge, g, par, mu, row, h);
}
template <typename T, int POLICY, bool ONFLY>
__device__ __forceinline__ void load_link_rep(Link<T, 3>& u, const void* gauge, const Geo& g, int par, int mu, int row, int h) {
    if (!ONFLY) {
        load_link<T, POLICY>(u, gauge, g, par, mu, row, h);
        return;
    }
    Link<T, 2> f;
    load_link<T, POLICY>(f, gauge, g, par, mu, row, h);
    const T a0 = f.a.re, a3 = f.a.im, a2 = f.b.re, a1 = f.b.im;
    const T d = a0 * a0 - (a1 * a1 + a2 * a2 + a3 * a3);
    u.r[0] = d + 2 * a1 * a1;          u.r[1] = 2 * (a1 * a2 + a0 * a3);  u.r[2] = 2 * (a1 * a3 - a0 * a2);
    u.r[3] = 2 * (a2 * a1 - a0 * a3);  u.r[4] = d + 2 * a2 * a2;          u.r[5] = 2 * (a2 * a3 + a0 * a1);
    u.r[6] = 2 * (a3 * a1 + a0 * a2);  u.r[7] = 2 * (a3 * a2 - a0 * a1);  u.r[8] = d + 2 * a3 * a3;
}

// complex 3 x 3 links: NK complex planes per row, complex index (((par*4 + mu)*R + row)*NK + k)*L3h + h (128-bit loads in fp64,
// 64-bit in fp32).  TWOROWS = false: all nine entries stored (NK = 9).  TWOROWS = true (HR_LINKS_COMPRESSED): the first two rows are
// stored (NK = 6, 96 instead of 144 bytes in fp64) and the third is rebuilt in registers, row2 = conj(row0 x row1) — exact for
// det U = 1, U unitary, the usual two-row storage of SU(3) links.
template <typename T, int POLICY, bool TWOROWS>
__device__ __forceinline__ void load_link_rep(LinkC3<T>& u, const void* gauge, const Geo& g, int par, int mu, int row, int h) {
    typedef typename std::conditional<sizeof(T) == 8, double2, float2>::type pair_t;
    constexpr int NK = TWOROWS ? 6 : 9;
    const pair_t* p = reinterpret_cast<const pair_t*>(gauge) + ((size_t)(par * 4 + mu) * g.R + row) * (NK * g.L3h) + h;
#pragma unroll
    for (int k = 0; k < NK; ++k) {
        const pair_t v = POLICY == LD_KEEP ? __ldg(p + (size_t)k * g.L3h) : __ldcs(p + (size_t)k * g.L3h);
        u.m[k] = mk<T>(v.x, v.y);
    }
    if (TWOROWS) {
        u.m[6] = conj(u.m[1] * u.m[5] - u.m[2] * u.m[4]);
        u.m[7] = conj(u.m[2] * u.m[3] - u.m[0] * u.m[5]);
        u.m[8] = conj(u.m[0] * u.m[4] - u.m[1] * u.m[3]);
    }
}
template <typename T>
__device__ __forceinline__ void mul_link(cplx<T>* chi, const LinkC3<T>& u, const cplx<T>* h) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        chi[a] = u.m[3 * a] * h[0];
        cmad(chi[a], u.m[3 * a + 1], h[1]);
        cmad(chi[a], u.m[3 * a + 2], h[2]);
    }
}
template <typename T>
__device__ __forceinline__ void mul_link_dag(cplx<T>* chi, const LinkC3<T>& u, const cplx<T>* h) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        chi[a] = conj(u.m[a]) * h[0];
        cmadc(chi[a], u.m[3 + a], h[1]);
        cmadc(chi[a], u.m[6 + a], h[2]);
    }
}

// chi = U h  /  chi = U^dag h  on the colour index of one spin component
template <typename T>
__device__ __forceinline__ void mul_link(cplx<T>* chi, const Link<T, 2>& u, const cplx<T>* h) {
    // [ a  b ; -b* a* ]
    chi[0] = u.a * h[0]; cmad(chi[0], u.b, h[1]);
    chi[1] = conj(u.a) * h[1]; cmadc(chi[1], -u.b, h[0]);
}
template <typename T>
__device__ __forceinline__ void mul_link_dag(cplx<T>* chi, const Link<T, 2>& u, const cplx<T>* h) {
    // [ a* -b ; b* a ]
    chi[0] = conj(u.a) * h[0]; cmad(chi[0], -u.b, h[1]);
    chi[1] = u.a * h[1]; cmadc(chi[1], u.b, h[0]);
}
template <typename T>
__device__ __forceinline__ void mul_link(cplx<T>* chi, const Link<T, 3>& u, const cplx<T>* h) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        chi[a].re = u.r[a * 3] * h[0].re; chi[a].im = u.r[a * 3] * h[0].im;
#pragma unroll
        for (int b = 1; b < 3; ++b) {
            chi[a].re = fma(u.r[a * 3 + b], h[b].re, chi[a].re);
            chi[a].im = fma(u.r[a * 3 + b], h[b].im, chi[a].im);
        }
    }
}
template <typename T>
__device__ __forceinline__ void mul_link_dag(cplx<T>* chi, const Link<T, 3>& u, const cplx<T>* h) {
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        chi[a].re = u.r[a] * h[0].re; chi[a].im = u.r[a] * h[0].im;
#pragma unroll
        for (int b = 1; b < 3; ++b) {
            chi[a].re = fma(u.r[b * 3 + a], h[b].re, chi[a].re);
            chi[a].im = fma(u.r[b * 3 + a], h[b].im, chi[a].im);
        }
    }
}

// ------------------------------------------------------------------ one term of the hopping sum
// acc += (1 + S gamma_MU) W psi, W = U (FWD, S = -1: the x+mu term) or U^dag (S = +1: the x-mu term),
// in the chiral basis of SURVEY.md §8(c) A2 (gamma5 = diag(1,1,-1,-1)).  (1 + S gamma_MU) has rank 2:
// project to the two upper spin components h0,h1, multiply by the link, rebuild the lower two:
//   mu=0: h0 = p0 - S p2,   h1 = p1 - S p3;    r2 = -S h0,   r3 = -S h1
//   mu=1: h0 = p0 - S i p3, h1 = p1 - S i p2;  r2 = S i h1,  r3 = S i h0
//   mu=2: h0 = p0 - S p3,   h1 = p1 + S p2;    r2 = S h1,    r3 = -S h0
//   mu=3: h0 = p0 - S i p2, h1 = p1 + S i p3;  r2 = S i h0,  r3 = -S i h1
// psi and acc are [spin][colour] flattened: component spin*N + colour.
// The two halves of a term: hop_project forms the half spinor (h0, h1) = upper two spin components of
// (1 + S gamma_MU) psi; hop_apply multiplies it by the link and adds the rebuilt four components to acc.
template <typename T, int N, int MU, bool FWD>
__device__ __forceinline__ void hop_project(cplx<T>* h0, cplx<T>* h1, const cplx<T>* p) {
#pragma unroll
    for (int c = 0; c < N; ++c) {
        const cplx<T> p0 = p[c], p1 = p[N + c], p2 = p[2 * N + c], p3 = p[3 * N + c];
        if (MU == 0) {
            h0[c] = FWD ? p0 + p2 : p0 - p2;
            h1[c] = FWD ? p1 + p3 : p1 - p3;
        } else if (MU == 1) {
            h0[c] = FWD ? p0 + timesI(p3) : p0 - timesI(p3);
            h1[c] = FWD ? p1 + timesI(p2) : p1 - timesI(p2);
        } else if (MU == 2) {
            h0[c] = FWD ? p0 + p3 : p0 - p3;
            h1[c] = FWD ? p1 - p2 : p1 + p2;
        } else {
            h0[c] = FWD ? p0 + timesI(p2) : p0 - timesI(p2);
            h1[c] = FWD ? p1 - timesI(p3) : p1 + timesI(p3);
        }
    }
}
// acc += the four spin components rebuilt from the link-multiplied half spinor (c0, c1)
template <typename T, int N, int MU, bool FWD>
__device__ __forceinline__ void hop_rebuild(cplx<T>* acc, const cplx<T>* c0, const cplx<T>* c1);
template <typename T, int N, int MU, bool FWD, typename LinkT>
__device__ __forceinline__ void hop_apply(cplx<T>* acc, const cplx<T>* h0, const cplx<T>* h1, const LinkT& u) {
    cplx<T> c0[N], c1[N];
    if (FWD) { mul_link(c0, u, h0); mul_link(c1, u, h1); }
    else     { mul_link_dag(c0, u, h0); mul_link_dag(c1, u, h1); }
    hop_rebuild<T, N, MU, FWD>(acc, c0, c1);
}
template <typename T, int N, int MU, bool FWD>
__device__ __forceinline__ void hop_rebuild(cplx<T>* acc, const cplx<T>* c0, const cplx<T>* c1) {
#pragma unroll
    for (int c = 0; c < N; ++c) {
        acc[c] = acc[c] + c0[c];
        acc[N + c] = acc[N + c] + c1[c];
        if (MU == 0) {
            acc[2 * N + c] = FWD ? acc[2 * N + c] + c0[c] : acc[2 * N + c] - c0[c];
            acc[3 * N + c] = FWD ? acc[3 * N + c] + c1[c] : acc[3 * N + c] - c1[c];
        } else if (MU == 1) {
            acc[2 * N + c] = FWD ? acc[2 * N + c] - timesI(c1[c]) : acc[2 * N + c] + timesI(c1[c]);
            acc[3 * N + c] = FWD ? acc[3 * N + c] - timesI(c0[c]) : acc[3 * N + c] + timesI(c0[c]);
        } else if (MU == 2) {
            acc[2 * N + c] = FWD ? acc[2 * N + c] - c1[c] : acc[2 * N + c] + c1[c];
            acc[3 * N + c] = FWD ? acc[3 * N + c] + c0[c] : acc[3 * N + c] - c0[c];
        } else {
            acc[2 * N + c] = FWD ? acc[2 * N + c] - timesI(c0[c]) : acc[2 * N + c] + timesI(c0[c]);
            acc[3 * N + c] = FWD ? acc[3 * N + c] + timesI(c1[c]) : acc[3 * N + c] - timesI(c1[c]);
        }
    }
}
template <typename T, int N, int MU, bool FWD, typename LinkT>
__device__ __forceinline__ void hop_term(cplx<T>* acc, const cplx<T>* p, const LinkT& u) {
    cplx<T> h0[N], h1[N];
    hop_project<T, N, MU, FWD>(h0, h1, p);
    hop_apply<T, N, MU, FWD>(acc, h0, h1, u);
}

// ------------------------------------------------------------------ hermitian 4x4 block times 4-vector
// blk: 16 reals = d0..d3, then lower entries (1,0) (2,0) (3,0) (2,1) (3,1) (3,2) as re,im.
template <typename T>
__device__ __forceinline__ void herm4_matvec(cplx<T>* y, const T* blk, const cplx<T>* x) {
    const cplx<T> l10 = mk<T>(blk[4], blk[5]), l20 = mk<T>(blk[6], blk[7]), l30 = mk<T>(blk[8], blk[9]);
    const cplx<T> l21 = mk<T>(blk[10], blk[11]), l31 = mk<T>(blk[12], blk[13]), l32 = mk<T>(blk[14], blk[15]);
    y[0] = blk[0] * x[0]; cmadc(y[0], l10, x[1]); cmadc(y[0], l20, x[2]); cmadc(y[0], l30, x[3]);
    y[1] = blk[1] * x[1]; cmad(y[1], l10, x[0]); cmadc(y[1], l21, x[2]); cmadc(y[1], l31, x[3]);
    y[2] = blk[2] * x[2]; cmad(y[2], l20, x[0]); cmad(y[2], l21, x[1]); cmadc(y[2], l32, x[3]);
    y[3] = blk[3] * x[3]; cmad(y[3], l30, x[0]); cmad(y[3], l31, x[1]); cmad(y[3], l32, x[2]);
}

// hermitian D x D block times D-vector, D = 2N (2 spins of one chirality x N colours): blk = D real diagonal entries, then the
// strictly-lower entries column by column ((1,0) (2,0) .. (D-1,0) (2,1) ..) as re,im — D*D reals.  Generic form of herm4_matvec.
template <typename T, int D>
__device__ __forceinline__ void herm_matvec(cplx<T>* y, const T* blk, const cplx<T>* x) {
#pragma unroll
    for (int i = 0; i < D; ++i) y[i] = blk[i] * x[i];
#pragma unroll
    for (int j = 0; j < D; ++j)
#pragma unroll
        for (int i = j + 1; i < D; ++i) {
            const int k = D + 2 * (j * (2 * D - j - 1) / 2 + (i - j - 1));
            const cplx<T> l = mk<T>(blk[k], blk[k + 1]);
            cmad(y[i], l, x[j]);     // row i, column j: L_ij x_j
            cmadc(y[j], l, x[i]);    // row j, column i: conj(L_ij) x_i
        }
}

// reals of the two blocks of one site: 2 (2N)^2
template <int N> struct CloverSize { static constexpr int reals = 2 * (2 * N) * (2 * N); };

// the block reals of one site from the clover field [par][row][chunk][h].  POLICY: streaming in the site-diagonal kernels; in the hop
// epilogues the blocks bypass L1 allocation (LD_NOALLOC), which the link and phi loads need more (E2 724 -> 717 us, H3c 620 -> 607 us
// at 48^4, while the plain clover apply loses 2.5 % with it)
template <typename T, int N = 2, int POLICY = LD_STREAM>
__device__ __forceinline__ void load_clover(T* blk, const void* field, const Geo& g, int par, int row, int h) {
    constexpr int CCH = CloverSize<N>::reals * sizeof(T) / 16;
    typedef typename Chunk<T>::type chunk_t;
    const chunk_t* p = reinterpret_cast<const chunk_t*>(field) + ((size_t)par * g.R + row) * (CCH * g.L3h) + h;
#pragma unroll
    for (int c = 0; c < CCH; ++c) {
        chunk_to_reals(ldg16<POLICY>(p + (size_t)c * g.L3h), blk + c * (16 / sizeof(T)));
    }
}

// y = B x for a spinor of 4N complex numbers: block 0 on components 0..2N-1 (chirality +), block 1 on the rest
template <typename T, int N = 2>
__device__ __forceinline__ void clover_matvec(cplx<T>* y, const T* blk, const cplx<T>* x) {
    if (N == 2) {
        herm4_matvec(y, blk, x);
        herm4_matvec(y + 4, blk + 16, x + 4);
    } else {
        herm_matvec<T, 2 * N>(y, blk, x);
        herm_matvec<T, 2 * N>(y + 2 * N, blk + 4 * N * N, x + 2 * N);
    }
}

// ------------------------------------------------------------------ host-side bookkeeping (hr_api.cu)
void set_error(const char* fmt, ...);
void count_launch(int n = 1);
int check_launch(const char* what);

// hr_hop.cu: run one hop (H1/H2/H3) with the kernel g->kernel selects; epi is an EPI_* of hr_hop_generic.cuh
struct HopArgs;
int run_hop(const hr_geom* g, const HopArgs& a, int epi, cudaStream_t st);
bool tiled_supported(const hr_geom* g);
bool tiled_chosen(const hr_geom* g);
int kernel_plan(const hr_geom* g, int both, int* info);
int sm_count();
// hr_hop_cg.cu: a parity hop with an axpy-type epilogue followed by a POST_* stage of the CG solver (hr_hop_generic.cuh);
// hop_post_blocks = the number of partial sums such a launch writes to HopArgs::partial
int run_hop_post(const hr_geom* g, const HopArgs& a, int epi, int post, cudaStream_t st);
int hop_post_blocks(const hr_geom* g);   // both: 0 parity hop, 1 paired-parity launch, 2 full D with phi == in

}  // namespace hr
