// hr_hop_generic.cuh — the generic hopping kernel: one thread per output site, any even extents >= 2.
// Steps H1/H2/H3 of DESIGN.md §2 (BASELINE.json north_star "Hopping kernel"; PAPER.md:31, 39
// "inner Dirac kernel").  Used for small or oddly-shaped lattices and as the fallback of the tiled kernel.
#pragma once

#include "hr_common.cuh"

namespace hr {

// epilogue of a hop (H2): what is written for output site x, with h = H in(x) the bare hopping sum
enum {
    EPI_NONE = 0,        // out = h
    EPI_AXPY = 1,        // out = a*phi(x) + c*h
    EPI_CLOVER_INV = 2,  // out = B(x) h                 (B = blocks of `clover`, e.g. A_oo^-1)
    EPI_CLOVER_AXPY = 3  // out = B(x) phi(x) + c*h      (B = A_ee)
};

// what happens to the epilogue's result w(x) (SURVEY.md §8(f) item 2 "fused dot products and axpys in the hop epilogue"):
//   POST_STORE     : out = w
//   POST_G5_NORM   : out = gamma5 w,  partial += |w|^2                                        (s = gamma5 Dhat p and <p, Dhat^dag Dhat p>)
//   POST_CG_UPDATE : r -= alpha gamma5 w,  partial += |r|^2   (w is not stored)                 (the CG update after the second Dhat;
//                    x += alpha p rides with p = r + beta p in cg_direction_kernel, which reads p anyway)
enum { POST_STORE = 0, POST_G5_NORM = 1, POST_CG_UPDATE = 2 };

struct HopArgs {
    const void* gauge;   // gauge field in the fermion representation, device layout
    const void* in;      // both == 0: half field of parity 1-parity; both == 1: full field
    void* out;           // both == 0: half field of parity `parity`;  both == 1: full field
    const void* phi;     // same shape as out (EPI_AXPY, EPI_CLOVER_AXPY)
    const void* clover;  // full-lattice block field (EPI_CLOVER_*)
    double a, c;
    int parity;          // output parity when both == 0
    int both;            // 1: full-lattice launch, both output parities (in / out / phi are full fields)
    // POST_* stages of the CG solver (hr_solver.cu), applied to the value the epilogue would have stored:
    double* partial = nullptr;        // one partial sum per CTA (fixed order inside the CTA)
    const double* cg_alpha = nullptr; // device scalar alpha (POST_CG_UPDATE)
    void* cg_r = nullptr;             // half field of the output parity (POST_CG_UPDATE): r -= alpha gamma5 w
    int slab_w1 = 0;     // > 0: the generic kernel walks the lattice in x1-slabs of this width (launch_hop_generic sets it)
    int open_mask = 0;   // bit mu set: direction mu is cut between ranks (hr_hop_local): the forward term of sites with
                         // x_mu = L_mu-1 and the backward term of sites with x_mu = 0 are left out here and added from
                         // the received faces by the boundary kernel (hr_halo.cu)
};

// PHI_POLICY: LD_STREAM when phi is read by this kernel only; LD_KEEP in the full-lattice launch (H3), where
// phi is the other parity pass's gather input
template <typename T, int N, int EPI, int PHI_POLICY = LD_STREAM, int POST = POST_STORE>
__device__ __forceinline__ void hop_epilogue(cplx<T>* acc, const Geo& g, const HopArgs& a, const void* phi_half,
                                             void* out_half, int p, int row, int h, double* part = nullptr, T alpha = (T)0,
                                             const cplx<T>* phi_pre = nullptr) {   // phi_pre: phi(x) already in registers (EPI_AXPY)
    constexpr int NC = 4 * N;
    typedef SiteIO<T, NC> IO;
    const size_t first = (size_t)row * (IO::NCH * g.L3h) + h;
    if (EPI == EPI_AXPY) {
        cplx<T> phi_ld[NC];
        if (!phi_pre) IO::template load<PHI_POLICY>(phi_ld, phi_half, first, g.L3h);
        const cplx<T>* phi = phi_pre ? phi_pre : phi_ld;
        const T ca = (T)a.a, cc = (T)a.c;
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            acc[k].re = fma(cc, acc[k].re, ca * phi[k].re);
            acc[k].im = fma(cc, acc[k].im, ca * phi[k].im);
        }
    } else if (EPI == EPI_CLOVER_INV) {
        T blk[CloverSize<N>::reals];
        cplx<T> y[NC];
        load_clover<T, N, LD_NOALLOC>(blk, a.clover, g, p, row, h);
        clover_matvec<T, N>(y, blk, acc);
#pragma unroll
        for (int k = 0; k < NC; ++k) acc[k] = y[k];
    } else if (EPI == EPI_CLOVER_AXPY) {
        T blk[CloverSize<N>::reals];
        cplx<T> phi[NC], y[NC];
        load_clover<T, N, LD_NOALLOC>(blk, a.clover, g, p, row, h);
        IO::template load<PHI_POLICY>(phi, phi_half, first, g.L3h);
        clover_matvec<T, N>(y, blk, phi);
        const T cc = (T)a.c;
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            acc[k].re = fma(cc, acc[k].re, y[k].re);
            acc[k].im = fma(cc, acc[k].im, y[k].im);
        }
    }
    if (POST == POST_STORE) {
        IO::store(out_half, first, g.L3h, acc);
    } else if (POST == POST_G5_NORM) {
        double n2 = 0.0;
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            n2 += (double)acc[k].re * (double)acc[k].re + (double)acc[k].im * (double)acc[k].im;
            if (k >= 2 * N) acc[k] = -acc[k];              // gamma5 = diag(1, 1, -1, -1) on the spin index
        }
        *part += n2;
        IO::store(out_half, first, g.L3h, acc);
    } else {
        cplx<T> v[NC];
        IO::template load<LD_STREAM>(v, a.cg_r, first, g.L3h);
        double n2 = 0.0;
#pragma unroll
        for (int k = 0; k < NC; ++k) {
            const T sa = k >= 2 * N ? alpha : -alpha;      // r -= alpha gamma5 w
            v[k].re = fma(sa, acc[k].re, v[k].re);
            v[k].im = fma(sa, acc[k].im, v[k].im);
            n2 += (double)v[k].re * (double)v[k].re + (double)v[k].im * (double)v[k].im;
        }
        *part += n2;
        IO::store(a.cg_r, first, g.L3h, v);
    }
}

// sum of `v` over the first `nthreads` threads of the CTA in a fixed order (warp tree, then warp sums in index order); valid in
// thread 0.  `red`: at least nthreads / 32 doubles of shared memory; `barrier_id`: a named barrier all nthreads threads reach.
__device__ __forceinline__ double cta_sum_fixed(double v, double* red, int nthreads, int barrier_id) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    asm volatile("bar.sync %0, %1;" ::"r"(barrier_id), "r"(nthreads) : "memory");     // everybody is done with the memory `red` aliases
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    asm volatile("bar.sync %0, %1;" ::"r"(barrier_id), "r"(nthreads) : "memory");
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int i = 0; i < nthreads / 32; ++i) t += red[i];
    return t;
}

// resident CTAs per SM the kernel is compiled for: the fp64 kernels with three colours need 130-138 registers left alone (3 CTAs of
// 4 warps per SM: 18 % of the warp slots, DRAM 58-68 % busy); held to 128 registers (4 CTAs, a few bytes of spills) the SU(3) hop at
// 48^4 goes from 729 to 634 us.  5 CTAs (102 registers) spill heavily and lose 25 %; the other instantiations gain nothing.
template <typename T, int N> constexpr int generic_min_ctas() { return (N == 3 && sizeof(T) == 8) ? 4 : 1; }
// C3: the links are complex 3 x 3 matrices stored in full (HR_REP_SU3; N = 3)
template <typename T, int N, int EPI, bool ONFLY, bool C3 = false, bool BOTH = false, int POST = POST_STORE>
__global__ void __launch_bounds__(128, generic_min_ctas<T, N>()) hop_generic_kernel(Geo g, HopArgs a) {
    static_assert(!C3 || N == 3, "complex 3 x 3 links: N = 3 (ONFLY then means: two rows stored, third rebuilt)");
    typedef typename std::conditional<C3, LinkC3<T>, Link<T, N>>::type link_t;
    constexpr int NC = 4 * N;
    typedef SiteIO<T, NC> IO;
    // full-lattice launch: the output parity is the fastest-varying part of blockIdx.x, so the two CTAs that use a link
    // (forward term of parity p, backward term of parity 1-p at the neighbouring sites) run next to each other and the second
    // use hits L2 — links and phi are then loaded at normal priority (BOTH), else streamed
    const int bid = BOTH ? (int)(blockIdx.x >> 1) : (int)blockIdx.x;
    int cb = bid * blockDim.x + threadIdx.x;
    const bool valid = cb < g.Vh;
    if (!valid) {
        if (POST == POST_STORE) return;
        cb = g.Vh - 1;        // a reduction follows: stay, shadow the last site, store and add nothing
    }
    const int p = BOTH ? (int)(blockIdx.x & 1) : a.parity;
    constexpr int LINKPOL = BOTH ? LD_KEEP : LD_STREAM;
    const size_t half_bytes = (size_t)g.Vh * IO::NCH * 16;
    const char* in_half = reinterpret_cast<const char*>(a.in) + (BOTH ? (size_t)(1 - p) * half_bytes : 0);
    char* out_half = reinterpret_cast<char*>(a.out) + (BOTH ? (size_t)p * half_bytes : 0);
    const char* phi_half = a.phi ? reinterpret_cast<const char*>(a.phi) + (BOTH ? (size_t)p * half_bytes : 0) : nullptr;

    // Site order.  Default: checkerboard index = (row, h) with row = (x0 L1 + x1) L2 + x2.  With slabs (full-lattice launches on
    // lattices whose x0-plane does not stay in L2 between its uses as x0-1, x0 and x0+1 neighbour): slab of x1 first, then x0, then
    // the rows of the slab — the reuse distance along x0 shrinks from a plane to a slab of it.
    int row, h;
    if (a.slab_w1 > 0) {
        const int slab_rows = a.slab_w1 * g.s1, slab_plane = slab_rows * g.L3h, per_slab = g.L0 * slab_plane;
        const int sl = cb / per_slab, r0 = cb - sl * per_slab;
        const int xx0 = r0 / slab_plane, r1 = r0 - xx0 * slab_plane;
        const int lrow = r1 / g.L3h;
        h = r1 - lrow * g.L3h;
        row = xx0 * g.s0 + sl * slab_rows + lrow;
    } else {
        row = cb / g.L3h;
        h = cb - row * g.L3h;
    }
    const int x0 = row / g.s0, rem = row - x0 * g.s0;
    const int x1 = rem / g.s1, x2 = rem - x1 * g.s1;
    const int r = (x0 + x1 + x2 + p) & 1;  // x3 = 2h + r

    // neighbour rows (periodic) and pair indices in the opposite-parity arrays
    const int row_f0 = row + (x0 == g.L0 - 1 ? -(g.L0 - 1) * g.s0 : g.s0);
    const int row_b0 = row + (x0 == 0 ? (g.L0 - 1) * g.s0 : -g.s0);
    const int row_f1 = row + (x1 == g.L1 - 1 ? -(g.L1 - 1) * g.s1 : g.s1);
    const int row_b1 = row + (x1 == 0 ? (g.L1 - 1) * g.s1 : -g.s1);
    const int row_f2 = row + (x2 == g.L2 - 1 ? -(g.L2 - 1) : 1);
    const int row_b2 = row + (x2 == 0 ? (g.L2 - 1) : -1);
    const int h_f3 = r ? (h == g.L3h - 1 ? 0 : h + 1) : h;
    const int h_b3 = r ? h : (h == 0 ? g.L3h - 1 : h - 1);

    cplx<T> acc[NC];
#pragma unroll
    for (int k = 0; k < NC; ++k) acc[k] = mk<T>((T)0, (T)0);

    const int stride = g.L3h;
    const int rowlen = IO::NCH * g.L3h;
    const int om = a.open_mask;   // terms that cross a rank boundary are the boundary kernel's (0 on one GPU)
#define HR_HOP_DIR(MU, ROWF, HF, ROWB, HB, ATHI, ATLO)                                          \
    {                                                                                           \
        cplx<T> nb[NC];                                                                         \
        link_t u;                                                                               \
        if (!(((om >> MU) & 1) && (ATHI))) {                                                    \
            load_link_rep<T, LINKPOL, ONFLY>(u, a.gauge, g, p, MU, row, h);                     \
            IO::template load<LD_KEEP>(nb, in_half, (size_t)(ROWF) * rowlen + (HF), stride);    \
            hop_term<T, N, MU, true>(acc, nb, u);                                               \
        }                                                                                       \
        if (!(((om >> MU) & 1) && (ATLO))) {                                                    \
            load_link_rep<T, LINKPOL, ONFLY>(u, a.gauge, g, 1 - p, MU, ROWB, HB);               \
            IO::template load<LD_KEEP>(nb, in_half, (size_t)(ROWB) * rowlen + (HB), stride);    \
            hop_term<T, N, MU, false>(acc, nb, u);                                              \
        }                                                                                       \
    }
    HR_HOP_DIR(0, row_f0, h, row_b0, h, x0 == g.L0 - 1, x0 == 0)
    HR_HOP_DIR(1, row_f1, h, row_b1, h, x1 == g.L1 - 1, x1 == 0)
    HR_HOP_DIR(2, row_f2, h, row_b2, h, x2 == g.L2 - 1, x2 == 0)
    HR_HOP_DIR(3, row, h_f3, row, h_b3, r == 1 && h == g.L3h - 1, r == 0 && h == 0)
#undef HR_HOP_DIR

    if (POST == POST_STORE) {
        hop_epilogue<T, N, EPI, (BOTH ? LD_KEEP : LD_STREAM)>(acc, g, a, phi_half, out_half, p, row, h);
    } else {
        __shared__ double red[4];
        double part = 0.0;
        if (valid) hop_epilogue<T, N, EPI, LD_STREAM, POST>(acc, g, a, phi_half, out_half, p, row, h, &part, POST == POST_CG_UPDATE ? (T)*a.cg_alpha : (T)0);
        const double tot = cta_sum_fixed(part, red, 128, 1);
        if (threadIdx.x == 0) a.partial[blockIdx.x] = tot;
    }
}

// x1-slab width for the generic kernel's site order (0 = plain order): full-lattice launches whose two live x0-planes (both
// parities, spinors + links + output) exceed what L2 keeps; the widest divisor of L1 whose slab fits (profiles/r02_adjoint.md)
inline int generic_slab_w1(const Geo& g, bool both, size_t site_bytes) {
    if (!both) return 0;
    const int L1 = g.s0 / g.s1;
    const double plane = 2.0 * 2.0 * (double)g.s0 * g.L3h * site_bytes;      // two planes, two parities
    if (plane <= 64e6) return 0;          // half of L2: the plain order already gets the x0 neighbours from L2
    int best = 1;                          // 48^4 adjoint fp64: widths 8-12 are best (915 -> 815 us), 16+ lose again
    for (int w = 1; w < L1; ++w)
        if (L1 % w == 0 && plane * w / L1 <= 40e6) best = w;
    return best;
}

template <typename T, int N, bool ONFLY, bool C3, bool BOTH>
inline int launch_hop_generic_both(const Geo& g, const HopArgs& a_in, int epi, cudaStream_t st) {
    HopArgs a = a_in;
    a.slab_w1 = generic_slab_w1(g, BOTH, (size_t)(16 * N + 4 * (C3 ? (ONFLY ? 12 : 18) : ONFLY ? 4 : N == 2 ? 4 : 9)) * sizeof(T));
    dim3 block(128), grid(((g.Vh + 127) / 128) * (BOTH ? 2 : 1));
    switch (epi) {
        case EPI_NONE: hop_generic_kernel<T, N, EPI_NONE, ONFLY, C3, BOTH><<<grid, block, 0, st>>>(g, a); break;
        case EPI_AXPY: hop_generic_kernel<T, N, EPI_AXPY, ONFLY, C3, BOTH><<<grid, block, 0, st>>>(g, a); break;
        case EPI_CLOVER_INV: hop_generic_kernel<T, N, EPI_CLOVER_INV, ONFLY, C3, BOTH><<<grid, block, 0, st>>>(g, a); break;
        case EPI_CLOVER_AXPY: hop_generic_kernel<T, N, EPI_CLOVER_AXPY, ONFLY, C3, BOTH><<<grid, block, 0, st>>>(g, a); break;
        default: set_error("unknown epilogue %d", epi); return HR_EINVAL;
    }
    count_launch();
    return check_launch("hop_generic_kernel");
}

// the CG stages: parity hop with an axpy-type epilogue and a POST stage; blocks = the number of partial sums written
template <typename T, int N, bool ONFLY, bool C3>
inline int launch_hop_generic_post(const Geo& g, const HopArgs& a, int epi, int post, cudaStream_t st) {
    dim3 block(128), grid((g.Vh + 127) / 128);
    if (epi == EPI_AXPY && post == POST_G5_NORM) hop_generic_kernel<T, N, EPI_AXPY, ONFLY, C3, false, POST_G5_NORM><<<grid, block, 0, st>>>(g, a);
    else if (epi == EPI_AXPY && post == POST_CG_UPDATE) hop_generic_kernel<T, N, EPI_AXPY, ONFLY, C3, false, POST_CG_UPDATE><<<grid, block, 0, st>>>(g, a);
    else if (epi == EPI_CLOVER_AXPY && post == POST_G5_NORM) hop_generic_kernel<T, N, EPI_CLOVER_AXPY, ONFLY, C3, false, POST_G5_NORM><<<grid, block, 0, st>>>(g, a);
    else if (epi == EPI_CLOVER_AXPY && post == POST_CG_UPDATE) hop_generic_kernel<T, N, EPI_CLOVER_AXPY, ONFLY, C3, false, POST_CG_UPDATE><<<grid, block, 0, st>>>(g, a);
    else { set_error("hop with a CG stage: epilogue %d / stage %d", epi, post); return HR_EINVAL; }
    count_launch();
    return check_launch("hop_generic_kernel");
}

template <typename T, int N, bool ONFLY = false, bool C3 = false>
inline int launch_hop_generic(const Geo& g, const HopArgs& a, int epi, cudaStream_t st) {
    if (a.both) return launch_hop_generic_both<T, N, ONFLY, C3, true>(g, a, epi, st);
    return launch_hop_generic_both<T, N, ONFLY, C3, false>(g, a, epi, st);
}

}  // namespace hr
