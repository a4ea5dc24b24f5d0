// hr_hop_tiled.cuh — the x0-marching tiled hopping kernel (steps H1/H2/H3 of DESIGN.md §2, design in §5.2).
//
// One CTA owns a T1 x T2 tile of x3-rows in the (x1,x2) plane and marches along x0 through a segment of
// planes.  A producer thread moves whole x3-rows of the input half field (contiguous runs of the device
// layout) into shared memory with 1-D bulk asynchronous copies (cp.async.bulk, completion on
// an mbarrier): the tile rows of plane x0+1 into a 4-slot ring (each plane serves three steps: as x0+1, x0
// and x0-1 neighbour) and the one-row halo of the centre plane in x1 and x2 into a double buffer.
// Consumer threads (one per output site of the tile) gather the 8 neighbour spinors from shared memory;
// links are read straight from global memory (each is used once per kernel) and re-loaded into the same
// registers right after their use, for the next step, so a link load has a whole step to complete.
// Bytes in flight are therefore bounded by shared memory, not by registers (the generic kernel's limit:
// profiles/r01_generic_hop.md), and an input row crosses L2->SM (1 + 2/T1 + 2/T2) times instead of ~5.4.
#pragma once

#include <atomic>

#include "hr_hop_generic.cuh"

namespace hr {

constexpr bool HOP_ALINK = true;      // link slots in shared memory where an instantiation has them (launch_hop_tiled_l3h)
constexpr int TILED_RING = 4;         // ring slots: planes x0-1, x0, x0+1 live + one being filled
constexpr int TILED_HALO = 2;         // halo buffers: one in use, one being filled (a third one costs the L1 the link loads need)

// Per-precision choices, each made by measurement at 48^4 (profiles/r01_tiled_variants.md):
//   PIN     : __syncwarp() after each link re-load, which stops ptxas from sinking the loads to the end of the step
//   NBDB    : read the neighbour of term t+1 from shared memory before computing term t (two register images)
//   LINKPOL : cache policy of the link loads (LD_STREAM = ld.global.cs, LD_KEEP = ld.global.nc)
template <typename T> struct TiledTuning;
template <> struct TiledTuning<double> { static constexpr bool PIN = false, NBDB = false; static constexpr int LINKPOL = LD_KEEP; };
template <> struct TiledTuning<float> { static constexpr bool PIN = true, NBDB = true; static constexpr int LINKPOL = LD_STREAM; };
// consumer threads the kernel is compiled for (one per output site of a T1 x T2 tile of rows): 192 for the small tiles
// (2 x 4 rows of L3h <= 24 sites, 2 x 2 rows of L3h <= 48), 384 for 4 x 4 rows
constexpr int tiled_max_consumers(int t1, int t2) { return t1 * t2 <= 8 ? 192 : 384; }

// ------------------------------------------------------------------ mbarrier / bulk-copy primitives (PTX)
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "HR_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra HR_DONE_%=;\n"
        "bra HR_WAIT_%=;\n"
        "HR_DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity)
        : "memory");
}
// global -> shared bulk copy of `bytes` (multiple of 16, both addresses 16-byte aligned); completes on `bar`
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

// NC complex numbers of one site from a shared-memory row image (chunk c at byte offset c*L3h*16 from `p`)
template <typename T, int NC>
__device__ __forceinline__ void lds_site(cplx<T>* s, const char* p, int chunk_stride_bytes);
template <>
__device__ __forceinline__ void lds_site<double, 8>(cplx<double>* s, const char* p, int cs) {
#pragma unroll
    for (int c = 0; c < 8; ++c) {
        const double2 v = *reinterpret_cast<const double2*>(p + c * cs);
        s[c] = mk<double>(v.x, v.y);
    }
}
template <>
__device__ __forceinline__ void lds_site<double, 12>(cplx<double>* s, const char* p, int cs) {
#pragma unroll
    for (int c = 0; c < 12; ++c) {
        const double2 v = *reinterpret_cast<const double2*>(p + c * cs);
        s[c] = mk<double>(v.x, v.y);
    }
}
template <>
__device__ __forceinline__ void lds_site<float, 8>(cplx<float>* s, const char* p, int cs) {
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const float4 v = *reinterpret_cast<const float4*>(p + c * cs);
        s[2 * c] = mk<float>(v.x, v.y);
        s[2 * c + 1] = mk<float>(v.z, v.w);
    }
}
template <>
__device__ __forceinline__ void lds_site<float, 12>(cplx<float>* s, const char* p, int cs) {
#pragma unroll
    for (int c = 0; c < 6; ++c) {
        const float4 v = *reinterpret_cast<const float4*>(p + c * cs);
        s[2 * c] = mk<float>(v.x, v.y);
        s[2 * c + 1] = mk<float>(v.z, v.w);
    }
}

// OPEN kernels: a term that crosses a cut is left out by multiplying its link by zero — branch-free, so that the instruction
// schedule stays that of the periodic kernel (skipping the term with a branch cost 14 % of the interior kernel: 247 against 216 us)
template <bool OPEN, typename T>
__device__ __forceinline__ Link<T, 2> open_link(const Link<T, 2>& u, bool cut) {
    if (!OPEN) return u;
    const T m = cut ? (T)0 : (T)1;
    Link<T, 2> v;
    v.a = mk<T>(u.a.re * m, u.a.im * m);
    v.b = mk<T>(u.b.re * m, u.b.im * m);
    return v;
}
template <bool OPEN, typename T>
__device__ __forceinline__ Link<T, 3> open_link(const Link<T, 3>& u, bool cut) {
    if (!OPEN) return u;
    const T m = cut ? (T)0 : (T)1;
    Link<T, 3> v;
#pragma unroll
    for (int k = 0; k < 9; ++k) v.r[k] = u.r[k] * m;
    return v;
}

// Links through shared memory.  A load into registers that is requested one step ahead does not get a step of lead: ptxas puts
// every global load of the loop on ONE scoreboard, so the first use of a link at the top of a step waits for ALL outstanding link
// loads, the ones requested a few hundred instructions earlier included, and a DRAM latency is exposed in every step (18-24 % of the
// stall samples, profiles/r02_kernels.md).  cp.async groups complete in order and cp.async.wait_group N waits for all but the N
// newest: each link has its own slot (32 bytes fp64, 16 bytes fp32), is re-requested into it right after its use, and is waited
// for with N = 6 — exactly the seven-requests-ago one.  A thread reads only slots it filled itself, so no barrier is needed.
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NPENDING> __device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;" ::"n"(NPENDING) : "memory");
}

// (alpha, beta) of a compressed link from its slot; volatile keeps the reads behind the wait_group
__device__ __forceinline__ void lds_link(cplx<double>* ab, uint32_t slot, int chunk_stride) {
    asm volatile("ld.volatile.shared.v2.f64 {%0, %1}, [%2];" : "=d"(ab[0].re), "=d"(ab[0].im) : "r"(slot));
    asm volatile("ld.volatile.shared.v2.f64 {%0, %1}, [%2];" : "=d"(ab[1].re), "=d"(ab[1].im) : "r"(slot + chunk_stride));
}
__device__ __forceinline__ void lds_link(cplx<float>* ab, uint32_t slot, int) {
    asm volatile("ld.volatile.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(ab[0].re), "=f"(ab[0].im), "=f"(ab[1].re), "=f"(ab[1].im) : "r"(slot));
}

// launch geometry chosen on the host (hr_hop.cu)
struct TiledPlan {
    int t1, t2;        // tile shape in rows (x1, x2): selects the kernel instantiation
    int nt1, nt2;      // tiles along x1, x2
    int nseg, seglen;  // x0 segments per tile and their length (nseg*seglen == L0)
    int nconsumer;     // consumer threads (multiple of 32, >= T1*T2*L3h)
    int rowb;          // bytes of one x3-row of the input half field
    size_t smem;       // dynamic shared memory
};

// ------------------------------------------------------------------ the kernel
// grid.x = (both ? 2 : 1) * nt1 * nt2 * nseg; with both == 1 the output parity is the fastest-varying part
// of blockIdx.x, so the two CTAs that use a link (forward term of parity p, backward term of parity 1-p)
// run next to each other and the second use hits L2.
// Shared memory: [16 mbarriers][ring: TILED_RING planes of T1*T2 rows][halo: TILED_HALO buffers of 2*T2 + 2*T1 rows]
//   halo buffer rows: [x1-1 line: T2 rows][x1+T1 line: T2 rows][x2-1 rows: T1][x2+T2 rows: T1]
// SHARE = false: one output parity per launch.
// SHARE = true : full-lattice launch, the two parities as neighbouring CTAs; links and phi are also read by the CTA of
//         the other parity, so they are loaded with normal L2 priority.  (The plain full operator D with phi == in has
//         its own kernel, hr_dirac_tiled.cuh; this path serves the clover-improved one and the adjoint representation.)
// L3H: compile-time L3/2 (0 = read it from the geometry): the strides between the 16-byte chunks of a site are then
// immediates in every LDS / LDG / STG (about a quarter fewer instructions per site)
// OPEN: the hop of one rank of a decomposed lattice (hr_hop_local): for the directions in HopArgs::open_mask the forward term of
// sites with x_mu = L_mu-1 and the backward term of sites with x_mu = 0 are left out (the boundary kernel of hr_halo.cu adds them
// from the received faces); the producer still copies the wrapped-around rows, they are simply not used.
// POST: a stage of the CG solver applied to the epilogue's result (hr_hop_generic.cuh: POST_*); the CTA then writes one partial sum
// ALINK: the eight links of a site travel through cp.async slots in shared memory instead of registers (see cp_async16 above;
// fundamental representation, one output parity)
template <typename T, int N, int EPI, int T1, int T2, bool SHARE, bool ONFLY, int L3H, bool OPEN = false, int POST = POST_STORE, bool ALINK = false>
__global__ void __launch_bounds__(tiled_max_consumers(T1, T2) + 32, (!SHARE && sizeof(T) == 4 && N == 2 && T1 * T2 <= 8) ? 2 : 1)
    hop_tiled_kernel(Geo g_in, HopArgs a, TiledPlan pl) {
    Geo g = g_in;
    if (L3H > 0) g.L3h = L3H;
    constexpr int NC = 4 * N;
    typedef SiteIO<T, NC> IO;
    constexpr int TR = T1 * T2;            // tile rows
    constexpr int HR = 2 * T2 + 2 * T1;    // halo rows
    constexpr int LP = SHARE ? LD_KEEP : TiledTuning<T>::LINKPOL;
    constexpr bool PIN = TiledTuning<T>::PIN, NBDB = TiledTuning<T>::NBDB;
    extern __shared__ __align__(128) char smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);
    char* ring = smem + 128;
    const int rowb = L3H > 0 ? SiteIO<T, 4 * N>::NCH * L3H * 16 : pl.rowb;
    const int planeb = TR * rowb;
    const int halob = HR * rowb;
    char* halo = ring + TILED_RING * planeb;
    char* lbuf = halo + TILED_HALO * halob;          // ALINK: link slots [link][chunk][consumer thread]
    static_assert(!ALINK || (N == 2 && !ONFLY && !SHARE), "link slots: compressed fundamental links, one output parity");
    const uint32_t bar_full = smem_u32(bars);            // [TILED_RING]
    const uint32_t bar_empty = smem_u32(bars + 4);       // [TILED_RING]
    const uint32_t bar_hempty = smem_u32(bars + 8);      // [TILED_HALO]

    const int tid = threadIdx.x;
    const int ncw = pl.nconsumer >> 5;  // consumer warps
    if (tid == 0) {
        for (int i = 0; i < TILED_RING; ++i) {
            mbar_init(bar_full + 8 * i, 1);
            mbar_init(bar_empty + 8 * i, ncw);
        }
        for (int i = 0; i < TILED_HALO; ++i) mbar_init(bar_hempty + 8 * i, ncw);
        mbar_fence_init();
    }
    __syncthreads();

    // ---- which work: parity, tile, x0 segment
    int bid = blockIdx.x;
    int p = a.parity;
    if (a.both) { p = bid & 1; bid >>= 1; }
    const int seg = bid / (pl.nt1 * pl.nt2);
    const int tile = bid - seg * (pl.nt1 * pl.nt2);
    const int t1 = tile / pl.nt2, t2 = tile - t1 * pl.nt2;
    const int xs = seg * pl.seglen, nsteps = pl.seglen;
    const int L0 = g.L0, L1 = g.s0 / g.s1, L2 = g.s1;

    const size_t half_bytes = (size_t)g.Vh * IO::NCH * 16;
    const char* in_half = reinterpret_cast<const char*>(a.in) + (a.both ? (size_t)(1 - p) * half_bytes : 0);
    char* out_half = reinterpret_cast<char*>(a.out) + (a.both ? (size_t)p * half_bytes : 0);
    const char* phi_half = a.phi ? reinterpret_cast<const char*>(a.phi) + (a.both ? (size_t)p * half_bytes : 0) : nullptr;

    if (tid >= pl.nconsumer) {
        // ================================================================ producer (one thread)
        if (tid != pl.nconsumer) return;
        const int x1base = t1 * T1, x2base = t2 * T2;
        const int x1lo = (x1base - 1 + L1) % L1, x1hi = (x1base + T1) % L1;
        const int x2lo = (x2base - 1 + L2) % L2, x2hi = (x2base + T2) % L2;
        for (int j = 0; j < nsteps + 2; ++j) {   // iteration j: plane x0 = xs-1+j into ring slot j%4, with its halo if it will be a centre
            const int slot = j & (TILED_RING - 1);
            const uint32_t use = (uint32_t)(j / TILED_RING);
            mbar_wait(bar_empty + 8 * slot, (use & 1) ^ 1);
            const int hc = j - (3 - TILED_HALO);              // centre plane whose halo rides with this iteration
            const bool with_halo = (hc >= 1 && hc <= nsteps);   // plane hc is the centre of step hc-1
            const int hb = hc % TILED_HALO;
            if (with_halo) mbar_wait(bar_hempty + 8 * hb, ((uint32_t)((hc - 1) / TILED_HALO) & 1) ^ 1);
            const uint32_t full = bar_full + 8 * slot;
            mbar_expect_tx(full, (uint32_t)(planeb + (with_halo ? halob : 0)));
            const int x0p = (xs - 1 + j + L0) % L0;
            const uint32_t dst = smem_u32(ring + slot * planeb);
#pragma unroll
            for (int aa = 0; aa < T1; ++aa) {
                const size_t row = ((size_t)x0p * L1 + x1base + aa) * L2 + x2base;
                bulk_g2s(dst + aa * T2 * rowb, in_half + row * rowb, (uint32_t)(T2 * rowb), full);
            }
            if (with_halo) {
                const int x0h = (xs - 1 + hc + L0) % L0;
                const uint32_t hd = smem_u32(halo + hb * halob);
                bulk_g2s(hd, in_half + (((size_t)x0h * L1 + x1lo) * L2 + x2base) * rowb, (uint32_t)(T2 * rowb), full);
                bulk_g2s(hd + T2 * rowb, in_half + (((size_t)x0h * L1 + x1hi) * L2 + x2base) * rowb, (uint32_t)(T2 * rowb), full);
#pragma unroll
                for (int aa = 0; aa < T1; ++aa) {
                    const size_t rb = ((size_t)x0h * L1 + x1base + aa) * L2;
                    bulk_g2s(hd + (2 * T2 + aa) * rowb, in_half + (rb + x2lo) * rowb, (uint32_t)rowb, full);
                    bulk_g2s(hd + (2 * T2 + T1 + aa) * rowb, in_half + (rb + x2hi) * rowb, (uint32_t)rowb, full);
                }
            }
        }
        return;
    }

    // ================================================================ consumers: one thread per output site
    const int L3h = g.L3h;
    const bool active = tid < TR * L3h;
    const int ctid = active ? tid : 0;               // idle threads shadow site 0 (no global access)
    const int lr = ctid / L3h, h = ctid - lr * L3h;   // local row in the tile, pair index
    const int la = lr / T2, lb = lr - la * T2;
    const int x1 = t1 * T1 + la, x2 = t2 * T2 + lb;
    const int cs = L3h * 16;                          // byte stride between chunks of a site in a row image
    // shared-memory byte offsets of the neighbour rows, relative to the centre ring slot (in-tile) or the
    // halo buffer; constant over the march
    const bool f1_in = la + 1 < T1, b1_in = la > 0, f2_in = lb + 1 < T2, b2_in = lb > 0;
    const int off_f1 = (f1_in ? (lr + T2) : (T2 + lb)) * rowb;
    const int off_b1 = (b1_in ? (lr - T2) : lb) * rowb;
    const int off_f2 = (f2_in ? (lr + 1) : (2 * T2 + T1 + la)) * rowb;
    const int off_b2 = (b2_in ? (lr - 1) : (2 * T2 + la)) * rowb;
    const int off_c = lr * rowb;
    // global rows: own row at plane x0 is row0 + x0*s0; backward-link rows in x1, x2 likewise
    const int row0 = x1 * g.s1 + x2;
    const int rowb1_0 = ((x1 == 0 ? L1 - 1 : x1 - 1)) * g.s1 + x2;
    const int rowb2_0 = x1 * g.s1 + (x2 == 0 ? L2 - 1 : x2 - 1);

    const int om = OPEN ? a.open_mask : 0;
    const bool cut_f1 = ((om >> 1) & 1) && x1 == L1 - 1, cut_b1 = ((om >> 1) & 1) && x1 == 0;
    const bool cut_f2 = ((om >> 2) & 1) && x2 == L2 - 1, cut_b2 = ((om >> 2) & 1) && x2 == 0;

    Link<T, N> uf[ALINK ? 1 : 4], ub[ALINK ? 1 : 4];
    // ALINK: slot j of this thread holds link j of the CURRENT step, j = 0..7 in the order of use (U_0(x), U_0(x-0), U_1(x), ...);
    // it is re-requested for the next step right after its use and waited for with cp.async.wait_group 7
    constexpr int LCH = SiteIO<T, 2>::NCH;
    const uint32_t lslot = smem_u32(lbuf) + (uint32_t)tid * 16;
    const int lchb = pl.nconsumer * 16;
    auto link_request = [&](int j, int par, int mu, int row, int hh) {
        const char* src = reinterpret_cast<const char*>(a.gauge) + (((size_t)(par * 4 + mu) * g.R + row) * (LCH * L3h) + hh) * 16;
#pragma unroll
        for (int c = 0; c < LCH; ++c) cp_async16(lslot + (j * LCH + c) * lchb, src + (size_t)c * cs);
        cp_async_commit();
    };
    auto link_get = [&](Link<T, 2>& u, int j) {
        cp_async_wait<7>();
        cplx<T> ab[2];
        lds_link(ab, lslot + j * LCH * lchb, lchb);
        u.a = ab[0];
        u.b = ab[1];
    };
    {   // links of the first step
        const int row = row0 + xs * g.s0;
        const int r = (xs + x1 + x2 + p) & 1;
        if constexpr (ALINK) {
            link_request(0, p, 0, row, h);
            link_request(1, 1 - p, 0, row0 + (xs == 0 ? L0 - 1 : xs - 1) * g.s0, h);
            link_request(2, p, 1, row, h);
            link_request(3, 1 - p, 1, rowb1_0 + xs * g.s0, h);
            link_request(4, p, 2, row, h);
            link_request(5, 1 - p, 2, rowb2_0 + xs * g.s0, h);
            link_request(6, p, 3, row, h);
            link_request(7, 1 - p, 3, row, r ? h : (h == 0 ? L3h - 1 : h - 1));
        } else {
        load_link_rep<T, LP, ONFLY>(uf[0], a.gauge, g, p, 0, row, h);
        load_link_rep<T, LP, ONFLY>(ub[0], a.gauge, g, 1 - p, 0, row0 + (xs == 0 ? L0 - 1 : xs - 1) * g.s0, h);
        load_link_rep<T, LP, ONFLY>(uf[1], a.gauge, g, p, 1, row, h);
        load_link_rep<T, LP, ONFLY>(ub[1], a.gauge, g, 1 - p, 1, rowb1_0 + xs * g.s0, h);
        load_link_rep<T, LP, ONFLY>(uf[2], a.gauge, g, p, 2, row, h);
        load_link_rep<T, LP, ONFLY>(ub[2], a.gauge, g, 1 - p, 2, rowb2_0 + xs * g.s0, h);
        load_link_rep<T, LP, ONFLY>(uf[3], a.gauge, g, p, 3, row, h);
        load_link_rep<T, LP, ONFLY>(ub[3], a.gauge, g, 1 - p, 3, row, r ? h : (h == 0 ? L3h - 1 : h - 1));
        }
    }

    double cg_part = 0.0;                                                           // POST stages: this thread's share of the CTA's partial sum
    const T cg_alpha = POST == POST_CG_UPDATE ? (T)*a.cg_alpha : (T)0;
    for (int k = 0; k < nsteps; ++k) {
        const int x0 = xs + k;
        const int r = (x0 + x1 + x2 + p) & 1;
        const int hf3 = r ? (h == L3h - 1 ? 0 : h + 1) : h;
        const int hb3 = r ? h : (h == 0 ? L3h - 1 : h - 1);
        const bool cut_f0 = (om & 1) && x0 == L0 - 1, cut_b0 = (om & 1) && x0 == 0;
        const bool cut_f3 = ((om >> 3) & 1) && r == 1 && h == L3h - 1, cut_b3 = ((om >> 3) & 1) && r == 0 && h == 0;
        const char* sprev = ring + (k & 3) * planeb;
        const char* scur = ring + ((k + 1) & 3) * planeb;
        const char* snext = ring + ((k + 2) & 3) * planeb;
        const int hb = (k + 1) % TILED_HALO;
        const char* shalo = halo + hb * halob;
        if (k == 0) {
            mbar_wait(bar_full, 0);
            mbar_wait(bar_full + 8, 0);
        }
        mbar_wait(bar_full + 8 * ((k + 2) & 3), ((uint32_t)(k + 2) >> 2) & 1);

        // next step's plane (clamped on the last step: the reload is then harmless and unused)
        const int xn = (k + 1 < nsteps) ? x0 + 1 : x0;
        const int rown = row0 + xn * g.s0;
        const int rn = (xn + x1 + x2 + p) & 1;
        const int hb3n = rn ? h : (h == 0 ? L3h - 1 : h - 1);

        // Eight terms.  The neighbour of term t+1 is read from shared memory before term t is computed
        // (two register images, nbA / nbB), and each link is re-loaded for the next step right after its
        // use; __syncwarp() keeps the compiler from sinking those loads to the end of the step (where
        // their latency would be exposed at the top of the next one).
        cplx<T> acc[NC], nbA[NC], nbB[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) acc[c] = mk<T>((T)0, (T)0);

#define HR_NB_NEXT(BUF, ADDR) if (NBDB) lds_site<T, NC>(BUF, ADDR, cs)
#define HR_NB_NOW(BUF, ADDR) if (!NBDB) lds_site<T, NC>(BUF, ADDR, cs)
#define HR_PIN() if (PIN) __syncwarp()
        cplx<T>* const nb0 = nbA;
        cplx<T>* const nb1 = NBDB ? nbB : nbA;
        const char* const a0f = snext + off_c + h * 16;
        const char* const a0b = sprev + off_c + h * 16;
        const char* const a1f = (f1_in ? scur : shalo) + off_f1 + h * 16;
        const char* const a1b = (b1_in ? scur : shalo) + off_b1 + h * 16;
        const char* const a2f = (f2_in ? scur : shalo) + off_f2 + h * 16;
        const char* const a2b = (b2_in ? scur : shalo) + off_b2 + h * 16;
        const char* const a3f = scur + off_c + hf3 * 16;
        const char* const a3b = scur + off_c + hb3 * 16;
        // ALINK + axpy epilogue: phi(x) is requested here, a step's worth of arithmetic before its use — with the links in their slots it is
        // the only global load of the loop, so its scoreboard waits for nothing else
        cplx<T> phi_pre[(ALINK && EPI == EPI_AXPY) ? NC : 1];
        if constexpr (ALINK && EPI == EPI_AXPY) {
            if (active) IO::template load<LD_STREAM>(phi_pre, phi_half, (size_t)(row0 + x0 * g.s0) * (IO::NCH * L3h) + h, L3h);
        }
        if constexpr (ALINK) {
            Link<T, 2> u;
            lds_site<T, NC>(nbA, a0f, cs);
            lds_site<T, NC>(nbB, a0b, cs);
            link_get(u, 0);
            hop_term<T, N, 0, true>(acc, nbA, open_link<OPEN>(u, cut_f0));
            link_request(0, p, 0, rown, h);
            lds_site<T, NC>(nbA, a1f, cs);
            link_get(u, 1);
            hop_term<T, N, 0, false>(acc, nbB, open_link<OPEN>(u, cut_b0));
            link_request(1, 1 - p, 0, row0 + (xn == 0 ? L0 - 1 : xn - 1) * g.s0, h);
            lds_site<T, NC>(nbB, a1b, cs);
            link_get(u, 2);
            hop_term<T, N, 1, true>(acc, nbA, open_link<OPEN>(u, cut_f1));
            link_request(2, p, 1, rown, h);
            lds_site<T, NC>(nbA, a2f, cs);
            link_get(u, 3);
            hop_term<T, N, 1, false>(acc, nbB, open_link<OPEN>(u, cut_b1));
            link_request(3, 1 - p, 1, rowb1_0 + xn * g.s0, h);
            lds_site<T, NC>(nbB, a2b, cs);
            link_get(u, 4);
            hop_term<T, N, 2, true>(acc, nbA, open_link<OPEN>(u, cut_f2));
            link_request(4, p, 2, rown, h);
            lds_site<T, NC>(nbA, a3f, cs);
            link_get(u, 5);
            hop_term<T, N, 2, false>(acc, nbB, open_link<OPEN>(u, cut_b2));
            link_request(5, 1 - p, 2, rowb2_0 + xn * g.s0, h);
            lds_site<T, NC>(nbB, a3b, cs);
            link_get(u, 6);
            hop_term<T, N, 3, true>(acc, nbA, open_link<OPEN>(u, cut_f3));
            link_request(6, p, 3, rown, h);
            link_get(u, 7);
            hop_term<T, N, 3, false>(acc, nbB, open_link<OPEN>(u, cut_b3));
            link_request(7, 1 - p, 3, rown, hb3n);
        } else {
        HR_NB_NEXT(nb0, a0f);
        HR_NB_NEXT(nb1, a0b); HR_NB_NOW(nb0, a0f);
        hop_term<T, N, 0, true>(acc, nb0, open_link<OPEN>(uf[0], cut_f0));
        load_link_rep<T, LP, ONFLY>(uf[0], a.gauge, g, p, 0, rown, h);
        HR_PIN();
        HR_NB_NEXT(nb0, a1f); HR_NB_NOW(nb1, a0b);
        hop_term<T, N, 0, false>(acc, nb1, open_link<OPEN>(ub[0], cut_b0));
        load_link_rep<T, LP, ONFLY>(ub[0], a.gauge, g, 1 - p, 0, row0 + (xn == 0 ? L0 - 1 : xn - 1) * g.s0, h);
        HR_PIN();
        HR_NB_NEXT(nb1, a1b); HR_NB_NOW(nb0, a1f);
        hop_term<T, N, 1, true>(acc, nb0, open_link<OPEN>(uf[1], cut_f1));
        load_link_rep<T, LP, ONFLY>(uf[1], a.gauge, g, p, 1, rown, h);
        HR_PIN();
        HR_NB_NEXT(nb0, a2f); HR_NB_NOW(nb1, a1b);
        hop_term<T, N, 1, false>(acc, nb1, open_link<OPEN>(ub[1], cut_b1));
        load_link_rep<T, LP, ONFLY>(ub[1], a.gauge, g, 1 - p, 1, rowb1_0 + xn * g.s0, h);
        HR_PIN();
        HR_NB_NEXT(nb1, a2b); HR_NB_NOW(nb0, a2f);
        hop_term<T, N, 2, true>(acc, nb0, open_link<OPEN>(uf[2], cut_f2));
        load_link_rep<T, LP, ONFLY>(uf[2], a.gauge, g, p, 2, rown, h);
        HR_PIN();
        HR_NB_NEXT(nb0, a3f); HR_NB_NOW(nb1, a2b);
        hop_term<T, N, 2, false>(acc, nb1, open_link<OPEN>(ub[2], cut_b2));
        load_link_rep<T, LP, ONFLY>(ub[2], a.gauge, g, 1 - p, 2, rowb2_0 + xn * g.s0, h);
        HR_PIN();
        HR_NB_NEXT(nb1, a3b); HR_NB_NOW(nb0, a3f);
        hop_term<T, N, 3, true>(acc, nb0, open_link<OPEN>(uf[3], cut_f3));
        load_link_rep<T, LP, ONFLY>(uf[3], a.gauge, g, p, 3, rown, h);
        HR_PIN();
        HR_NB_NOW(nb1, a3b);
        hop_term<T, N, 3, false>(acc, nb1, open_link<OPEN>(ub[3], cut_b3));
        load_link_rep<T, LP, ONFLY>(ub[3], a.gauge, g, 1 - p, 3, rown, hb3n);
        }
#undef HR_NB_NEXT
#undef HR_NB_NOW
#undef HR_PIN

        // all shared-memory reads of this step are consumed: hand the oldest plane and the halo buffer back
        __syncwarp();
        if ((tid & 31) == 0) {
            mbar_arrive(bar_empty + 8 * (k & 3));
            mbar_arrive(bar_hempty + 8 * hb);
        }
        // (requesting phi before the eight terms was measured slower at 48^4)
        constexpr bool PHI_PRE = ALINK && EPI == EPI_AXPY;
        if (POST == POST_STORE) {
            if (active) hop_epilogue<T, N, EPI, (SHARE ? LD_KEEP : LD_STREAM)>(acc, g, a, phi_half, out_half, p, row0 + x0 * g.s0, h, nullptr, (T)0, PHI_PRE ? phi_pre : nullptr);
        } else {
            if (active) hop_epilogue<T, N, EPI, LD_STREAM, POST>(acc, g, a, phi_half, out_half, p, row0 + x0 * g.s0, h, &cg_part, cg_alpha, PHI_PRE ? phi_pre : nullptr);
        }
    }
    if (ALINK) cp_async_wait<0>();   // the unused requests of the last step must not outlive the CTA
    if (POST != POST_STORE) {   // every plane and halo copy has been waited for and read: the ring is free to hold the warp sums
        const double tot = cta_sum_fixed(cg_part, reinterpret_cast<double*>(ring), pl.nconsumer, 1);
        if (tid == 0) a.partial[blockIdx.x] = tot;
    }
}

// ------------------------------------------------------------------ host side
constexpr size_t TILED_SMEM_LIMIT = 227 * 1024;

// the opt-in to > 48 KiB of dynamic shared memory is a per-device attribute of the kernel function: set once per
// instantiation and device (`flags`: 64 zero-initialised entries owned by the launch function of that instantiation;
// two host threads may both set the attribute, which is idempotent)
inline int opt_in_shared_memory(const void* kern, std::atomic<unsigned char>* flags, const char* name) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) { (void)cudaGetLastError(); dev = 0; }
    if (!flags[dev].load(std::memory_order_acquire)) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TILED_SMEM_LIMIT);
        if (e != cudaSuccess) { set_error("cudaFuncSetAttribute(%s): %s", name, cudaGetErrorString(e)); return HR_ECUDA; }
        flags[dev].store(1, std::memory_order_release);
    }
    return HR_OK;
}

// x0 segments per tile: minimise waves x (segment length + pipeline fill) over the divisors of L0
inline int tiled_segments(int L0, long tiles, long slots) {
    double best = 1e300;
    int nseg = 1;
    for (int ns = 1; ns <= L0; ++ns) {
        if (L0 % ns) continue;
        const long waves = (tiles * ns + slots - 1) / slots;
        const double cost = (double)waves * (L0 / ns + 3);
        if (cost < best - 1e-9) { best = cost; nseg = ns; }
    }
    return nseg;
}

inline bool tiled_plan_shape(const hr_geom* hg, int both, int num_sms, int t1, int t2, TiledPlan& pl) {
    const Geo g = make_geo(hg);
    const int L1 = hg->L[1], L2 = hg->L[2], L0 = hg->L[0];
    if (L1 % t1 || L2 % t2) return false;
    const int sites = t1 * t2 * g.L3h;
    if (sites > tiled_max_consumers(t1, t2)) return false;
    pl.t1 = t1;
    pl.t2 = t2;
    pl.nconsumer = (sites + 31) & ~31;
    pl.rowb = spinor_chunks(hg->rep, hg->prec) * g.L3h * 16;
    pl.smem = 128 + (size_t)pl.rowb * (TILED_RING * t1 * t2 + TILED_HALO * (2 * t1 + 2 * t2));
    if (pl.smem > TILED_SMEM_LIMIT) return false;
    pl.nt1 = L1 / t1;
    pl.nt2 = L2 / t2;
    const int cps = (!both && 2 * pl.smem + 2048 <= 228 * 1024 && hg->prec == HR_PREC_F32 && hg->rep == HR_REP_FUND && t1 * t2 <= 8) ? 2 : 1;  // CTAs per SM
    pl.nseg = tiled_segments(L0, (long)pl.nt1 * pl.nt2 * (both ? 2 : 1), (long)(num_sms > 0 ? num_sms : 148) * cps);
    pl.seglen = L0 / pl.nseg;
    return true;
}

// fills pl; false if the lattice fits no instantiated tile shape.  fp32 fundamental rows are half as long,
// so a 4 x 4 tile fits (2 row-loads per site instead of 2.5); everything else uses 2 x 4, or 2 x 2 for longer rows
// (24 < L3/2 <= 48) or L2 not a multiple of 4 (fundamental representation only).
inline bool tiled_plan(const hr_geom* hg, int both, int num_sms, TiledPlan& pl) {
    if (hg->prec == HR_PREC_F32 && hg->rep == HR_REP_FUND && tiled_plan_shape(hg, both, num_sms, 4, 4, pl)) return true;
    if (tiled_plan_shape(hg, both, num_sms, 2, 4, pl)) return true;
    return hg->rep == HR_REP_FUND && tiled_plan_shape(hg, both, num_sms, 2, 2, pl);
}

template <typename T, int N, int EPI, bool SHARE, int T1, int T2, bool ONFLY, int L3H, bool OPEN = false, int POST = POST_STORE>
inline int launch_hop_tiled_l3h(const Geo& g, const HopArgs& a, const TiledPlan& pl, cudaStream_t st) {
    // Link slots (ALINK) where the instantiation has them and 8 links x 16 / 32 bytes per consumer thread still fit.  Measured at 48^4
    // (profiles/r02_hop_alink.md): the bare and axpy hops gain (fp64 215.8 -> 206 us; 64^4 817 -> 694 us), the clover epilogues lose
    // (their 256-byte block loads need the L1 that the slots take: E2 724 -> 768 us) and so does the fp64 CG update stage (1320 -> 1328 us per
    // iteration); the norm stage and the fp32 CG stages gain.
    constexpr bool CAN_ALINK = HOP_ALINK && N == 2 && !SHARE && !ONFLY && (EPI == EPI_NONE || EPI == EPI_AXPY) && (POST != POST_CG_UPDATE || sizeof(T) == 4);
    if constexpr (CAN_ALINK) {
        const size_t smem = pl.smem + (size_t)8 * SiteIO<T, 2>::NCH * 16 * pl.nconsumer;
        if (smem <= TILED_SMEM_LIMIT) {
            auto kern = hop_tiled_kernel<T, N, EPI, T1, T2, SHARE, ONFLY, L3H, OPEN, POST, true>;
            static std::atomic<unsigned char> configured[64];
            const int rc = opt_in_shared_memory(reinterpret_cast<const void*>(kern), configured, "hop_tiled_kernel");
            if (rc != HR_OK) return rc;
            kern<<<(unsigned)(pl.nt1 * pl.nt2 * pl.nseg), pl.nconsumer + 32, smem, st>>>(g, a, pl);
            count_launch();
            return check_launch("hop_tiled_kernel");
        }
    }
    auto kern = hop_tiled_kernel<T, N, EPI, T1, T2, SHARE, ONFLY, L3H, OPEN, POST>;
    static std::atomic<unsigned char> configured[64];
    const int rc = opt_in_shared_memory(reinterpret_cast<const void*>(kern), configured, "hop_tiled_kernel");
    if (rc != HR_OK) return rc;
    const unsigned grid = (unsigned)((a.both ? 2 : 1) * pl.nt1 * pl.nt2 * pl.nseg);
    kern<<<grid, pl.nconsumer + 32, pl.smem, st>>>(g, a, pl);
    count_launch();
    return check_launch("hop_tiled_kernel");
}

template <typename T, int N, int EPI, bool SHARE, int T1, int T2, bool ONFLY, bool OPEN = false, int POST = POST_STORE>
inline int launch_hop_tiled_shape(const Geo& g, const HopArgs& a, const TiledPlan& pl, cudaStream_t st) {
    // compile-time L3/2 = 24 for the fp64 fundamental kernels (measured at 48^4: hop 219.3 -> 216.1 us; the fp32 4 x 4
    // kernel got slower with it)
    constexpr bool SPECIALISE = N == 2 && sizeof(T) == 8;
    if (SPECIALISE && g.L3h == 24) return launch_hop_tiled_l3h<T, N, EPI, SHARE, T1, T2, ONFLY, (SPECIALISE ? 24 : 0), OPEN, POST>(g, a, pl, st);
    return launch_hop_tiled_l3h<T, N, EPI, SHARE, T1, T2, ONFLY, 0, OPEN, POST>(g, a, pl, st);
}

template <typename T, int N, int EPI, bool SHARE, bool ONFLY, bool OPEN = false, int POST = POST_STORE>
inline int launch_hop_tiled_epi(const Geo& g, const HopArgs& a, const TiledPlan& pl, cudaStream_t st) {
    if (pl.t1 == 2 && pl.t2 == 4) return launch_hop_tiled_shape<T, N, EPI, SHARE, 2, 4, ONFLY, OPEN, POST>(g, a, pl, st);
    if (N == 2 && pl.t1 == 2 && pl.t2 == 2) return launch_hop_tiled_shape<T, 2, EPI, SHARE, 2, 2, false, OPEN, POST>(g, a, pl, st);
    if (sizeof(T) == 4 && N == 2 && pl.t1 == 4 && pl.t2 == 4) return launch_hop_tiled_shape<float, 2, EPI, SHARE, 4, 4, false, OPEN, POST>(g, a, pl, st);
    set_error("hop_tiled_kernel: no instantiation for a %d x %d tile", pl.t1, pl.t2);
    return HR_EUNSUPPORTED;
}

template <typename T, int N, bool ONFLY = false>
inline int launch_hop_tiled(const Geo& g, const HopArgs& a, int epi, const TiledPlan& pl, cudaStream_t st) {
    switch (epi) {
        case EPI_NONE: return launch_hop_tiled_epi<T, N, EPI_NONE, false, ONFLY>(g, a, pl, st);
        case EPI_AXPY:
            if (a.both) return launch_hop_tiled_epi<T, N, EPI_AXPY, true, ONFLY>(g, a, pl, st);
            return launch_hop_tiled_epi<T, N, EPI_AXPY, false, ONFLY>(g, a, pl, st);
        case EPI_CLOVER_INV: return launch_hop_tiled_epi<T, N, EPI_CLOVER_INV, false, ONFLY>(g, a, pl, st);
        case EPI_CLOVER_AXPY:
            if (a.both) return launch_hop_tiled_epi<T, N, EPI_CLOVER_AXPY, true, ONFLY>(g, a, pl, st);   // H3c: links re-read by the other parity's CTA
            return launch_hop_tiled_epi<T, N, EPI_CLOVER_AXPY, false, ONFLY>(g, a, pl, st);
        default: set_error("unknown epilogue %d", epi); return HR_EINVAL;
    }
}

// the open-boundary instantiations (fundamental representation, one parity per launch) live in their own translation unit,
// hr_hop_open.cu, so that they compile in parallel with the rest
template <typename T>
int launch_hop_tiled_open(const Geo& g, const HopArgs& a, int epi, const TiledPlan& pl, cudaStream_t st);

}  // namespace hr
