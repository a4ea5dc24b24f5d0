// hr_dirac_tiled.cuh — the full-lattice operator D psi = (4+m0) psi - 1/2 H psi in ONE launch (step H3 of DESIGN.md §2,
// design in §5.3): an x0-marching tile kernel in which one CTA computes BOTH parities of its tile.
//
// Same pipeline as hop_tiled_kernel (hr_hop_tiled.cuh): a producer thread moves whole x3-rows of the input field into
// shared memory with 1-D bulk asynchronous copies that complete on mbarriers; consumer threads gather from there.
// What differs, and why (profiles/r02_kernels.md):
//   * A consumer thread owns a spatial column (x1, x2, x3) and keeps it for the whole march, so the parity of its site
//     alternates from plane to plane.  Its own spinors are then the x0 neighbours of its own sites: psi(x0+1) is read
//     from shared memory once and serves three steps from registers — as the forward neighbour, as the axpy operand
//     phi(x) = psi(x) of the next step, and (spin-projected, 8 reals instead of 16) as the backward neighbour of the
//     step after.  Per output site that is 7 spinor reads from shared memory instead of 9 + a global phi read.
//   * The link U_0(x) is used by the forward term at x and by the backward term at x+0 — the same thread one step
//     later: it stays in registers (7 link loads per site instead of 8).
//   * The other seven links of a site do NOT travel through registers: each thread owns seven slots in shared memory that it
//     fills with cp.async and re-requests right after use (ALINK, see cp_async16 below) — a register load requested a step
//     ahead is in fact waited for together with every later global load of the warp (one scoreboard).
//   * Plane x0-1 is never read from shared memory: the ring holds planes x0, x0+1 and the plane(s) in flight (3 slots in fp64 with
//     ALINK, else 4); the halo rows (x1 and x2 neighbours of the tile edge, centre plane only) have their own buffers
//     and their own mbarriers so that they do not hold the plane copies back, and are requested before the plane.
//   * The eight terms run x0-1, x3+-, [halo wait] x1+-, x2+-, x0+1, and the neighbour of term t+1 is read from shared memory
//     before term t is computed (two register images).
//   * Every plane and halo buffer holds the even and the odd half-rows ([parity][row]); both uses of a link happen in
//     the same CTA in the same step, so the second one hits L1/L2 and DRAM sees every link once.
#pragma once

#include "hr_hop_tiled.cuh"

namespace hr {

// Buffers with the links in registers (ALINK = false, the form for rows too long for the link slots): DT_RING ring slots hold
// planes x0, x0+1 and two planes in flight, DT_HALO halo buffers the halo of the centre plane and one in flight; more than
// ~196 KiB of shared memory then starves the L1 the link loads go through (profiles/r02_kernels.md).
constexpr int DT_RING = 4;
constexpr int DT_HALO = 2;
// With the links in shared-memory slots (ALINK) nothing goes through L1 and all 227 KiB can be used.  fp64 (2 x 2 tile): 3 planes + 2 halo
// buffers + link slots = 211 KiB at L3 = 48 — no room for more.  fp32 (2 x 4 tile): 4 planes + 2 halo buffers + link slots = 210 KiB: the
// plane in flight then has almost three steps to land instead of almost two; with 3 planes + 3 halo buffers (223 KiB) the wait for the
// x0+1 plane was the top stall of the fp32 kernel (11.5 % of the samples, profiles/r02_dirac_alink.md section 8): 179.2 -> 175.1 us.
__host__ __device__ constexpr int dt_ring(bool alink, size_t real_bytes) { return (alink && real_bytes == 8) ? 3 : DT_RING; }
__host__ __device__ constexpr int dt_nhalo(bool alink, size_t real_bytes) { return DT_HALO; }

// consumer threads the kernel is compiled for: one per site of a T1 x T2 tile of full x3-rows of up to 48 sites (2 x 2, 2 x 4 tiles) or
// up to 96 sites (the 1 x 2 tile of long rows, L3 = 50 .. 96)
constexpr int dt_max_consumers(int t1, int t2) { return t1 * t2 * (t1 * t2 <= 2 ? 96 : 48); }

struct DiracPlan {
    int t1, t2;        // tile shape in rows (x1, x2)
    int nt1, nt2;      // tiles along x1, x2
    int nseg, seglen;  // x0 segments per tile and their length
    int nconsumer;     // consumer threads: 2 * (T1*T2*L3h rounded up to a warp)
    int rowb;          // bytes of one x3-row of one parity
    int alink;         // links through cp.async slots in shared memory (else in registers)
    size_t smem;
};

// The producer of the full-lattice kernels (one thread): per iteration the T1 x T2 tile rows of plane j, both parity images, into
// ring slot j % DT_RING and the halo rows of centre plane j - HLAG into halo buffer (pc-1) % DT_HALO; waits on the slot's "empty"
// mbarrier, arms its "full" mbarrier with the byte count.  Shared by dirac_tiled_kernel and dirac_split_kernel (hr_dirac_split.cuh).
template <int T1, int T2, int RING, int NHALO>
__device__ __forceinline__ void dirac_producer(const char* in, size_t half_bytes, char* ring, char* halo, int rowb, uint32_t bar_full,
                                               uint32_t bar_empty, uint32_t bar_hfull, uint32_t bar_hempty, int t1, int t2, int xs,
                                               int nsteps, int L0, int L1, int L2) {
    constexpr int TR = T1 * T2, HR = 2 * T2 + 2 * T1;
    const int planeb = 2 * TR * rowb, halob = 2 * HR * rowb;
    const int x1base = t1 * T1, x2base = t2 * T2;
    const int x1lo = (x1base - 1 + L1) % L1, x1hi = (x1base + T1) % L1;
    const int x2lo = (x2base - 1 + L2) % L2, x2hi = (x2base + T2) % L2;
    // plane P can be requested once plane P - RING is dead (after step P - RING - 1), the halo of centre Pc once
    // that of centre Pc - NHALO is (after step Pc - NHALO - 1): iteration j issues plane j and the halo of centre
    // j - (RING - NHALO), which become free at the same time
    constexpr int HLAG = RING - NHALO;
    static_assert(HLAG >= 0 && HLAG <= RING - 2, "iterations up to the request of the halo of plane 1 must not wait for a consumer");
    for (int j = 0; j < nsteps + 2 + HLAG; ++j) {
        const int pc = j - HLAG;   // halo of a centre plane (the planes 1..nsteps are centres)
        if (pc >= 1 && pc <= nsteps) {
            const int hb = (pc - 1) % NHALO;
            mbar_wait(bar_hempty + 8 * hb, (((uint32_t)(pc - 1) / NHALO) & 1) ^ 1);
            const uint32_t full = bar_hfull + 8 * hb;
            mbar_expect_tx(full, (uint32_t)halob);
            const int x0h = (xs - 1 + pc + L0) % L0;
#pragma unroll
            for (int pp = 0; pp < 2; ++pp) {
                const char* src = in + pp * half_bytes;
                const uint32_t hd = smem_u32(halo + hb * halob + pp * HR * rowb);
                bulk_g2s(hd, src + (((size_t)x0h * L1 + x1lo) * L2 + x2base) * rowb, (uint32_t)(T2 * rowb), full);
                bulk_g2s(hd + T2 * rowb, src + (((size_t)x0h * L1 + x1hi) * L2 + x2base) * rowb, (uint32_t)(T2 * rowb), full);
#pragma unroll
                for (int aa = 0; aa < T1; ++aa) {
                    const size_t rb = ((size_t)x0h * L1 + x1base + aa) * L2;
                    bulk_g2s(hd + (2 * T2 + aa) * rowb, src + (rb + x2lo) * rowb, (uint32_t)rowb, full);
                    bulk_g2s(hd + (2 * T2 + T1 + aa) * rowb, src + (rb + x2hi) * rowb, (uint32_t)rowb, full);
                }
            }
        }
        if (j < nsteps + 2) {   // plane P = j
            const int slot = j % RING;
            mbar_wait(bar_empty + 8 * slot, (((uint32_t)j / RING) & 1) ^ 1);
            const uint32_t full = bar_full + 8 * slot;
            mbar_expect_tx(full, (uint32_t)planeb);
            const int x0p = (xs - 1 + j + L0) % L0;
#pragma unroll
            for (int pp = 0; pp < 2; ++pp) {
                const uint32_t dst = smem_u32(ring + slot * planeb + pp * TR * rowb);
#pragma unroll
                for (int aa = 0; aa < T1; ++aa) {
                    const size_t row = ((size_t)x0p * L1 + x1base + aa) * L2 + x2base;
                    bulk_g2s(dst + aa * T2 * rowb, in + pp * half_bytes + row * rowb, (uint32_t)(T2 * rowb), full);
                }
            }
        }
    }
}

// grid.x = nt1 * nt2 * nseg.  Shared memory: [16 mbarriers][DT_RING planes][DT_HALO halo buffers],
//   plane: [parity 0,1][T1*T2 rows];  halo buffer: [parity 0,1][x1-1 line: T2 rows][x1+T1 line: T2][x2-1: T1][x2+T2: T1]
// Plane index P = x0 - xs + 1 (P = 0 is the plane below the segment, read once in the prologue), ring slot P % DT_RING;
// the halo of centre plane P sits in halo buffer (P-1) % NHALO.
// ALINK: links through cp.async slots in shared memory (see above) instead of registers; the fp64 form then has a 3-slot ring.
template <typename T, int T1, int T2, int L3H, bool ALINK>
__global__ void __launch_bounds__(dt_max_consumers(T1, T2) + 32, 1) dirac_tiled_kernel(Geo g_in, HopArgs a, DiracPlan pl) {
    constexpr int N = 2, NC = 8;
    constexpr int RING = dt_ring(ALINK, sizeof(T)), NHALO = dt_nhalo(ALINK, sizeof(T));
    typedef SiteIO<T, NC> IO;
    constexpr int TR = T1 * T2, HR = 2 * T2 + 2 * T1;
    constexpr int LP = LD_KEEP;   // both uses of a link are in this CTA: keep the line for the second one
    Geo g = g_in;
    if (L3H > 0) g.L3h = L3H;
    extern __shared__ __align__(128) char smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);
    char* ring = smem + 128;
    const int rowb = L3H > 0 ? IO::NCH * L3H * 16 : pl.rowb;
    const int planeb = 2 * TR * rowb, halob = 2 * HR * rowb;
    char* halo = ring + RING * planeb;
    char* lbuf = halo + NHALO * halob;   // ALINK: link slots [link][chunk][consumer thread]
    static_assert(RING >= 3 && RING <= 4 && NHALO >= 2 && NHALO <= 4, "16 mbarriers: 4 + 4 + 4 + 4");
    const uint32_t bar_full = smem_u32(bars);          // [RING]
    const uint32_t bar_empty = smem_u32(bars + 4);     // [RING]
    const uint32_t bar_hfull = smem_u32(bars + 8);     // [NHALO]
    const uint32_t bar_hempty = smem_u32(bars + 12);   // [NHALO]

    const int tid = threadIdx.x;
    const int ncw = pl.nconsumer >> 5;
    if (tid == 0) {
        for (int i = 0; i < RING; ++i) { mbar_init(bar_full + 8 * i, 1); mbar_init(bar_empty + 8 * i, ncw); }
        for (int i = 0; i < NHALO; ++i) { mbar_init(bar_hfull + 8 * i, 1); mbar_init(bar_hempty + 8 * i, ncw); }
        mbar_fence_init();
    }
    __syncthreads();

    const int bid = blockIdx.x;
    const int seg = bid / (pl.nt1 * pl.nt2);
    const int tile = bid - seg * (pl.nt1 * pl.nt2);
    const int t1 = tile / pl.nt2, t2 = tile - t1 * pl.nt2;
    const int xs = seg * pl.seglen, nsteps = pl.seglen;
    const int L0 = g.L0, L1 = g.s0 / g.s1, L2 = g.s1;
    const size_t half_bytes = (size_t)g.Vh * IO::NCH * 16;
    const char* in = reinterpret_cast<const char*>(a.in);

    if (tid >= pl.nconsumer) {
        // ================================================================ producer (one thread)
        if (tid != pl.nconsumer) return;
        dirac_producer<T1, T2, RING, NHALO>(in, half_bytes, ring, halo, rowb, bar_full, bar_empty, bar_hfull, bar_hempty, t1, t2, xs, nsteps, L0, L1, L2);
        return;
    }

    // ================================================================ consumers: one thread per spatial column
    const int L3h = g.L3h;
    const int nsp = pl.nconsumer >> 1;               // threads per x3-offset class q (x3 = 2h + q)
    const int q = tid >= nsp ? 1 : 0;
    const int stid = tid - q * nsp;
    const bool active = stid < TR * L3h;
    const int ctid = active ? stid : 0;              // idle threads shadow column 0 and store nothing
    const int lr = ctid / L3h, h = ctid - lr * L3h;
    const int la = lr / T2, lb = lr - la * T2;
    const int x1 = t1 * T1 + la, x2 = t2 * T2 + lb;
    const int cs = L3h * 16;
    const int hf3 = q ? (h == L3h - 1 ? 0 : h + 1) : h;      // pair index of the x3+1 / x3-1 neighbour (other parity image)
    const int hb3 = q ? h : (h == 0 ? L3h - 1 : h - 1);
    const bool f1_in = la + 1 < T1, b1_in = la > 0, f2_in = lb + 1 < T2, b2_in = lb > 0;
    // byte offsets inside one parity image of a plane (in-tile neighbour) or of a halo buffer
    const int off_c = lr * rowb + h * 16;
    const int off_f1 = (f1_in ? (lr + T2) : (T2 + lb)) * rowb + h * 16;
    const int off_b1 = (b1_in ? (lr - T2) : lb) * rowb + h * 16;
    const int off_f2 = (f2_in ? (lr + 1) : (2 * T2 + T1 + la)) * rowb + h * 16;
    const int off_b2 = (b2_in ? (lr - 1) : (2 * T2 + la)) * rowb + h * 16;
    const int off_f3 = lr * rowb + hf3 * 16, off_b3 = lr * rowb + hb3 * 16;
    const int pimg = TR * rowb, himg = HR * rowb;    // image strides (parity 1 follows parity 0)
    const int row0 = x1 * g.s1 + x2;
    const int rowb1_0 = (x1 == 0 ? L1 - 1 : x1 - 1) * g.s1 + x2;
    const int rowb2_0 = x1 * g.s1 + (x2 == 0 ? L2 - 1 : x2 - 1);
    const T ca = (T)a.a, cc = (T)a.c;

    // ---- prologue: psi(xs) of this column, the projected psi(xs-1), U_0(xs-1), the links of the first step
    cplx<T> psic[NC], hb0[N], hb1[N];
    Link<T, N> ul[ALINK ? 1 : 7], ub0;    // ub0 = U_0(x - 0): the U_0(x) of the previous step; ul: the seven others when they live in registers
    // link j of this site: 0..5 = U_1(x), U_1(x-1), U_2(x), U_2(x-2), U_3(x), U_3(x-3); 6 = U_0(x)
    constexpr int LCH = SiteIO<T, 2>::NCH;                     // 16-byte chunks of a compressed link
    const uint32_t lslot = smem_u32(lbuf) + (uint32_t)tid * 16;
    const int lchb = pl.nconsumer * 16;                        // one chunk of one link for all consumer threads
    // ALINK: the address of link j is carried from step to step — one x0-plane further and into the other parity half, since the
    // parity of the column's site alternates: + s0 rows +- the parity stride, the sign swapping every step and opposite for the
    // forward links (parity of the site) and the backward ones (other parity) — instead of the full index arithmetic
    // ((par*4 + mu)*R + row)*W + h per link and step.  fp64: seven 64-bit pointers.  fp32 (13 warps: 128 registers at most): seven
    // 32-bit offsets in 16-byte units from the start of the gauge field (the plan refuses fields of 2^32 chunks or more).
    constexpr bool RUN64 = ALINK && sizeof(T) == 8, RUN32 = ALINK && sizeof(T) == 4;
    const char* lptr[RUN64 ? 7 : 1];
    uint32_t loff[RUN32 ? 7 : 1];
    const long long lrow = (long long)(LCH * L3h);                                   // 16-byte chunks of one row of links of one parity and direction
    const long long dplus = ((long long)g.s0 + 4 * (long long)g.R) * lrow, dminus = ((long long)g.s0 - 4 * (long long)g.R) * lrow;
    long long dstep_f = 0, dstep_b = 0;                                              // this step's advance of the forward / backward links (bytes)
    uint32_t ostep_f = 0, ostep_b = 0;                                               // the same in chunks, modulo 2^32
    bool more = true;                                                                // a next step exists (its links are requested)
    auto link_issue = [&](int j) {
        const char* src = RUN64 ? lptr[RUN64 ? j : 0] : reinterpret_cast<const char*>(a.gauge) + (size_t)loff[RUN32 ? j : 0] * 16;
#pragma unroll
        for (int c = 0; c < LCH; ++c) cp_async16(lslot + (j * LCH + c) * lchb, src + (size_t)c * cs);
    };
    auto link_request = [&](int j, int par, int mu, int row, int hh) {      // prologue (and every step with the links in registers)
        if constexpr (ALINK) {
            const size_t chunk = ((size_t)(par * 4 + mu) * g.R + row) * (LCH * L3h) + hh;
            if constexpr (RUN64) lptr[j] = reinterpret_cast<const char*>(a.gauge) + chunk * 16;
            else loff[j] = (uint32_t)chunk;
            link_issue(j);
            cp_async_commit();
        } else {
            load_link_rep<T, LP, false>(ul[j], a.gauge, g, par, mu, row, hh);
        }
    };
    auto link_next = [&](int j, bool fwd, int par, int mu, int row, int hh) {
        if constexpr (ALINK) {
            if constexpr (RUN64) lptr[j] += fwd ? dstep_f : dstep_b;
            else loff[j] += fwd ? ostep_f : ostep_b;
            if (more) link_issue(j);     // no request past the last plane of the segment (the address may lie outside the field)
            cp_async_commit();           // the (possibly empty) group keeps the wait_group count
        } else {
            load_link_rep<T, LP, false>(ul[j], a.gauge, g, par, mu, row, hh);
        }
    };
    auto link_get = [&](Link<T, N>& u, int j) {
        if constexpr (ALINK) {
            cp_async_wait<6>();      // all but the six newest requests have landed: slot j has
            cplx<T> ab[2];
            lds_link(ab, lslot + j * LCH * lchb, lchb);
            u.a = ab[0];
            u.b = ab[1];
        } else {
            u = ul[j];
        }
    };
    {
        const int p0 = (xs + x1 + x2 + q) & 1;
        const int row = row0 + xs * g.s0;
        link_request(0, p0, 3, row, h);
        link_request(1, 1 - p0, 3, row, hb3);
        link_request(2, p0, 1, row, h);
        link_request(3, 1 - p0, 1, rowb1_0 + xs * g.s0, h);
        link_request(4, p0, 2, row, h);
        link_request(5, 1 - p0, 2, rowb2_0 + xs * g.s0, h);
        link_request(6, p0, 0, row, h);
        load_link_rep<T, LP, false>(ub0, a.gauge, g, 1 - p0, 0, row0 + (xs == 0 ? L0 - 1 : xs - 1) * g.s0, h);
        mbar_wait(bar_full, 0);
        mbar_wait(bar_full + 8, 0);
        cplx<T> below[NC];
        lds_site<T, NC>(below, ring + (1 - p0) * pimg + off_c, cs);
        hop_project<T, N, 0, false>(hb0, hb1, below);
        lds_site<T, NC>(psic, ring + planeb + p0 * pimg + off_c, cs);
        __syncwarp();
        if ((tid & 31) == 0) mbar_arrive(bar_empty);
    }

    for (int k = 0; k < nsteps; ++k) {
        const int x0 = xs + k;
        const int p = (x0 + x1 + x2 + q) & 1;
        const char* scur = ring + ((k + 1) % RING) * planeb + (1 - p) * pimg;     // neighbours live in the other parity's image
        const char* snext = ring + ((k + 2) % RING) * planeb + (1 - p) * pimg;
        const int hbuf = k % NHALO;
        const char* shalo = halo + hbuf * halob + (1 - p) * himg;
        // next step's plane and parity (clamped on the last step: the reload is then harmless and unused)
        const int xn = (k + 1 < nsteps) ? x0 + 1 : x0;
        const int pn = (xn + x1 + x2 + q) & 1;
        const int rown = row0 + xn * g.s0;
        if constexpr (ALINK) {
            more = k + 1 < nsteps;
            if constexpr (RUN64) {
                dstep_f = 16 * (p ? dminus : dplus);
                dstep_b = 16 * (p ? dplus : dminus);
            } else {
                ostep_f = (uint32_t)(p ? dminus : dplus);
                ostep_b = (uint32_t)(p ? dplus : dminus);
            }
        }

        // Eight terms: x0-1 from registers, x3+- from the centre plane, then (halo wait) x1+-, x2+- from the centre plane and its halo
        // rows, last x0+1 from the newest plane.  Each link is re-requested for the next step right after its use.
        cplx<T> acc[NC], nb[NC], nb2[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) acc[c] = mk<T>((T)0, (T)0);
        Link<T, N> u;
        // the neighbour of term t+1 is read from shared memory before term t is computed (two register images)
        lds_site<T, NC>(nb, scur + off_f3, cs);
        hop_apply<T, N, 0, false>(acc, hb0, hb1, ub0);
        lds_site<T, NC>(nb2, scur + off_b3, cs);
        link_get(u, 0);
        hop_term<T, N, 3, true>(acc, nb, u);
        link_next(0, true, pn, 3, rown, h);
        mbar_wait(bar_hfull + 8 * hbuf, ((uint32_t)k / NHALO) & 1);
        lds_site<T, NC>(nb, (f1_in ? scur : shalo) + off_f1, cs);
        link_get(u, 1);
        hop_term<T, N, 3, false>(acc, nb2, u);
        link_next(1, false, 1 - pn, 3, rown, hb3);
        lds_site<T, NC>(nb2, (b1_in ? scur : shalo) + off_b1, cs);
        link_get(u, 2);
        hop_term<T, N, 1, true>(acc, nb, u);
        link_next(2, true, pn, 1, rown, h);
        lds_site<T, NC>(nb, (f2_in ? scur : shalo) + off_f2, cs);
        link_get(u, 3);
        hop_term<T, N, 1, false>(acc, nb2, u);
        link_next(3, false, 1 - pn, 1, rowb1_0 + xn * g.s0, h);
        lds_site<T, NC>(nb2, (b2_in ? scur : shalo) + off_b2, cs);
        link_get(u, 4);
        hop_term<T, N, 2, true>(acc, nb, u);
        link_next(4, true, pn, 2, rown, h);
        // x0+1: this column's own spinor of the next plane — its copy had two steps to land
        mbar_wait(bar_full + 8 * ((k + 2) % RING), ((uint32_t)(k + 2) / RING) & 1);
        lds_site<T, NC>(nb, snext + off_c, cs);
        link_get(u, 5);
        hop_term<T, N, 2, false>(acc, nb2, u);
        link_next(5, false, 1 - pn, 2, rowb2_0 + xn * g.s0, h);
        link_get(u, 6);
        hop_term<T, N, 0, true>(acc, nb, u);
        ub0 = u;
        link_next(6, true, pn, 0, rown, h);
        // the centre plane and its halo are consumed
        __syncwarp();
        if ((tid & 31) == 0) {
            mbar_arrive(bar_empty + 8 * ((k + 1) % RING));
            mbar_arrive(bar_hempty + 8 * hbuf);
        }
        // out = (4+m0) psi(x) - 1/2 H psi(x)
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            acc[c].re = fma(cc, acc[c].re, ca * psic[c].re);
            acc[c].im = fma(cc, acc[c].im, ca * psic[c].im);
        }
        if (active) IO::store(reinterpret_cast<char*>(a.out) + (size_t)p * half_bytes, (size_t)(row0 + x0 * g.s0) * (IO::NCH * L3h) + h, L3h, acc);
        hop_project<T, N, 0, false>(hb0, hb1, psic);
#pragma unroll
        for (int c = 0; c < NC; ++c) psic[c] = nb[c];
    }
    if constexpr (ALINK) cp_async_wait<0>();   // the unused requests of the last step must not outlive the CTA
}

// ------------------------------------------------------------------ host side
inline bool dirac_plan_shape(const hr_geom* hg, int num_sms, int t1, int t2, DiracPlan& pl, bool alink = true) {
    const Geo g = make_geo(hg);
    const int L1 = hg->L[1], L2 = hg->L[2], L0 = hg->L[0];
    if (L1 % t1 || L2 % t2) return false;
    const int sites = t1 * t2 * g.L3h;            // per x3-offset class
    if (2 * sites > dt_max_consumers(t1, t2)) return false;
    pl.t1 = t1;
    pl.t2 = t2;
    pl.nconsumer = 2 * ((sites + 31) & ~31);
    if (pl.nconsumer > dt_max_consumers(t1, t2)) return false;
    pl.rowb = spinor_chunks(hg->rep, hg->prec) * g.L3h * 16;
    // the fp32 kernel addresses its link slots' sources by 32-bit chunk offsets
    if (alink && hg->prec == HR_PREC_F32 && (unsigned long long)8 * g.R * link_chunks(hg->prec) * g.L3h >= (1ull << 32)) alink = false;
    pl.alink = alink ? 1 : 0;
    const int ring = dt_ring(alink, real_bytes(hg->prec)), nhalo = dt_nhalo(alink, real_bytes(hg->prec));
    pl.smem = 128 + (size_t)pl.rowb * 2 * (ring * t1 * t2 + nhalo * (2 * t1 + 2 * t2)) +
              (alink ? (size_t)7 * link_chunks(hg->prec) * 16 * pl.nconsumer : 0);
    if (pl.smem > TILED_SMEM_LIMIT) return alink ? dirac_plan_shape(hg, num_sms, t1, t2, pl, false) : false;
    pl.nt1 = L1 / t1;
    pl.nt2 = L2 / t2;
    pl.nseg = tiled_segments(L0, (long)pl.nt1 * pl.nt2, num_sms > 0 ? num_sms : 148);
    pl.seglen = L0 / pl.nseg;
    return true;
}

// fundamental representation only: 2 x 2 rows in fp64, 2 x 4 in fp32 (rows half as long), 1 x 2 for rows too long for those
inline bool dirac_plan(const hr_geom* hg, int num_sms, DiracPlan& pl, bool alink = true) {
    if (hg->rep != HR_REP_FUND) return false;
    if (hg->prec == HR_PREC_F32 && dirac_plan_shape(hg, num_sms, 2, 4, pl, alink)) return true;
    if (dirac_plan_shape(hg, num_sms, 2, 2, pl, alink)) return true;
    return dirac_plan_shape(hg, num_sms, 1, 2, pl, alink);      // long rows (L3 = 50 .. 96)
}

template <typename T, int T1, int T2, int L3H, bool ALINK>
inline int launch_dirac_tiled_l3h(const Geo& g, const HopArgs& a, const DiracPlan& pl, cudaStream_t st) {
    auto kern = dirac_tiled_kernel<T, T1, T2, L3H, ALINK>;
    static std::atomic<unsigned char> configured[64];
    const int rc = opt_in_shared_memory(reinterpret_cast<const void*>(kern), configured, "dirac_tiled_kernel");
    if (rc != HR_OK) return rc;
    kern<<<(unsigned)(pl.nt1 * pl.nt2 * pl.nseg), pl.nconsumer + 32, pl.smem, st>>>(g, a, pl);
    count_launch();
    return check_launch("dirac_tiled_kernel");
}

template <typename T, bool ALINK>
inline int launch_dirac_tiled_a(const Geo& g, const HopArgs& a, const DiracPlan& pl, cudaStream_t st) {
    if constexpr (sizeof(T) == 4) {
        if (pl.t1 == 2 && pl.t2 == 4) {
            if (g.L3h == 24) return launch_dirac_tiled_l3h<T, 2, 4, 24, ALINK>(g, a, pl, st);
            return launch_dirac_tiled_l3h<T, 2, 4, 0, ALINK>(g, a, pl, st);
        }
    }
    if (pl.t1 == 1 && pl.t2 == 2) return launch_dirac_tiled_l3h<T, 1, 2, 0, ALINK>(g, a, pl, st);
    if (g.L3h == 24) return launch_dirac_tiled_l3h<T, 2, 2, 24, ALINK>(g, a, pl, st);
    return launch_dirac_tiled_l3h<T, 2, 2, 0, ALINK>(g, a, pl, st);
}
template <typename T>
inline int launch_dirac_tiled(const Geo& g, const HopArgs& a, const DiracPlan& pl, cudaStream_t st) {
    return pl.alink ? launch_dirac_tiled_a<T, true>(g, a, pl, st) : launch_dirac_tiled_a<T, false>(g, a, pl, st);
}

}  // namespace hr
