// hr_halo.cu — the sharded (domain-decomposed) hop: face packing and the boundary kernel.
//
// PAPER.md:31 §2.1: "inner computations ... boundary calculation ... a kernel that synchronizes the send buffer";
// communications overlap the inner kernel; Fig. 4: all four dimensions parallelised.
// Each rank holds a local lattice in the ordinary device layout.  For a direction mu that is cut between ranks, the
// terms of the hopping sum that cross the cut are left out of the local kernel (HopArgs::open_mask) and arrive as
// faces of spin-projected half spinors — 2N complex numbers per face site instead of 4N, and the backward face already
// multiplied by the sender's link, so links never move:
//   face 2mu   ("down", sites with x_mu = 0,       sent to the rank at -mu): (h0, h1) of (1 - gamma_mu) psi(y)
//             -> the receiver's forward term at x = y - mu (its x_mu = L_mu-1):  acc += rebuild(U_mu(x) h)
//   face 2mu+1 ("up",   sites with x_mu = L_mu-1,  sent to the rank at +mu): U_mu(y)^dag (h0, h1) of (1 + gamma_mu) psi(y)
//             -> the receiver's backward term at x = y + mu (its x_mu = 0):      acc += rebuild(w)
// A face holds the sites of ONE parity (the input parity of the hop), indexed by the three other coordinates:
//   fi = lex3(other coordinates, last one fastest) / 2, chunk c of face site fi at 16-byte index c*nface + fi
// (sender and receiver agree on fi because they share the other three coordinates).  hr_halo_pack may write a face
// straight into the neighbour's receive buffer when that is peer-mapped (NVLink): the pointer is the caller's.
#include "hr_hop_generic.cuh"

namespace hr {

struct FaceGeo {
    int mu;          // the cut direction
    int o[3];        // the other directions, increasing
    int E[3];        // their extents
    int nface;       // face sites of one parity = E0*E1*E2/2
};

static FaceGeo make_face(const hr_geom* hg, int mu) {
    FaceGeo f;
    f.mu = mu;
    int k = 0;
    for (int d = 0; d < 4; ++d)
        if (d != mu) { f.o[k] = d; f.E[k] = hg->L[d]; ++k; }
    f.nface = f.E[0] * f.E[1] * f.E[2] / 2;
    return f;
}

// coordinates of face site fi of parity `par` on the plane x_mu = xmu
__device__ __forceinline__ void face_site(const FaceGeo& f, int fi, int xmu, int par, int x[4]) {
    const int pair = 2 * fi;
    const int c2 = pair % f.E[2];
    const int t = pair / f.E[2];
    const int c1 = t % f.E[1], c0 = t / f.E[1];
    const int r = (par + xmu + c0 + c1 + c2) & 1;      // c2 is even: the two sites of the pair are c2 and c2+1
    x[f.mu] = xmu;
    x[f.o[0]] = c0;
    x[f.o[1]] = c1;
    x[f.o[2]] = c2 + r;
}

// half spinor (2N complex) <-> face buffer chunks
template <typename T, int N>
__device__ __forceinline__ void face_store(void* face, int nface, int fi, const cplx<T>* h0, const cplx<T>* h1) {
    cplx<T> v[2 * N];
#pragma unroll
    for (int c = 0; c < N; ++c) { v[c] = h0[c]; v[N + c] = h1[c]; }
    SiteIO<T, 2 * N>::store(face, (size_t)fi, nface, v);
}
template <typename T, int N>
__device__ __forceinline__ void face_load(const void* face, int nface, int fi, cplx<T>* h0, cplx<T>* h1) {
    cplx<T> v[2 * N];
    SiteIO<T, 2 * N>::template load<LD_STREAM>(v, face, (size_t)fi, nface);
#pragma unroll
    for (int c = 0; c < N; ++c) { h0[c] = v[c]; h1[c] = v[N + c]; }
}

template <typename T, int N, int MU, bool UP, bool ONFLY, bool C3>
__device__ __forceinline__ void pack_one(const Geo& g, const FaceGeo& f, int par, const void* gauge, const void* in_half, void* face, int fi) {
    constexpr int NC = 4 * N;
    int x[4];
    face_site(f, fi, UP ? (MU == 0 ? g.L0 : MU == 1 ? g.L1 : MU == 2 ? g.L2 : 2 * g.L3h) - 1 : 0, par, x);
    const int row = (x[0] * g.L1 + x[1]) * g.L2 + x[2], h = x[3] >> 1;
    cplx<T> psi[NC], h0[N], h1[N];
    SiteIO<T, NC>::template load<LD_KEEP>(psi, in_half, (size_t)row * (SiteIO<T, NC>::NCH * g.L3h) + h, g.L3h);
    if (!UP) {
        hop_project<T, N, MU, true>(h0, h1, psi);                  // (1 - gamma_mu) psi: the neighbour's forward term
        face_store<T, N>(face, f.nface, fi, h0, h1);
    } else {
        hop_project<T, N, MU, false>(h0, h1, psi);                 // (1 + gamma_mu) psi, times this site's link^dag
        typename std::conditional<C3, LinkC3<T>, Link<T, N>>::type u;    // C3: complex 3 x 3 links (HR_REP_SU3)
        load_link_rep<T, LD_STREAM, ONFLY>(u, gauge, g, par, MU, row, h);
        cplx<T> c0[N], c1[N];
        mul_link_dag(c0, u, h0);
        mul_link_dag(c1, u, h1);
        face_store<T, N>(face, f.nface, fi, c0, c1);
    }
}

// one thread per face site, blockIdx.y = the face (2 per cut direction): ONE launch packs every face of the rank.
// in_half: half field of parity `par`
struct PackJob {
    FaceGeo f[4];
    void* face[8];
    int slot[8];     // slot[j] = face index 2*mu + up of the j-th face to pack
    int nslots;
};
template <typename T, int N, bool ONFLY, bool C3>
__global__ void __launch_bounds__(128) halo_pack_kernel(Geo g, PackJob job, int par, const void* gauge, const void* in_half) {
    const int fidx = job.slot[blockIdx.y];
    const int mu = fidx >> 1, up = fidx & 1;
    const FaceGeo& f = job.f[mu];
    const int fi = blockIdx.x * blockDim.x + threadIdx.x;
    if (fi >= f.nface) return;
    void* face = job.face[fidx];
#define HR_PACK(MU)                                                                        \
    if (mu == MU) {                                                                        \
        if (up) pack_one<T, N, MU, true, ONFLY, C3>(g, f, par, gauge, in_half, face, fi);      \
        else pack_one<T, N, MU, false, ONFLY, C3>(g, f, par, gauge, in_half, face, fi);      \
    }
    HR_PACK(0) HR_PACK(1) HR_PACK(2) HR_PACK(3)
#undef HR_PACK
}

// Boundary kernel: the terms of the hopping sum that crossed a cut, for the output sites on the faces, combined into `out` the way
// the local kernel's epilogue would have: out += c * t (EPI_NONE: c = 1; EPI_AXPY, EPI_CLOVER_AXPY) or out += B(x) t (EPI_CLOVER_INV).
// Output sites with x_mu = L_mu-1 take the face received from the rank at +mu (its "down" face, multiplied here by the local link),
// output sites with x_mu = 0 the "up" face of the rank at -mu.  par = output parity.
//
// ONE launch serves every cut direction: blockIdx.y runs over the (direction, side) faces, one thread per face site.  Edge and corner
// sites lie on the faces of several directions; a site is OWNED by its lowest cut direction — the thread that meets it on a face of a
// higher direction leaves — and the owner adds the terms of all directions the site is on a face of, in increasing direction, with one
// read-modify-write of the output spinor (no two threads touch the same site: deterministic, no atomics).
struct BoundaryJob {
    FaceGeo f[4];
    const void* lo[4];   // face for the sites with x_mu = 0      (the -mu neighbour's up face)
    const void* hi[4];   // face for the sites with x_mu = L_mu-1 (the +mu neighbour's down face)
    int cut[4];
    int slot[8];         // slot[j] = 2*mu + side of the j-th face
    int nslots;
};

// index of site x in the face of direction f.mu (inverse of face_site)
__device__ __forceinline__ int face_index(const FaceGeo& f, const int x[4]) {
    return ((x[f.o[0]] * f.E[1] + x[f.o[1]]) * f.E[2] + x[f.o[2]]) >> 1;
}

// t += the term of direction MU that crossed the cut, for output site (row, h) = x on side `up` of that direction
template <typename T, int N, int MU, bool ONFLY, bool C3>
__device__ __forceinline__ void boundary_term(cplx<T>* t, const Geo& g, const BoundaryJob& job, int par, const HopArgs& a, int up, const int x[4],
                                              int row, int h) {
    const FaceGeo& f = job.f[MU];
    const int fi = face_index(f, x);
    cplx<T> h0[N], h1[N];
    face_load<T, N>(up ? job.hi[MU] : job.lo[MU], f.nface, fi, h0, h1);
    if (up) {
        typename std::conditional<C3, LinkC3<T>, Link<T, N>>::type u;    // C3: complex 3 x 3 links (HR_REP_SU3)
        load_link_rep<T, LD_STREAM, ONFLY>(u, a.gauge, g, par, MU, row, h);
        hop_apply<T, N, MU, true>(t, h0, h1, u);
    } else {
        hop_rebuild<T, N, MU, false>(t, h0, h1);
    }
}

template <typename T, int N, int EPI, bool ONFLY, bool C3>
__global__ void __launch_bounds__(128) halo_boundary_kernel(Geo g, BoundaryJob job, int par, HopArgs a) {
    constexpr int NC = 4 * N;
    typedef SiteIO<T, NC> IO;
    const int fidx = job.slot[blockIdx.y];
    const int mu = fidx >> 1, side = fidx & 1;
    const int fi = blockIdx.x * blockDim.x + threadIdx.x;
    if (fi >= job.f[mu].nface) return;
    const int L[4] = {g.L0, g.L1, g.L2, 2 * g.L3h};
    int x[4];
    face_site(job.f[mu], fi, side ? L[mu] - 1 : 0, par, x);
    for (int nu = 0; nu < mu; ++nu)
        if (job.cut[nu] && (x[nu] == 0 || x[nu] == L[nu] - 1)) return;      // owned by a lower direction
    const int row = (x[0] * g.L1 + x[1]) * g.L2 + x[2], h = x[3] >> 1;
    const size_t first = (size_t)row * (IO::NCH * g.L3h) + h;
    cplx<T> o[NC], t[NC];
    IO::template load<LD_KEEP>(o, a.out, first, g.L3h);
    const T cc = EPI == EPI_NONE ? (T)1 : (T)a.c;
    bool any = false;
#pragma unroll
    for (int c = 0; c < NC; ++c) t[c] = mk<T>((T)0, (T)0);
#define HR_BND(MU)                                                                                         \
    if (MU >= mu && job.cut[MU] && (x[MU] == 0 || x[MU] == L[MU] - 1)) {                                   \
        boundary_term<T, N, MU, ONFLY, C3>(t, g, job, par, a, x[MU] == 0 ? 0 : 1, x, row, h);              \
        any = true;                                                                                        \
        if (EPI != EPI_CLOVER_INV) {   /* one direction at a time, like consecutive passes would */         \
            _Pragma("unroll") for (int c = 0; c < NC; ++c) {                                               \
                o[c].re = fma(cc, t[c].re, o[c].re); o[c].im = fma(cc, t[c].im, o[c].im);                  \
                t[c] = mk<T>((T)0, (T)0);                                                                  \
            }                                                                                              \
        }                                                                                                  \
    }
    HR_BND(0) HR_BND(1) HR_BND(2) HR_BND(3)
#undef HR_BND
    if (!any) return;
    if (EPI == EPI_CLOVER_INV) {      // B(x) is linear: one block product for the sum of the crossing terms
        T blk[CloverSize<N>::reals];
        cplx<T> y[NC];
        load_clover<T, N>(blk, a.clover, g, par, row, h);
        clover_matvec<T, N>(y, blk, t);
#pragma unroll
        for (int c = 0; c < NC; ++c) o[c] = o[c] + y[c];
    }
    IO::store(a.out, first, g.L3h, o);
}

template <typename T, int N, bool ONFLY, bool C3 = false>
static int pack_faces(const hr_geom* hg, const int* split, int par, const void* gauge, const void* in_half, void* const* face_out, cudaStream_t st) {
    const Geo g = make_geo(hg);
    PackJob job;
    job.nslots = 0;
    int maxface = 0;
    for (int mu = 0; mu < 4; ++mu) {
        job.f[mu] = make_face(hg, mu);
        job.face[2 * mu] = job.face[2 * mu + 1] = nullptr;
        if (!split[mu]) continue;
        for (int up = 0; up < 2; ++up) {
            job.face[2 * mu + up] = face_out[2 * mu + up];
            job.slot[job.nslots++] = 2 * mu + up;
        }
        if (job.f[mu].nface > maxface) maxface = job.f[mu].nface;
    }
    if (job.nslots == 0) return HR_OK;
    halo_pack_kernel<T, N, ONFLY, C3><<<dim3((maxface + 127) / 128, job.nslots), 128, 0, st>>>(g, job, par, gauge, in_half);
    count_launch();
    return check_launch("halo_pack_kernel");
}

template <typename T, int N, bool ONFLY, bool C3 = false>
static int add_boundary(const hr_geom* hg, const int* split, const HopArgs& a, int epi, const void* const* face_in, cudaStream_t st) {
    const Geo g = make_geo(hg);
    BoundaryJob job;
    job.nslots = 0;
    int maxface = 0;
    for (int mu = 0; mu < 4; ++mu) {
        job.f[mu] = make_face(hg, mu);
        job.cut[mu] = split[mu] ? 1 : 0;
        job.lo[mu] = job.hi[mu] = nullptr;
        if (!split[mu]) continue;
        // output sites at x_mu = 0 take the -mu neighbour's up face (index 2mu+1); those at x_mu = L-1 the +mu neighbour's down face
        job.lo[mu] = face_in[2 * mu + 1];
        job.hi[mu] = face_in[2 * mu];
        job.slot[job.nslots++] = 2 * mu;
        job.slot[job.nslots++] = 2 * mu + 1;
        if (job.f[mu].nface > maxface) maxface = job.f[mu].nface;
    }
    if (job.nslots == 0) return HR_OK;
    const dim3 grid((maxface + 127) / 128, job.nslots);
    switch (epi) {
        case EPI_NONE: halo_boundary_kernel<T, N, EPI_NONE, ONFLY, C3><<<grid, 128, 0, st>>>(g, job, a.parity, a); break;
        case EPI_AXPY: halo_boundary_kernel<T, N, EPI_AXPY, ONFLY, C3><<<grid, 128, 0, st>>>(g, job, a.parity, a); break;
        case EPI_CLOVER_INV: halo_boundary_kernel<T, N, EPI_CLOVER_INV, ONFLY, C3><<<grid, 128, 0, st>>>(g, job, a.parity, a); break;
        case EPI_CLOVER_AXPY: halo_boundary_kernel<T, N, EPI_CLOVER_AXPY, ONFLY, C3><<<grid, 128, 0, st>>>(g, job, a.parity, a); break;
        default: set_error("unknown epilogue %d", epi); return HR_EINVAL;
    }
    count_launch();
    return check_launch("halo_boundary_kernel");
}

#define HR_DISPATCH_REP(FN, ...)                                                                      \
    if (hg->rep == HR_REP_SU3) {                                                                      \
        if (hg->link_storage == HR_LINKS_COMPRESSED) {                                                \
            if (hg->prec == HR_PREC_F64) return FN<double, 3, true, true>(__VA_ARGS__);               \
            return FN<float, 3, true, true>(__VA_ARGS__);                                             \
        }                                                                                             \
        if (hg->prec == HR_PREC_F64) return FN<double, 3, false, true>(__VA_ARGS__);                  \
        return FN<float, 3, false, true>(__VA_ARGS__);                                                \
    }                                                                                                 \
    if (hg->rep == HR_REP_FUND) {                                                                     \
        if (hg->prec == HR_PREC_F64) return FN<double, 2, false>(__VA_ARGS__);                        \
        return FN<float, 2, false>(__VA_ARGS__);                                                      \
    }                                                                                                 \
    if (hg->link_storage == HR_LINKS_ONTHEFLY) {                                                      \
        if (hg->prec == HR_PREC_F64) return FN<double, 3, true>(__VA_ARGS__);                         \
        return FN<float, 3, true>(__VA_ARGS__);                                                       \
    }                                                                                                 \
    if (hg->prec == HR_PREC_F64) return FN<double, 3, false>(__VA_ARGS__);                            \
    return FN<float, 3, false>(__VA_ARGS__);

int run_halo_pack(const hr_geom* hg, const int* split, int par, const void* gauge, const void* in_half, void* const* face_out, cudaStream_t st) {
    HR_DISPATCH_REP(pack_faces, hg, split, par, gauge, in_half, face_out, st)
}

int run_halo_boundary(const hr_geom* hg, const int* split, const HopArgs& a, int epi, const void* const* face_in, cudaStream_t st) {
    HR_DISPATCH_REP(add_boundary, hg, split, a, epi, face_in, st)
}

size_t halo_face_bytes(const hr_geom* hg, int mu) {
    const FaceGeo f = make_face(hg, mu);
    return (size_t)f.nface * 2 * ncolour(hg->rep) * 2 * real_bytes(hg->prec);
}

}  // namespace hr
