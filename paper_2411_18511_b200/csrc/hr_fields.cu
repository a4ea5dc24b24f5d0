// hr_fields.cu — layout permutations (pack/unpack), the representation kernel R1 and the clover
// kernels C1/C2/C3 of libhr_dslash.
#include "hr_common.cuh"

namespace hr {

// lexicographic site -> (parity, row, h)
struct SiteRef {
    int par, row, h;
};
__device__ __forceinline__ SiteRef site_of_lex(const Geo& g, int lex) {
    const int L3 = 2 * g.L3h;
    const int x3 = lex % L3;
    const int row = lex / L3;
    const int x0 = row / g.s0, rem = row - x0 * g.s0;
    const int x1 = rem / g.s1, x2 = rem - x1 * g.s1;
    SiteRef s;
    s.par = (x0 + x1 + x2 + x3) & 1;
    s.row = row;
    s.h = x3 >> 1;
    return s;
}
// coordinates (any integers, wrapped periodically) -> (parity, row, h)
__device__ __forceinline__ SiteRef site_of_coords(const Geo& g, int x0, int x1, int x2, int x3) {
    const int L3 = 2 * g.L3h;
    x0 = (x0 + g.L0) % g.L0; x1 = (x1 + g.L1) % g.L1; x2 = (x2 + g.L2) % g.L2; x3 = (x3 + L3) % L3;
    SiteRef s;
    s.par = (x0 + x1 + x2 + x3) & 1;
    s.row = (x0 * g.L1 + x1) * g.L2 + x2;
    s.h = x3 >> 1;
    return s;
}

// ------------------------------------------------------------------ pack / unpack: pure permutations
// Generic 16-byte-chunk permutation.  Canonical: [lex][item 0..NI-1][SRC chunks]; of each item the first
// NCH chunks are kept (NCH == SRC except for compressed links, where SRC = 2*NCH).  Device:
//   [par][item][row][NCH][h].   Spinor and clover use NI = 1; compressed links NI = 4 (mu).
template <bool PACK>
__global__ void permute_chunks_kernel(Geo g, int NI, int NCH, int SRC, const uint4* __restrict__ src, uint4* __restrict__ dst) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = 2LL * g.Vh * NI * NCH;
    if (t >= total) return;
    const int c = (int)(t % NCH);
    const int item = (int)((t / NCH) % NI);
    const int lex = (int)(t / ((long long)NCH * NI));
    const SiteRef s = site_of_lex(g, lex);
    const size_t ic = ((size_t)lex * NI + item) * SRC + c;
    const size_t id = (((size_t)(s.par * NI + item) * g.R + s.row) * NCH + c) * g.L3h + s.h;
    if (PACK) dst[id] = src[ic];
    else dst[ic] = src[id];
}

// second row of an unpacked fundamental link: (-conj(beta), conj(alpha))
template <typename T>
__global__ void rebuild_second_row_kernel(long long nlinks, T* canon) {
    const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= nlinks) return;
    T* u = canon + k * 8;
    u[4] = -u[2]; u[5] = u[3];
    u[6] = u[0]; u[7] = -u[1];
}

// adjoint links: canonical [lex][mu][9] reals <-> device [par][mu][row][9][h]; the same permutation with T = double2 / float2
// moves the 9 complex entries of an HR_REP_SU3 link
// NK: entries of a link kept on the device (9, or 6 = the first two rows of an HR_REP_SU3 link with HR_LINKS_COMPRESSED); the
// canonical array always has 9 per link
template <typename T, bool PACK, int NK>
__global__ void permute_adj_kernel(Geo g, const T* __restrict__ src, T* __restrict__ dst) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = 2LL * g.Vh * 4 * NK;
    if (t >= total) return;
    const int k = (int)(t % NK);
    const int mu = (int)((t / NK) % 4);
    const int lex = (int)(t / (4 * NK));
    const SiteRef s = site_of_lex(g, lex);
    const size_t id = (((size_t)(s.par * 4 + mu) * g.R + s.row) * NK + k) * g.L3h + s.h;
    const size_t ic = ((size_t)lex * 4 + mu) * 9 + k;
    if (PACK) dst[id] = src[ic];
    else dst[ic] = src[id];
}

// third row of every canonical complex 3 x 3 link from the first two: row2 = conj(row0 x row1) (unpack of two-row storage)
template <typename T>
__global__ void rebuild_third_row_kernel(long long nlinks, T* __restrict__ canon) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nlinks) return;
    cplx<T>* m = reinterpret_cast<cplx<T>*>(canon) + t * 9;
    m[6] = conj(m[1] * m[5] - m[2] * m[4]);
    m[7] = conj(m[2] * m[3] - m[0] * m[5]);
    m[8] = conj(m[0] * m[4] - m[1] * m[3]);
}

static inline unsigned blocks_for(long long n, int bs) { return (unsigned)((n + bs - 1) / bs); }

int permute_chunks(bool pack, const Geo& g, int NI, int NCH, int SRC, const void* src, void* dst, cudaStream_t st) {
    const long long total = 2LL * g.Vh * NI * NCH;
    if (pack)
        permute_chunks_kernel<true><<<blocks_for(total, 256), 256, 0, st>>>(g, NI, NCH, SRC, (const uint4*)src, (uint4*)dst);
    else
        permute_chunks_kernel<false><<<blocks_for(total, 256), 256, 0, st>>>(g, NI, NCH, SRC, (const uint4*)src, (uint4*)dst);
    count_launch();
    return check_launch("permute_chunks_kernel");
}

int rebuild_second_row(const Geo& g, int prec, void* canon, cudaStream_t st) {
    const long long nl = 8LL * g.Vh;
    if (prec == HR_PREC_F64) rebuild_second_row_kernel<double><<<blocks_for(nl, 256), 256, 0, st>>>(nl, (double*)canon);
    else rebuild_second_row_kernel<float><<<blocks_for(nl, 256), 256, 0, st>>>(nl, (float*)canon);
    count_launch();
    return check_launch("rebuild_second_row_kernel");
}

template <typename T, int NK>
static void permute_adj_launch(bool pack, const Geo& g, const void* src, void* dst, cudaStream_t st) {
    const unsigned nb = blocks_for(2LL * g.Vh * 4 * NK, 256);
    if (pack) permute_adj_kernel<T, true, NK><<<nb, 256, 0, st>>>(g, (const T*)src, (T*)dst);
    else permute_adj_kernel<T, false, NK><<<nb, 256, 0, st>>>(g, (const T*)src, (T*)dst);
}

// complex_entries: HR_REP_SU3 links; two_rows: only their first two rows live on the device (unpack rebuilds the third)
int permute_adj(bool pack, const Geo& g, int prec, const void* src, void* dst, cudaStream_t st, bool complex_entries, bool two_rows) {
    if (complex_entries && two_rows) {
        if (prec == HR_PREC_F64) permute_adj_launch<double2, 6>(pack, g, src, dst, st);
        else permute_adj_launch<float2, 6>(pack, g, src, dst, st);
        count_launch();
        if (!pack) {
            const long long nl = 8LL * g.Vh;
            if (prec == HR_PREC_F64) rebuild_third_row_kernel<double><<<blocks_for(nl, 256), 256, 0, st>>>(nl, (double*)dst);
            else rebuild_third_row_kernel<float><<<blocks_for(nl, 256), 256, 0, st>>>(nl, (float*)dst);
            count_launch();
        }
        return check_launch("permute_adj_kernel");
    }
    if (complex_entries) {
        if (prec == HR_PREC_F64) permute_adj_launch<double2, 9>(pack, g, src, dst, st);
        else permute_adj_launch<float2, 9>(pack, g, src, dst, st);
    } else if (prec == HR_PREC_F64) {
        permute_adj_launch<double, 9>(pack, g, src, dst, st);
    } else {
        permute_adj_launch<float, 9>(pack, g, src, dst, st);
    }
    count_launch();
    return check_launch("permute_adj_kernel");
}

// ------------------------------------------------------------------ R1: adjoint links from fundamental ones
// R^{ab} = 1/2 tr(sigma_a U sigma_b U^dag)  (BASELINE.json north_star).  With U = a0 + i a.sigma
// (alpha = a0 + i a3, beta = a2 + i a1) the trace evaluates to
//     R_ab = (a0^2 - |a|^2) delta_ab + 2 a_a a_b + 2 a0 eps_abc a_c .
// One thread per link; fundamental and adjoint gauge fields share the [par][mu][row][..][h] indexing.
template <typename T>
__global__ void represent_kernel(Geo g, const void* __restrict__ ufund, T* __restrict__ uadj) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = 8LL * g.Vh;  // 2 parities x 4 mu x Vh
    if (t >= total) return;
    const int h = (int)(t % g.L3h);
    const long long pr = t / g.L3h;  // (par*4+mu)*R + row
    cplx<T> ab[2];
    constexpr int LCH = SiteIO<T, 2>::NCH;
    SiteIO<T, 2>::template load<LD_STREAM>(ab, ufund, (size_t)pr * (LCH * g.L3h) + h, g.L3h);
    const T a0 = ab[0].re, a3 = ab[0].im, a2 = ab[1].re, a1 = ab[1].im;
    const T d = a0 * a0 - (a1 * a1 + a2 * a2 + a3 * a3);
    T r[9];
    r[0] = d + 2 * a1 * a1;           r[1] = 2 * (a1 * a2 + a0 * a3);   r[2] = 2 * (a1 * a3 - a0 * a2);
    r[3] = 2 * (a2 * a1 - a0 * a3);   r[4] = d + 2 * a2 * a2;           r[5] = 2 * (a2 * a3 + a0 * a1);
    r[6] = 2 * (a3 * a1 + a0 * a2);   r[7] = 2 * (a3 * a2 - a0 * a1);   r[8] = d + 2 * a3 * a3;
    T* o = uadj + (size_t)pr * (9 * g.L3h) + h;
#pragma unroll
    for (int k = 0; k < 9; ++k) __stcs(o + (size_t)k * g.L3h, r[k]);
}

int run_represent(const Geo& g, int prec, const void* ufund, void* uadj, cudaStream_t st) {
    const long long total = 8LL * g.Vh;
    if (prec == HR_PREC_F64) represent_kernel<double><<<blocks_for(total, 256), 256, 0, st>>>(g, ufund, (double*)uadj);
    else represent_kernel<float><<<blocks_for(total, 256), 256, 0, st>>>(g, ufund, (float*)uadj);
    count_launch();
    return check_launch("represent_kernel");
}

// R1 for complex 3 x 3 links: the two-index antisymmetric representation.  U acts on
// antisymmetric matrices as e -> U e U^T; in the basis e^a = (E_ij - E_ji)/sqrt(2), a = (i<j) = (0,1), (0,2), (1,2), the matrix of
// that action is the second compound of U — its 2 x 2 minors:
//     R_ab = U_ik U_jl - U_il U_jk     with (i,j) the pair a (rows) and (k,l) the pair b (columns).
// For N = 3 it is again special unitary, so it is stored like the fundamental field (all three rows, or the first two) and every
// HR_REP_SU3 operator runs on it unchanged.  One thread per link.
template <typename T, bool TWOROWS>
__global__ void represent_antisym_su3_kernel(Geo g, const void* __restrict__ ufund, void* __restrict__ urep) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long total = 8LL * g.Vh;  // 2 parities x 4 mu x Vh
    if (t >= total) return;
    const int h = (int)(t % g.L3h);
    const long long pr = t / g.L3h;      // (par*4+mu)*R + row
    const int pm = (int)(pr / g.R), row = (int)(pr - (long long)pm * g.R);
    LinkC3<T> u;
    load_link_rep<T, LD_STREAM, TWOROWS>(u, ufund, g, pm >> 2, pm & 3, row, h);
    constexpr int NK = TWOROWS ? 6 : 9;
    typedef typename std::conditional<sizeof(T) == 8, double2, float2>::type pair_t;
    pair_t* o = reinterpret_cast<pair_t*>(urep) + (size_t)pr * (NK * g.L3h) + h;
    const int pi[3] = {0, 0, 1}, pj[3] = {1, 2, 2};
#pragma unroll
    for (int a = 0; a < (TWOROWS ? 2 : 3); ++a) {
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const cplx<T> m = u.m[3 * pi[a] + pi[b]] * u.m[3 * pj[a] + pj[b]] - u.m[3 * pi[a] + pj[b]] * u.m[3 * pj[a] + pi[b]];
            pair_t v;
            v.x = m.re;
            v.y = m.im;
            __stcs(o + (size_t)(3 * a + b) * g.L3h, v);
        }
    }
}

int run_represent_antisym_su3(const Geo& g, int prec, bool tworows, const void* ufund, void* urep, cudaStream_t st) {
    const long long total = 8LL * g.Vh;
    const unsigned nb = blocks_for(total, 256);
    if (prec == HR_PREC_F64) {
        if (tworows) represent_antisym_su3_kernel<double, true><<<nb, 256, 0, st>>>(g, ufund, urep);
        else represent_antisym_su3_kernel<double, false><<<nb, 256, 0, st>>>(g, ufund, urep);
    } else {
        if (tworows) represent_antisym_su3_kernel<float, true><<<nb, 256, 0, st>>>(g, ufund, urep);
        else represent_antisym_su3_kernel<float, false><<<nb, 256, 0, st>>>(g, ufund, urep);
    }
    count_launch();
    return check_launch("represent_antisym_su3_kernel");
}

// ------------------------------------------------------------------ C1: clover blocks and their inverses
// SU(2) matrices as quaternions q = (q0, q1, q2, q3) <-> q0 + i (q1 s1 + q2 s2 + q3 s3):
//   product (a0,a)(b0,b) = (a0 b0 - a.b, a0 b + b0 a - a x b),  dagger = (a0, -a).
struct Quat {
    double q0, q1, q2, q3;
};
__device__ __forceinline__ Quat qmul(const Quat& a, const Quat& b) {
    Quat c;
    c.q0 = a.q0 * b.q0 - (a.q1 * b.q1 + a.q2 * b.q2 + a.q3 * b.q3);
    c.q1 = a.q0 * b.q1 + b.q0 * a.q1 - (a.q2 * b.q3 - a.q3 * b.q2);
    c.q2 = a.q0 * b.q2 + b.q0 * a.q2 - (a.q3 * b.q1 - a.q1 * b.q3);
    c.q3 = a.q0 * b.q3 + b.q0 * a.q3 - (a.q1 * b.q2 - a.q2 * b.q1);
    return c;
}
__device__ __forceinline__ Quat qdag(const Quat& a) {
    Quat c;
    c.q0 = a.q0; c.q1 = -a.q1; c.q2 = -a.q2; c.q3 = -a.q3;
    return c;
}
template <typename T>
__device__ __forceinline__ Quat link_quat(const void* ufund, const Geo& g, int x0, int x1, int x2, int x3, int mu) {
    const SiteRef s = site_of_coords(g, x0, x1, x2, x3);
    Link<T, 2> u;
    load_link<T, LD_KEEP>(u, ufund, g, s.par, mu, s.row, s.h);
    Quat q;
    q.q0 = (double)u.a.re; q.q3 = (double)u.a.im; q.q2 = (double)u.b.re; q.q1 = (double)u.b.im;
    return q;
}

// vector part of Q_mu,nu(x) = sum of the four plaquette leaves in the mu-nu plane that start and end at x,
// all traversed in the mu -> nu sense:
//   P1 = U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
//   P2 = U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu)
//   P3 = U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu)
//   P4 = U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag
// F^_mu,nu = (Q - Q^dag)/8 = (i/4) vec(Q).sigma, so  i F^_mu,nu = -(1/4) vec(Q).sigma.
template <typename T>
__device__ void clover_leaves(double* v, const void* ufund, const Geo& g, const int* x, int mu, int nu, double* w = nullptr) {
    int e[4] = {0, 0, 0, 0}, f[4] = {0, 0, 0, 0};
    e[mu] = 1;
    f[nu] = 1;
#define HR_U(DM, DN, DIR) link_quat<T>(ufund, g, x[0] + (DM) * e[0] + (DN) * f[0], x[1] + (DM) * e[1] + (DN) * f[1], \
                                       x[2] + (DM) * e[2] + (DN) * f[2], x[3] + (DM) * e[3] + (DN) * f[3], DIR)
    Quat p1 = qmul(qmul(HR_U(0, 0, mu), HR_U(1, 0, nu)), qmul(qdag(HR_U(0, 1, mu)), qdag(HR_U(0, 0, nu))));
    Quat p2 = qmul(qmul(HR_U(0, 0, nu), qdag(HR_U(-1, 1, mu))), qmul(qdag(HR_U(-1, 0, nu)), HR_U(-1, 0, mu)));
    Quat p3 = qmul(qmul(qdag(HR_U(-1, 0, mu)), qdag(HR_U(-1, -1, nu))), qmul(HR_U(-1, -1, mu), HR_U(0, -1, nu)));
    Quat p4 = qmul(qmul(qdag(HR_U(0, -1, nu)), HR_U(0, -1, mu)), qmul(HR_U(1, -1, nu), qdag(HR_U(0, 0, mu))));
#undef HR_U
    v[0] = p1.q1 + p2.q1 + p3.q1 + p4.q1;
    v[1] = p1.q2 + p2.q2 + p3.q2 + p4.q2;
    v[2] = p1.q3 + p2.q3 + p3.q3 + p4.q3;
    if (w) {   // adjoint representation: R(P) - R(P)^T = 4 q0 eps_abc q_c per leaf, so F^adj_ab = (1/2) eps_abc w_c
        w[0] = p1.q0 * p1.q1 + p2.q0 * p2.q1 + p3.q0 * p3.q1 + p4.q0 * p4.q1;
        w[1] = p1.q0 * p1.q2 + p2.q0 * p2.q2 + p3.q0 * p3.q2 + p4.q0 * p4.q2;
        w[2] = p1.q0 * p1.q3 + p2.q0 * p2.q3 + p3.q0 * p3.q3 + p4.q0 * p4.q3;
    }
}

struct dcplx {
    double re, im;
};
__device__ __forceinline__ dcplx dmul(dcplx a, dcplx b) { dcplx r; r.re = a.re * b.re - a.im * b.im; r.im = a.re * b.im + a.im * b.re; return r; }
__device__ __forceinline__ dcplx dsub(dcplx a, dcplx b) { dcplx r; r.re = a.re - b.re; r.im = a.im - b.im; return r; }

__device__ __forceinline__ dcplx dadd(dcplx a, dcplx b) { dcplx r; r.re = a.re + b.re; r.im = a.im + b.im; return r; }

// ---- small dense helpers for D x D complex matrices (D = 4: fundamental chirality blocks, D = 6: adjoint ones).
// Setup-time code (once per gauge update): clarity over speed, double precision throughout.
template <int D>
__device__ void matmul_d(dcplx (*C)[D], const dcplx (*A)[D], const dcplx (*B)[D]) {
    for (int i = 0; i < D; ++i)
        for (int j = 0; j < D; ++j) {
            dcplx a = {0.0, 0.0};
            for (int k = 0; k < D; ++k) a = dadd(a, dmul(A[i][k], B[k][j]));
            C[i][j] = a;
        }
}
// in-place inverse by Gauss-Jordan elimination with partial pivoting (row exchanges on [A | 1]).  The clover blocks
// are positive definite for the parameters of interest (eigenvalues (4+m0) +- O(csw |F|)), where no exchange happens;
// pivoting keeps the result finite and accurate for indefinite blocks too (small 4+m0, large csw, rough links).  An
// exactly singular block yields non-finite entries, which hr_clover_count_nonfinite reports.
template <int D>
__device__ void invert_d(dcplx (*A)[D]) {
    dcplx B[D][D];
    for (int i = 0; i < D; ++i)
        for (int j = 0; j < D; ++j) { B[i][j].re = (i == j) ? 1.0 : 0.0; B[i][j].im = 0.0; }
    for (int k = 0; k < D; ++k) {
        int r = k;
        double best = A[k][k].re * A[k][k].re + A[k][k].im * A[k][k].im;
        for (int i = k + 1; i < D; ++i) {
            const double n2 = A[i][k].re * A[i][k].re + A[i][k].im * A[i][k].im;
            if (n2 > best) { best = n2; r = i; }
        }
        if (r != k)
            for (int j = 0; j < D; ++j) {
                const dcplx ta = A[k][j]; A[k][j] = A[r][j]; A[r][j] = ta;
                const dcplx tb = B[k][j]; B[k][j] = B[r][j]; B[r][j] = tb;
            }
        dcplx inv;
        inv.re = A[k][k].re / best;
        inv.im = -A[k][k].im / best;
        for (int j = 0; j < D; ++j) { A[k][j] = dmul(A[k][j], inv); B[k][j] = dmul(B[k][j], inv); }
        for (int i = 0; i < D; ++i) {
            if (i == k) continue;
            const dcplx f = A[i][k];
            for (int j = 0; j < D; ++j) { A[i][j] = dsub(A[i][j], dmul(f, A[k][j])); B[i][j] = dsub(B[i][j], dmul(f, B[k][j])); }
        }
    }
    for (int i = 0; i < D; ++i)
        for (int j = 0; j < D; ++j) A[i][j] = B[i][j];
}
// E = exp(X): scaling and squaring with an order-16 Taylor polynomial (|X / 2^s|_inf <= 1/2, truncation
// < 0.5^17 / 17! ~ 2e-20)
template <int D>
__device__ void expm_d(dcplx (*E)[D], const dcplx (*X)[D]) {
    double nrm = 0.0;
    for (int i = 0; i < D; ++i) {
        double r = 0.0;
        for (int j = 0; j < D; ++j) r += fabs(X[i][j].re) + fabs(X[i][j].im);
        nrm = fmax(nrm, r);
    }
    int s = 0;
    double scale = 1.0;
    while (nrm * scale > 0.5 && s < 60) { scale *= 0.5; ++s; }
    dcplx Y[D][D], P[D][D], Tm[D][D];
    for (int i = 0; i < D; ++i)
        for (int j = 0; j < D; ++j) {
            Y[i][j].re = X[i][j].re * scale; Y[i][j].im = X[i][j].im * scale;
            P[i][j] = Y[i][j];                                   // current term Y^k / k!
            E[i][j].re = (i == j ? 1.0 : 0.0) + Y[i][j].re; E[i][j].im = Y[i][j].im;
        }
    for (int k = 2; k <= 16; ++k) {
        matmul_d<D>(Tm, P, Y);
        for (int i = 0; i < D; ++i)
            for (int j = 0; j < D; ++j) {
                P[i][j].re = Tm[i][j].re / k; P[i][j].im = Tm[i][j].im / k;
                E[i][j] = dadd(E[i][j], P[i][j]);
            }
    }
    for (int q = 0; q < s; ++q) {
        matmul_d<D>(Tm, E, E);
        for (int i = 0; i < D; ++i)
            for (int j = 0; j < D; ++j) E[i][j] = Tm[i][j];
    }
}
// hermitian D x D -> D*D reals (diagonal, then the strictly-lower entries column by column), hermitian part taken
template <typename T, int D>
__device__ void herm_to_reals_d(T* out, dcplx (*A)[D]) {
    for (int i = 0; i < D; ++i) out[i] = (T)A[i][i].re;
    int k = D;
    for (int j = 0; j < D; ++j)
        for (int i = j + 1; i < D; ++i) {
            out[k++] = (T)(0.5 * (A[i][j].re + A[j][i].re));
            out[k++] = (T)(0.5 * (A[i][j].im - A[j][i].im));
        }
}

// chirality blocks (pinned against the dense 8x8 form by tests/test_oracle_pins.py::test_O6_block_formula):
//   A+- = (4+m0) + (csw/2) [ tau1 (x) i(+-F01 - F23) + tau2 (x) i(+-F02 + F13) + tau3 (x) i(+-F03 - F12) ],
// tau_k on the spin index within the chirality, i F on colour; block index = spin*2 + colour.
template <typename T>
__global__ void clover_build_kernel(Geo g, double diag, double csw, int expo, const void* __restrict__ ufund, void* fwd, void* inv) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 2 * g.Vh) return;
    const int par = t / g.Vh, cb = t - par * g.Vh;
    const int row = cb / g.L3h, h = cb - row * g.L3h;
    int x[4];
    x[0] = row / g.s0;
    const int rem = row - x[0] * g.s0;
    x[1] = rem / g.s1;
    x[2] = rem - x[1] * g.s1;
    x[3] = 2 * h + ((x[0] + x[1] + x[2] + par) & 1);

    double a01[3], a02[3], a03[3], a12[3], a13[3], a23[3];
    clover_leaves<T>(a01, ufund, g, x, 0, 1);
    clover_leaves<T>(a02, ufund, g, x, 0, 2);
    clover_leaves<T>(a03, ufund, g, x, 0, 3);
    clover_leaves<T>(a12, ufund, g, x, 1, 2);
    clover_leaves<T>(a13, ufund, g, x, 1, 3);
    clover_leaves<T>(a23, ufund, g, x, 2, 3);

    // Pauli matrices as [k][row][col]
    const dcplx Z = {0.0, 0.0}, P1 = {1.0, 0.0}, M1 = {-1.0, 0.0}, PI = {0.0, 1.0}, MI = {0.0, -1.0};
    const dcplx pauli[3][2][2] = {{{Z, P1}, {P1, Z}}, {{Z, MI}, {PI, Z}}, {{P1, Z}, {Z, M1}}};

    T reals_f[32], reals_i[32];
    for (int chi = 0; chi < 2; ++chi) {
        const double s = chi == 0 ? 1.0 : -1.0;
        // m[k][j]: i F-combination of tau_{k+1} = sum_j m[k][j] sigma_{j+1}
        double m[3][3];
        for (int j = 0; j < 3; ++j) {
            m[0][j] = -0.25 * (s * a01[j] - a23[j]);
            m[1][j] = -0.25 * (s * a02[j] + a13[j]);
            m[2][j] = -0.25 * (s * a03[j] - a12[j]);
        }
        dcplx A[4][4];
        for (int sp = 0; sp < 2; ++sp)
            for (int c = 0; c < 2; ++c)
                for (int tp = 0; tp < 2; ++tp)
                    for (int d = 0; d < 2; ++d) {
                        dcplx acc = {(sp == tp && c == d) ? diag : 0.0, 0.0};
                        for (int k = 0; k < 3; ++k) {
                            dcplx X = {0.0, 0.0};
                            for (int j = 0; j < 3; ++j) { X.re += m[k][j] * pauli[j][c][d].re; X.im += m[k][j] * pauli[j][c][d].im; }
                            const dcplx tx = dmul(pauli[k][sp][tp], X);
                            acc.re += 0.5 * csw * tx.re;
                            acc.im += 0.5 * csw * tx.im;
                        }
                        A[sp * 2 + c][tp * 2 + d] = acc;
                    }
        if (expo) {
            // exponential clover (ref [6]): A_exp = diag exp(C/diag), A_exp^-1 = exp(-C/diag)/diag, C = A - diag
            dcplx X[4][4], E[4][4];
            for (int i = 0; i < 4; ++i)
                for (int j = 0; j < 4; ++j) {
                    X[i][j].re = (A[i][j].re - (i == j ? diag : 0.0)) / diag;
                    X[i][j].im = A[i][j].im / diag;
                }
            expm_d<4>(E, X);
            for (int i = 0; i < 4; ++i)
                for (int j = 0; j < 4; ++j) { A[i][j].re = diag * E[i][j].re; A[i][j].im = diag * E[i][j].im; X[i][j].re = -X[i][j].re; X[i][j].im = -X[i][j].im; }
            herm_to_reals_d<T, 4>(reals_f + 16 * chi, A);
            expm_d<4>(E, X);
            for (int i = 0; i < 4; ++i)
                for (int j = 0; j < 4; ++j) { A[i][j].re = E[i][j].re / diag; A[i][j].im = E[i][j].im / diag; }
            herm_to_reals_d<T, 4>(reals_i + 16 * chi, A);
        } else {
            herm_to_reals_d<T, 4>(reals_f + 16 * chi, A);
            invert_d<4>(A);
            herm_to_reals_d<T, 4>(reals_i + 16 * chi, A);
        }
    }
    constexpr int CCH = 32 * sizeof(T) / 16;
    constexpr int PER = 16 / sizeof(T);
    typedef typename Chunk<T>::type chunk_t;
    const size_t first = ((size_t)par * g.R + row) * (CCH * g.L3h) + h;
    for (int c = 0; c < CCH; ++c) {
        if (fwd) reinterpret_cast<chunk_t*>(fwd)[first + (size_t)c * g.L3h] = reals_to_chunk(reals_f + c * PER);
        if (inv) reinterpret_cast<chunk_t*>(inv)[first + (size_t)c * g.L3h] = reals_to_chunk(reals_i + c * PER);
    }
}


// C1 in the adjoint representation (oracle O10): 6 x 6 chirality blocks on (2 spin x 3 colour),
//   A+- = (4+m0) + (csw/2) [ tau1 (x) i(+-F01 - F23) + tau2 (x) i(+-F02 + F13) + tau3 (x) i(+-F03 - F12) ],
// with F^_mu,nu the real antisymmetric 3x3 matrix (Q - Q^T)/8 of the adjoint leaves.  The leaves are multiplied out
// in the fundamental representation (quaternions) and mapped leaf by leaf: R(P) - R(P)^T = 4 q0 eps_abc q_c.
// the two 6x6 blocks (72 reals) and their inverses from the six leaf vectors w[plane][c] (planes 01 02 03 12 13 23); all
// in double, one shared non-inlined routine for both field precisions
__device__ __noinline__ void clover_adj_blocks(double diag, double csw, int expo, const double (*w)[3], double* reals_f, double* reals_i) {
    const dcplx Z = {0.0, 0.0}, P1 = {1.0, 0.0}, M1 = {-1.0, 0.0}, PI = {0.0, 1.0}, MI = {0.0, -1.0};
    const dcplx pauli[3][2][2] = {{{Z, P1}, {P1, Z}}, {{Z, MI}, {PI, Z}}, {{P1, Z}, {Z, M1}}};
    const double eps[3][3][3] = {{{0, 0, 0}, {0, 0, 1}, {0, -1, 0}}, {{0, 0, -1}, {0, 0, 0}, {1, 0, 0}}, {{0, 1, 0}, {-1, 0, 0}, {0, 0, 0}}};
    const double *w01 = w[0], *w02 = w[1], *w03 = w[2], *w12 = w[3], *w13 = w[4], *w23 = w[5];
    for (int chi = 0; chi < 2; ++chi) {
        const double s = chi == 0 ? 1.0 : -1.0;
        double gk[3][3];   // gk[k][e]: F-combination of tau_{k+1} is the antisymmetric matrix eps_cde gk[k][e]
        for (int e = 0; e < 3; ++e) {
            gk[0][e] = 0.5 * (s * w01[e] - w23[e]);
            gk[1][e] = 0.5 * (s * w02[e] + w13[e]);
            gk[2][e] = 0.5 * (s * w03[e] - w12[e]);
        }
        dcplx A[6][6];
        for (int sp = 0; sp < 2; ++sp)
            for (int c = 0; c < 3; ++c)
                for (int tp = 0; tp < 2; ++tp)
                    for (int d = 0; d < 3; ++d) {
                        dcplx acc = {(sp == tp && c == d) ? diag : 0.0, 0.0};
                        for (int k = 0; k < 3; ++k) {
                            double G = 0.0;
                            for (int e = 0; e < 3; ++e) G += eps[c][d][e] * gk[k][e];
                            const dcplx iG = {0.0, G};
                            const dcplx tx = dmul(pauli[k][sp][tp], iG);
                            acc.re += 0.5 * csw * tx.re;
                            acc.im += 0.5 * csw * tx.im;
                        }
                        A[sp * 3 + c][tp * 3 + d] = acc;
                    }
        if (expo) {
            dcplx X[6][6], E[6][6];
            for (int i = 0; i < 6; ++i)
                for (int j = 0; j < 6; ++j) { X[i][j].re = (A[i][j].re - (i == j ? diag : 0.0)) / diag; X[i][j].im = A[i][j].im / diag; }
            expm_d<6>(E, X);
            for (int i = 0; i < 6; ++i)
                for (int j = 0; j < 6; ++j) { A[i][j].re = diag * E[i][j].re; A[i][j].im = diag * E[i][j].im; X[i][j].re = -X[i][j].re; X[i][j].im = -X[i][j].im; }
            herm_to_reals_d<double, 6>(reals_f + 36 * chi, A);
            expm_d<6>(E, X);
            for (int i = 0; i < 6; ++i)
                for (int j = 0; j < 6; ++j) { A[i][j].re = E[i][j].re / diag; A[i][j].im = E[i][j].im / diag; }
            herm_to_reals_d<double, 6>(reals_i + 36 * chi, A);
        } else {
            herm_to_reals_d<double, 6>(reals_f + 36 * chi, A);
            invert_d<6>(A);
            herm_to_reals_d<double, 6>(reals_i + 36 * chi, A);
        }
    }
}

template <typename T>
__global__ void clover_build_adj_kernel(Geo g, double diag, double csw, int expo, const void* __restrict__ ufund, void* fwd, void* inv) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 2 * g.Vh) return;
    const int par = t / g.Vh, cb = t - par * g.Vh;
    const int row = cb / g.L3h, h = cb - row * g.L3h;
    int x[4];
    x[0] = row / g.s0;
    const int rem = row - x[0] * g.s0;
    x[1] = rem / g.s1;
    x[2] = rem - x[1] * g.s1;
    x[3] = 2 * h + ((x[0] + x[1] + x[2] + par) & 1);
    double v[3], w[6][3];
    clover_leaves<T>(v, ufund, g, x, 0, 1, w[0]);
    clover_leaves<T>(v, ufund, g, x, 0, 2, w[1]);
    clover_leaves<T>(v, ufund, g, x, 0, 3, w[2]);
    clover_leaves<T>(v, ufund, g, x, 1, 2, w[3]);
    clover_leaves<T>(v, ufund, g, x, 1, 3, w[4]);
    clover_leaves<T>(v, ufund, g, x, 2, 3, w[5]);
    constexpr int NR = 72;
    double rf[NR], ri[NR];
    clover_adj_blocks(diag, csw, expo, w, rf, ri);
    constexpr int CCH = NR * sizeof(T) / 16;
    constexpr int PER = 16 / sizeof(T);
    typedef typename Chunk<T>::type chunk_t;
    const size_t first = ((size_t)par * g.R + row) * (CCH * g.L3h) + h;
    for (int c = 0; c < CCH; ++c) {
        T ef[PER], ei[PER];
        for (int k = 0; k < PER; ++k) { ef[k] = (T)rf[c * PER + k]; ei[k] = (T)ri[c * PER + k]; }
        if (fwd) reinterpret_cast<chunk_t*>(fwd)[first + (size_t)c * g.L3h] = reals_to_chunk(ef);
        if (inv) reinterpret_cast<chunk_t*>(inv)[first + (size_t)c * g.L3h] = reals_to_chunk(ei);
    }
}

// C1 for complex 3 x 3 links (HR_REP_SU3; oracle O12): the same 6 x 6 chirality blocks on (2 spin x 3 colour),
//   A+- = (4+m0) + (csw/2) [ tau1 (x) i(+-F01 - F23) + tau2 (x) i(+-F02 + F13) + tau3 (x) i(+-F03 - F12) ],
// with F^_mu,nu = (Q - Q^dag)/8 the anti-hermitian part of the four leaves, multiplied out as complex 3 x 3 matrices.
template <typename T, bool TWOROWS>
__device__ __forceinline__ void link_c3(dcplx (*m)[3], const void* gauge, const Geo& g, int x0, int x1, int x2, int x3, int mu, bool dag) {
    const SiteRef s = site_of_coords(g, x0, x1, x2, x3);
    LinkC3<T> u;
    load_link_rep<T, LD_KEEP, TWOROWS>(u, gauge, g, s.par, mu, s.row, s.h);
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) {
            const cplx<T> z = dag ? u.m[3 * b + a] : u.m[3 * a + b];
            m[a][b].re = (double)z.re;
            m[a][b].im = dag ? -(double)z.im : (double)z.im;
        }
}

// F[a][b] = ((Q - Q^dag)/8)[a][b] of the mu-nu plane at x
template <typename T, bool TWOROWS>
__device__ void clover_leaves_c3(dcplx (*F)[3], const void* gauge, const Geo& g, const int* x, int mu, int nu) {
    int e[4] = {0, 0, 0, 0}, f[4] = {0, 0, 0, 0};
    e[mu] = 1;
    f[nu] = 1;
    dcplx Q[3][3], A[3][3], B[3][3], C[3][3];
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) Q[a][b].re = Q[a][b].im = 0.0;
    // the four links of a leaf as (displacement in mu, displacement in nu, direction, dagger), in path order
    const int path[4][4][4] = {
        {{0, 0, 0, 0}, {1, 0, 1, 0}, {0, 1, 0, 1}, {0, 0, 1, 1}},
        {{0, 0, 1, 0}, {-1, 1, 0, 1}, {-1, 0, 1, 1}, {-1, 0, 0, 0}},
        {{-1, 0, 0, 1}, {-1, -1, 1, 1}, {-1, -1, 0, 0}, {0, -1, 1, 0}},
        {{0, -1, 1, 1}, {0, -1, 0, 0}, {1, -1, 1, 0}, {0, 0, 0, 1}}};
    for (int leaf = 0; leaf < 4; ++leaf) {
        for (int k = 0; k < 4; ++k) {
            const int dm = path[leaf][k][0], dn = path[leaf][k][1], dir = path[leaf][k][2] ? nu : mu;
            link_c3<T, TWOROWS>(B, gauge, g, x[0] + dm * e[0] + dn * f[0], x[1] + dm * e[1] + dn * f[1], x[2] + dm * e[2] + dn * f[2],
                                x[3] + dm * e[3] + dn * f[3], dir, path[leaf][k][3] != 0);
            if (k == 0) {
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b) A[a][b] = B[a][b];
            } else {
                matmul_d<3>(C, A, B);
                for (int a = 0; a < 3; ++a)
                    for (int b = 0; b < 3; ++b) A[a][b] = C[a][b];
            }
        }
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) Q[a][b] = dadd(Q[a][b], A[a][b]);
    }
    for (int a = 0; a < 3; ++a)
        for (int b = 0; b < 3; ++b) {
            F[a][b].re = (Q[a][b].re - Q[b][a].re) / 8.0;
            F[a][b].im = (Q[a][b].im + Q[b][a].im) / 8.0;
        }
}

// the two 6 x 6 blocks and their inverses (or the exponential pair) from the six F matrices (planes 01 02 03 12 13 23)
__device__ __noinline__ void clover_c3_blocks(double diag, double csw, int expo, const dcplx (*F)[3][3], double* reals_f, double* reals_i) {
    const dcplx Z = {0.0, 0.0}, P1 = {1.0, 0.0}, M1 = {-1.0, 0.0}, PI = {0.0, 1.0}, MI = {0.0, -1.0};
    const dcplx pauli[3][2][2] = {{{Z, P1}, {P1, Z}}, {{Z, MI}, {PI, Z}}, {{P1, Z}, {Z, M1}}};
    for (int chi = 0; chi < 2; ++chi) {
        const double s = chi == 0 ? 1.0 : -1.0;
        dcplx A[6][6];
        for (int sp = 0; sp < 2; ++sp)
            for (int c = 0; c < 3; ++c)
                for (int tp = 0; tp < 2; ++tp)
                    for (int d = 0; d < 3; ++d) {
                        dcplx acc = {(sp == tp && c == d) ? diag : 0.0, 0.0};
                        for (int k = 0; k < 3; ++k) {
                            // G_k = +-F0k -+ ... : (s F01 - F23), (s F02 + F13), (s F03 - F12)
                            const dcplx a0 = F[k][c][d], a1 = F[k == 0 ? 5 : k == 1 ? 4 : 3][c][d];
                            const double sg = k == 1 ? 1.0 : -1.0;
                            const dcplx G = {s * a0.re + sg * a1.re, s * a0.im + sg * a1.im};
                            const dcplx iG = {-G.im, G.re};
                            const dcplx tx = dmul(pauli[k][sp][tp], iG);
                            acc.re += 0.5 * csw * tx.re;
                            acc.im += 0.5 * csw * tx.im;
                        }
                        A[sp * 3 + c][tp * 3 + d] = acc;
                    }
        if (expo) {
            dcplx X[6][6], E[6][6];
            for (int i = 0; i < 6; ++i)
                for (int j = 0; j < 6; ++j) { X[i][j].re = (A[i][j].re - (i == j ? diag : 0.0)) / diag; X[i][j].im = A[i][j].im / diag; }
            expm_d<6>(E, X);
            for (int i = 0; i < 6; ++i)
                for (int j = 0; j < 6; ++j) { A[i][j].re = diag * E[i][j].re; A[i][j].im = diag * E[i][j].im; X[i][j].re = -X[i][j].re; X[i][j].im = -X[i][j].im; }
            herm_to_reals_d<double, 6>(reals_f + 36 * chi, A);
            expm_d<6>(E, X);
            for (int i = 0; i < 6; ++i)
                for (int j = 0; j < 6; ++j) { A[i][j].re = E[i][j].re / diag; A[i][j].im = E[i][j].im / diag; }
            herm_to_reals_d<double, 6>(reals_i + 36 * chi, A);
        } else {
            herm_to_reals_d<double, 6>(reals_f + 36 * chi, A);
            invert_d<6>(A);
            herm_to_reals_d<double, 6>(reals_i + 36 * chi, A);
        }
    }
}

template <typename T, bool TWOROWS>
__global__ void clover_build_c3_kernel(Geo g, double diag, double csw, int expo, const void* __restrict__ gauge, void* fwd, void* inv) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= 2 * g.Vh) return;
    const int par = t / g.Vh, cb = t - par * g.Vh;
    const int row = cb / g.L3h, h = cb - row * g.L3h;
    int x[4];
    x[0] = row / g.s0;
    const int rem = row - x[0] * g.s0;
    x[1] = rem / g.s1;
    x[2] = rem - x[1] * g.s1;
    x[3] = 2 * h + ((x[0] + x[1] + x[2] + par) & 1);
    dcplx F[6][3][3];
    clover_leaves_c3<T, TWOROWS>(F[0], gauge, g, x, 0, 1);
    clover_leaves_c3<T, TWOROWS>(F[1], gauge, g, x, 0, 2);
    clover_leaves_c3<T, TWOROWS>(F[2], gauge, g, x, 0, 3);
    clover_leaves_c3<T, TWOROWS>(F[3], gauge, g, x, 1, 2);
    clover_leaves_c3<T, TWOROWS>(F[4], gauge, g, x, 1, 3);
    clover_leaves_c3<T, TWOROWS>(F[5], gauge, g, x, 2, 3);
    constexpr int NR = 72;
    double rf[NR], ri[NR];
    clover_c3_blocks(diag, csw, expo, F, rf, ri);
    constexpr int CCH = NR * sizeof(T) / 16;
    constexpr int PER = 16 / sizeof(T);
    typedef typename Chunk<T>::type chunk_t;
    const size_t first = ((size_t)par * g.R + row) * (CCH * g.L3h) + h;
    for (int c = 0; c < CCH; ++c) {
        T ef[PER], ei[PER];
        for (int k = 0; k < PER; ++k) { ef[k] = (T)rf[c * PER + k]; ei[k] = (T)ri[c * PER + k]; }
        if (fwd) reinterpret_cast<chunk_t*>(fwd)[first + (size_t)c * g.L3h] = reals_to_chunk(ef);
        if (inv) reinterpret_cast<chunk_t*>(inv)[first + (size_t)c * g.L3h] = reals_to_chunk(ei);
    }
}

int run_clover_build_c3(const Geo& g, int prec, bool two_rows, double diag, double csw, int expo, const void* gauge, void* fwd, void* inv, cudaStream_t st) {
    const unsigned nb = blocks_for(2LL * g.Vh, 64);
    if (prec == HR_PREC_F64) {
        if (two_rows) clover_build_c3_kernel<double, true><<<nb, 64, 0, st>>>(g, diag, csw, expo, gauge, fwd, inv);
        else clover_build_c3_kernel<double, false><<<nb, 64, 0, st>>>(g, diag, csw, expo, gauge, fwd, inv);
    } else {
        if (two_rows) clover_build_c3_kernel<float, true><<<nb, 64, 0, st>>>(g, diag, csw, expo, gauge, fwd, inv);
        else clover_build_c3_kernel<float, false><<<nb, 64, 0, st>>>(g, diag, csw, expo, gauge, fwd, inv);
    }
    count_launch();
    return check_launch("clover_build_c3_kernel");
}

int run_clover_build_adj(const Geo& g, int prec, double diag, double csw, int expo, const void* ufund, void* fwd, void* inv, cudaStream_t st) {
    const unsigned nb = blocks_for(2LL * g.Vh, 64);
    if (prec == HR_PREC_F64) clover_build_adj_kernel<double><<<nb, 64, 0, st>>>(g, diag, csw, expo, ufund, fwd, inv);
    else clover_build_adj_kernel<float><<<nb, 64, 0, st>>>(g, diag, csw, expo, ufund, fwd, inv);
    count_launch();
    return check_launch("clover_build_adj_kernel");
}

int run_clover_build(const Geo& g, int prec, double diag, double csw, int expo, const void* ufund, void* fwd, void* inv, cudaStream_t st) {
    const unsigned nb = blocks_for(2LL * g.Vh, 128);
    if (prec == HR_PREC_F64) clover_build_kernel<double><<<nb, 128, 0, st>>>(g, diag, csw, expo, ufund, fwd, inv);
    else clover_build_kernel<float><<<nb, 128, 0, st>>>(g, diag, csw, expo, ufund, fwd, inv);
    count_launch();
    return check_launch("clover_build_kernel");
}

// ------------------------------------------------------------------ C2/C3: out(x) = B(x) in(x)
template <typename T, int N>
__global__ void __launch_bounds__(128) clover_apply_kernel(Geo g, int parity, const void* __restrict__ blocks,
                                                           const void* __restrict__ in, void* __restrict__ out) {
    constexpr int NC = 4 * N;
    typedef SiteIO<T, NC> IO;
    const int cb = blockIdx.x * blockDim.x + threadIdx.x;
    if (cb >= g.Vh) return;
    const int p = parity == HR_BOTH ? (int)blockIdx.y : parity;
    const size_t half_bytes = (size_t)g.Vh * IO::NCH * 16;
    const size_t off = parity == HR_BOTH ? (size_t)p * half_bytes : 0;
    const int row = cb / g.L3h, h = cb - row * g.L3h;
    const size_t first = (size_t)row * (IO::NCH * g.L3h) + h;
    T blk[CloverSize<N>::reals];
    cplx<T> x[NC], y[NC];
    load_clover<T, N>(blk, blocks, g, p, row, h);
    IO::template load<LD_STREAM>(x, reinterpret_cast<const char*>(in) + off, first, g.L3h);
    clover_matvec<T, N>(y, blk, x);
    IO::store(reinterpret_cast<char*>(out) + off, first, g.L3h, y);
}

int run_clover_apply(const Geo& g, int rep, int prec, int parity, const void* blocks, const void* in, void* out, cudaStream_t st) {
    dim3 grid(blocks_for(g.Vh, 128), parity == HR_BOTH ? 2 : 1);
    if (rep == HR_REP_FUND) {
        if (prec == HR_PREC_F64) clover_apply_kernel<double, 2><<<grid, 128, 0, st>>>(g, parity, blocks, in, out);
        else clover_apply_kernel<float, 2><<<grid, 128, 0, st>>>(g, parity, blocks, in, out);
    } else {
        if (prec == HR_PREC_F64) clover_apply_kernel<double, 3><<<grid, 128, 0, st>>>(g, parity, blocks, in, out);
        else clover_apply_kernel<float, 3><<<grid, 128, 0, st>>>(g, parity, blocks, in, out);
    }
    count_launch();
    return check_launch("clover_apply_kernel");
}

// ---- number of non-finite reals in a block field (a singular block inverts to inf / nan)
template <typename T>
__global__ void count_nonfinite_kernel(const T* __restrict__ x, size_t n, unsigned long long* count) {
    unsigned long long bad = 0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        if (!isfinite(x[i])) ++bad;
    if (bad) atomicAdd(count, bad);
}

int run_count_nonfinite(int prec, const void* x, size_t bytes, unsigned long long* count_dev, cudaStream_t st) {
    cudaError_t e = cudaMemsetAsync(count_dev, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) { set_error("cudaMemsetAsync: %s", cudaGetErrorString(e)); return HR_ECUDA; }
    const size_t n = bytes / real_bytes(prec);
    const int grid = (int)((n + 255) / 256 < 148 * 8 ? (n + 255) / 256 : 148 * 8);
    if (prec == HR_PREC_F64) count_nonfinite_kernel<double><<<grid, 256, 0, st>>>(reinterpret_cast<const double*>(x), n, count_dev);
    else count_nonfinite_kernel<float><<<grid, 256, 0, st>>>(reinterpret_cast<const float*>(x), n, count_dev);
    count_launch();
    return check_launch("count_nonfinite_kernel");
}

}  // namespace hr
