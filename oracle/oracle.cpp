// oracle/oracle.cpp — CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, double-precision restatement of the operators on the hot path of
// arXiv 2411.18511 (HiRep Wilson-Dirac operator; §2.1, §2.2).
// The paper prints no formula; the definitions are BASELINE.json `north_star` and the
// readings fixed in SURVEY.md §8(c) (O1-O7, A1-A25), each cited where it is used.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may call this.  It shares no code, header, table or constant with the CUDA
// library under paper_2411_18511_b200/csrc and includes nothing from it.
//
// Style: canonical array-of-structs data (A3/A4), dense 4x4 gamma matrices applied as
// matrices (no half-spinor trick), std::complex<double>, explicit (x +- 1) mod L
// neighbours, no blocking, no fusion, no reordering.  Pinned by tests/test_oracle_pins.py
// (P1-P14, P20 for this file; P15-P19 for the numpy routines O8-O11 of oracle/__init__.py).
// Parity unpinned: nothing.
//
// Canonical layouts (A3/A4), V = L0 L1 L2 L3, lex(x) = ((x0 L1 + x1) L2 + x2) L3 + x3:
//   spinor      [lex][spin 0..3][colour 0..N-1][re,im]
//   fund gauge  [lex][mu][row][col][re,im]         (2x2 complex)
//   adj gauge   [lex][mu][a][b]                    (3x3 real)
//   rep-2 gauge [lex][mu][row][col][re,im]         (3x3 complex, e.g. SU(3) fundamental)
//   dense site matrix (clover) [lex][8][8][re,im], row/col index = spin*2 + colour
#include <complex>
#include <cstring>
#include <cmath>
#include <thread>
#include <vector>

typedef std::complex<double> cd;
static const cd I_(0.0, 1.0);

namespace {

struct Lat {
    int L[4];
    long V;
};

Lat make_lat(const int* L) {
    Lat g;
    g.V = 1;
    for (int m = 0; m < 4; ++m) { g.L[m] = L[m]; g.V *= L[m]; }
    return g;
}

void coords(const Lat& g, long s, int x[4]) {
    for (int m = 3; m >= 0; --m) { x[m] = (int)(s % g.L[m]); s /= g.L[m]; }
}

long lex(const Lat& g, const int x[4]) {
    return (((long)x[0] * g.L[1] + x[1]) * g.L[2] + x[2]) * g.L[3] + x[3];
}

// site x + dir * mu_hat, periodic (A5)
long shift(const Lat& g, long s, int mu, int dir) {
    int x[4];
    coords(g, s, x);
    x[mu] = ((x[mu] + dir) % g.L[mu] + g.L[mu]) % g.L[mu];
    return lex(g, x);
}

int parity(const Lat& g, long s) {
    int x[4];
    coords(g, s, x);
    return (x[0] + x[1] + x[2] + x[3]) & 1;
}

// A2: hermitian chiral gamma matrices, gamma5 = g0 g1 g2 g3 = diag(1,1,-1,-1)
void gamma_matrices(cd G[4][4][4]) {
    const cd o(0, 0), p(1, 0), m(-1, 0), i = I_, j = -I_;
    const cd g0[4][4] = {{o, o, m, o}, {o, o, o, m}, {m, o, o, o}, {o, m, o, o}};
    const cd g1[4][4] = {{o, o, o, j}, {o, o, j, o}, {o, i, o, o}, {i, o, o, o}};
    const cd g2[4][4] = {{o, o, o, m}, {o, o, p, o}, {o, p, o, o}, {m, o, o, o}};
    const cd g3[4][4] = {{o, o, j, o}, {o, o, o, i}, {i, o, o, o}, {o, j, o, o}};
    for (int a = 0; a < 4; ++a)
        for (int b = 0; b < 4; ++b) {
            G[0][a][b] = g0[a][b];
            G[1][a][b] = g1[a][b];
            G[2][a][b] = g2[a][b];
            G[3][a][b] = g3[a][b];
        }
}

// link U_mu(x) in the fermion representation as a complex NxN matrix.  rep 0: SU(2) fundamental (2x2 complex);
// rep 1: SU(2) adjoint (3x3 real); rep 2: a complex 3x3 link per direction, e.g. SU(3) fundamental (PAPER.md:13, 21
// "various gauge groups ... numbers of colors of 2 to 5") — O1-O3 are the same formulas, only
// the colour matrix that multiplies the spinor changes.
void link(int rep, const double* U, long x, int mu, cd M[3][3]) {
    if (rep == 0) {
        const cd* u = reinterpret_cast<const cd*>(U) + (x * 4 + mu) * 4;
        for (int r = 0; r < 2; ++r)
            for (int c = 0; c < 2; ++c) M[r][c] = u[r * 2 + c];
    } else if (rep == 2) {
        const cd* u = reinterpret_cast<const cd*>(U) + (x * 4 + mu) * 9;
        for (int r = 0; r < 3; ++r)
            for (int c = 0; c < 3; ++c) M[r][c] = u[r * 3 + c];
    } else {
        const double* u = U + (x * 4 + mu) * 9;
        for (int r = 0; r < 3; ++r)
            for (int c = 0; c < 3; ++c) M[r][c] = cd(u[r * 3 + c], 0.0);
    }
}

// O2 at one site: H psi(x) = sum_mu [(1-g_mu) U_mu(x) psi(x+mu) + (1+g_mu) U_mu(x-mu)^dag psi(x-mu)]
void hop_site(const Lat& g, int rep, const double* U, const cd* psi, long x, cd out[4][3]) {
    const int N = rep == 0 ? 2 : 3;
    cd G[4][4][4];
    gamma_matrices(G);
    for (int s = 0; s < 4; ++s)
        for (int c = 0; c < N; ++c) out[s][c] = 0.0;
    for (int mu = 0; mu < 4; ++mu) {
        cd M[3][3], t[4][3];
        // forward: (1 - gamma_mu) U_mu(x) psi(x + mu)
        long xp = shift(g, x, mu, +1);
        link(rep, U, x, mu, M);
        for (int s = 0; s < 4; ++s)
            for (int c = 0; c < N; ++c) {
                t[s][c] = 0.0;
                for (int d = 0; d < N; ++d) t[s][c] += M[c][d] * psi[(xp * 4 + s) * N + d];
            }
        for (int s = 0; s < 4; ++s)
            for (int sp = 0; sp < 4; ++sp) {
                cd P = (s == sp ? 1.0 : 0.0) - G[mu][s][sp];
                for (int c = 0; c < N; ++c) out[s][c] += P * t[sp][c];
            }
        // backward: (1 + gamma_mu) U_mu(x - mu)^dagger psi(x - mu)
        long xm = shift(g, x, mu, -1);
        link(rep, U, xm, mu, M);
        for (int s = 0; s < 4; ++s)
            for (int c = 0; c < N; ++c) {
                t[s][c] = 0.0;
                for (int d = 0; d < N; ++d) t[s][c] += std::conj(M[d][c]) * psi[(xm * 4 + s) * N + d];
            }
        for (int s = 0; s < 4; ++s)
            for (int sp = 0; sp < 4; ++sp) {
                cd P = (s == sp ? 1.0 : 0.0) + G[mu][s][sp];
                for (int c = 0; c < N; ++c) out[s][c] += P * t[sp][c];
            }
    }
}

// O1 at one site: D psi(x) = (4 + m0) psi(x) - 1/2 H psi(x)
void dirac_site(const Lat& g, int rep, double m0, const double* U, const cd* psi, long x, cd* out_site) {
    const int N = rep == 0 ? 2 : 3;
    cd h[4][3];
    hop_site(g, rep, U, psi, x, h);
    for (int s = 0; s < 4; ++s)
        for (int c = 0; c < N; ++c)
            out_site[s * N + c] = (4.0 + m0) * psi[(x * 4 + s) * N + c] - 0.5 * h[s][c];
}

// ---- 2x2 complex helpers for the clover leaves (fundamental links only) ----
struct M2 { cd a[2][2]; };

M2 fund(const double* U, long x, int mu) {
    const cd* u = reinterpret_cast<const cd*>(U) + (x * 4 + mu) * 4;
    M2 r;
    r.a[0][0] = u[0]; r.a[0][1] = u[1]; r.a[1][0] = u[2]; r.a[1][1] = u[3];
    return r;
}
M2 mul(const M2& x, const M2& y) {
    M2 r;
    for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2; ++j) r.a[i][j] = x.a[i][0] * y.a[0][j] + x.a[i][1] * y.a[1][j];
    return r;
}
M2 dag(const M2& x) {
    M2 r;
    for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2; ++j) r.a[i][j] = std::conj(x.a[j][i]);
    return r;
}
M2 add(const M2& x, const M2& y) {
    M2 r;
    for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2; ++j) r.a[i][j] = x.a[i][j] + y.a[i][j];
    return r;
}

// O5: F^_mu,nu(x) = (Q - Q^dag)/8, Q = sum of the four mu-nu leaves that start and end at x
M2 field_strength(const Lat& g, const double* U, long x, int mu, int nu) {
    long xpm = shift(g, x, mu, +1), xpn = shift(g, x, nu, +1);
    long xmm = shift(g, x, mu, -1), xmn = shift(g, x, nu, -1);
    long xmm_pn = shift(g, xmm, nu, +1), xmm_mn = shift(g, xmm, nu, -1), xpm_mn = shift(g, xpm, nu, -1);
    // P1 = U_mu(x) U_nu(x+mu) U_mu(x+nu)^dag U_nu(x)^dag
    M2 P1 = mul(mul(fund(U, x, mu), fund(U, xpm, nu)), mul(dag(fund(U, xpn, mu)), dag(fund(U, x, nu))));
    // P2 = U_nu(x) U_mu(x-mu+nu)^dag U_nu(x-mu)^dag U_mu(x-mu)
    M2 P2 = mul(mul(fund(U, x, nu), dag(fund(U, xmm_pn, mu))), mul(dag(fund(U, xmm, nu)), fund(U, xmm, mu)));
    // P3 = U_mu(x-mu)^dag U_nu(x-mu-nu)^dag U_mu(x-mu-nu) U_nu(x-nu)
    M2 P3 = mul(mul(dag(fund(U, xmm, mu)), dag(fund(U, xmm_mn, nu))), mul(fund(U, xmm_mn, mu), fund(U, xmn, nu)));
    // P4 = U_nu(x-nu)^dag U_mu(x-nu) U_nu(x+mu-nu) U_mu(x)^dag
    M2 P4 = mul(mul(dag(fund(U, xmn, nu)), fund(U, xmn, mu)), mul(fund(U, xpm_mn, nu), dag(fund(U, x, mu))));
    M2 Q = add(add(P1, P2), add(P3, P4));
    M2 Qd = dag(Q), F;
    for (int i = 0; i < 2; ++i)
        for (int j = 0; j < 2; ++j) F.a[i][j] = (Q.a[i][j] - Qd.a[i][j]) / 8.0;
    return F;
}

// O5/O6: dense 8x8 site matrix  diag*1 + csw (i/2) sum_{mu<nu} sigma_mu,nu (x) F^_mu,nu(x)
// sigma_mu,nu = (i/2)[gamma_mu, gamma_nu]
void clover_site(const Lat& g, double diag, double csw, const double* U, long x, cd A[8][8]) {
    cd G[4][4][4];
    gamma_matrices(G);
    for (int r = 0; r < 8; ++r)
        for (int c = 0; c < 8; ++c) A[r][c] = (r == c) ? cd(diag, 0.0) : cd(0.0, 0.0);
    for (int mu = 0; mu < 4; ++mu)
        for (int nu = mu + 1; nu < 4; ++nu) {
            cd sig[4][4];
            for (int a = 0; a < 4; ++a)
                for (int b = 0; b < 4; ++b) {
                    cd ab = 0.0, ba = 0.0;
                    for (int k = 0; k < 4; ++k) {
                        ab += G[mu][a][k] * G[nu][k][b];
                        ba += G[nu][a][k] * G[mu][k][b];
                    }
                    sig[a][b] = 0.5 * I_ * (ab - ba);
                }
            M2 F = field_strength(g, U, x, mu, nu);
            for (int s = 0; s < 4; ++s)
                for (int sp = 0; sp < 4; ++sp)
                    for (int c = 0; c < 2; ++c)
                        for (int cp = 0; cp < 2; ++cp)
                            A[s * 2 + c][sp * 2 + cp] += csw * 0.5 * I_ * sig[s][sp] * F.a[c][cp];
        }
}

// generic dense complex inverse, Gauss-Jordan with partial pivoting; returns 0, or 1 if singular
int invert_dense(int n, const cd* A, cd* Ainv) {
    std::vector<cd> W((size_t)n * 2 * n);
    for (int r = 0; r < n; ++r)
        for (int c = 0; c < n; ++c) {
            W[(size_t)r * 2 * n + c] = A[r * n + c];
            W[(size_t)r * 2 * n + n + c] = (r == c) ? 1.0 : 0.0;
        }
    for (int k = 0; k < n; ++k) {
        int piv = k;
        double best = std::abs(W[(size_t)k * 2 * n + k]);
        for (int r = k + 1; r < n; ++r) {
            double v = std::abs(W[(size_t)r * 2 * n + k]);
            if (v > best) { best = v; piv = r; }
        }
        if (best == 0.0) return 1;
        if (piv != k)
            for (int c = 0; c < 2 * n; ++c) std::swap(W[(size_t)k * 2 * n + c], W[(size_t)piv * 2 * n + c]);
        cd d = W[(size_t)k * 2 * n + k];
        for (int c = 0; c < 2 * n; ++c) W[(size_t)k * 2 * n + c] /= d;
        for (int r = 0; r < n; ++r) {
            if (r == k) continue;
            cd f = W[(size_t)r * 2 * n + k];
            if (f == cd(0.0, 0.0)) continue;
            for (int c = 0; c < 2 * n; ++c) W[(size_t)r * 2 * n + c] -= f * W[(size_t)k * 2 * n + c];
        }
    }
    for (int r = 0; r < n; ++r)
        for (int c = 0; c < n; ++c) Ainv[r * n + c] = W[(size_t)r * 2 * n + n + c];
    return 0;
}

template <class F>
void run_ranges(long begin, long end, int nthreads, F f) {
    if (nthreads <= 1) { f(begin, end); return; }
    std::vector<std::thread> th;
    long n = end - begin;
    for (int t = 0; t < nthreads; ++t) {
        long b = begin + n * t / nthreads, e = begin + n * (t + 1) / nthreads;
        th.emplace_back([=]() { f(b, e); });
    }
    for (auto& t : th) t.join();
}

}  // namespace

extern "C" {

// Fill G[mu][row][col][re,im] with the A2 gamma matrices (for tests that need the basis).
void orc_gamma(double* G) {
    cd g[4][4][4];
    gamma_matrices(g);
    std::memcpy(G, g, sizeof(g));
}

// O1 on lex sites [begin, end): out[x] = D psi(x).  rep 0: fund (N=2), rep 1: adjoint (N=3, real links), rep 2: N=3, complex links.
// Contiguous output ranges are split over `nthreads` std::threads (SURVEY §8(d) CPU baseline).
int orc_dirac(const int* L, int rep, double m0, const double* U, const double* psi, double* out,
              long begin, long end, int nthreads) {
    Lat g = make_lat(L);
    const int N = rep == 0 ? 2 : 3;
    const cd* p = reinterpret_cast<const cd*>(psi);
    cd* o = reinterpret_cast<cd*>(out);
    run_ranges(begin, end, nthreads, [=](long b, long e) {
        for (long x = b; x < e; ++x) dirac_site(g, rep, m0, U, p, x, o + x * 4 * N);
    });
    return 0;
}

// O1 on a list of sites: out[k] = D psi(sites[k])  (sampled parity checks at 48^4)
int orc_dirac_sites(const int* L, int rep, double m0, const double* U, const double* psi,
                    long nsites, const long* sites, double* out) {
    Lat g = make_lat(L);
    const int N = rep == 0 ? 2 : 3;
    const cd* p = reinterpret_cast<const cd*>(psi);
    cd* o = reinterpret_cast<cd*>(out);
    for (long k = 0; k < nsites; ++k) dirac_site(g, rep, m0, U, p, sites[k], o + k * 4 * N);
    return 0;
}

// O2: for lex sites x in [begin, end) of parity `out_parity`: out[x] = H psi(x) (bare sum, no -1/2).
// Sites of the other parity are left untouched.  psi is read only at sites of the opposite parity.
int orc_hop(const int* L, int rep, int out_parity, const double* U, const double* psi, double* out,
            long begin, long end, int nthreads) {
    Lat g = make_lat(L);
    const int N = rep == 0 ? 2 : 3;
    const cd* p = reinterpret_cast<const cd*>(psi);
    cd* o = reinterpret_cast<cd*>(out);
    run_ranges(begin, end, nthreads, [=](long b, long e) {
        for (long x = b; x < e; ++x) {
            if (parity(g, x) != out_parity) continue;
            cd h[4][3];
            hop_site(g, rep, U, p, x, h);
            for (int s = 0; s < 4; ++s)
                for (int c = 0; c < N; ++c) o[(x * 4 + s) * N + c] = h[s][c];
        }
    });
    return 0;
}

// O2 on a list of sites (any parity): out[k] = H psi(sites[k])
int orc_hop_sites(const int* L, int rep, const double* U, const double* psi, long nsites,
                  const long* sites, double* out) {
    Lat g = make_lat(L);
    const int N = rep == 0 ? 2 : 3;
    const cd* p = reinterpret_cast<const cd*>(psi);
    cd* o = reinterpret_cast<cd*>(out);
    for (long k = 0; k < nsites; ++k) {
        cd h[4][3];
        hop_site(g, rep, U, p, sites[k], h);
        for (int s = 0; s < 4; ++s)
            for (int c = 0; c < N; ++c) o[(k * 4 + s) * N + c] = h[s][c];
    }
    return 0;
}

// O3: D^ psi_e = (4+m0) psi_e - H_eo H_oe psi_e / (4 (4+m0)).  Full-lattice arrays; only the even
// entries of psi are read; out is written on even sites and set to 0 on odd sites.
int orc_dirac_eo(const int* L, int rep, double m0, const double* U, const double* psi, double* out,
                 int nthreads) {
    Lat g = make_lat(L);
    const int N = rep == 0 ? 2 : 3;
    const long n = g.V * 4 * N;
    std::vector<cd> pe(n), tmp(n, cd(0.0, 0.0)), h2(n, cd(0.0, 0.0));
    const cd* p = reinterpret_cast<const cd*>(psi);
    for (long x = 0; x < g.V; ++x)
        for (int k = 0; k < 4 * N; ++k) pe[x * 4 * N + k] = parity(g, x) == 0 ? p[x * 4 * N + k] : cd(0.0, 0.0);
    orc_hop(L, rep, 1, U, reinterpret_cast<const double*>(pe.data()), reinterpret_cast<double*>(tmp.data()), 0, g.V, nthreads);
    orc_hop(L, rep, 0, U, reinterpret_cast<const double*>(tmp.data()), reinterpret_cast<double*>(h2.data()), 0, g.V, nthreads);
    cd* o = reinterpret_cast<cd*>(out);
    const double d = 4.0 + m0;
    for (long x = 0; x < g.V; ++x)
        for (int k = 0; k < 4 * N; ++k) {
            long i = x * 4 * N + k;
            o[i] = parity(g, x) == 0 ? d * pe[i] - h2[i] / (4.0 * d) : cd(0.0, 0.0);
        }
    return 0;
}

// O4: R^{ab} = 1/2 tr(sigma_a U sigma_b U^dag) for n fundamental links [n][2][2] -> [n][3][3] real.
// Returns the largest |imaginary part| seen through *max_imag (should be rounding noise).
int orc_represent(long n, const double* Ufund, double* Uadj, double* max_imag) {
    const cd sig[3][2][2] = {{{0.0, 1.0}, {1.0, 0.0}}, {{0.0, -I_}, {I_, 0.0}}, {{1.0, 0.0}, {0.0, -1.0}}};
    const cd* u = reinterpret_cast<const cd*>(Ufund);
    double mi = 0.0;
    for (long k = 0; k < n; ++k) {
        M2 Um, Ud;
        Um.a[0][0] = u[k * 4 + 0]; Um.a[0][1] = u[k * 4 + 1]; Um.a[1][0] = u[k * 4 + 2]; Um.a[1][1] = u[k * 4 + 3];
        Ud = dag(Um);
        for (int a = 0; a < 3; ++a)
            for (int b = 0; b < 3; ++b) {
                M2 sa, sb;
                for (int i = 0; i < 2; ++i)
                    for (int j = 0; j < 2; ++j) { sa.a[i][j] = sig[a][i][j]; sb.a[i][j] = sig[b][i][j]; }
                M2 T = mul(mul(sa, Um), mul(sb, Ud));
                cd tr = 0.5 * (T.a[0][0] + T.a[1][1]);
                Uadj[k * 9 + a * 3 + b] = tr.real();
                if (std::fabs(tr.imag()) > mi) mi = std::fabs(tr.imag());
            }
    }
    if (max_imag) *max_imag = mi;
    return 0;
}

// O5: F^_mu,nu(x) for every site: F[lex][2][2][re,im]
int orc_field_strength(const int* L, const double* U, int mu, int nu, double* F) {
    Lat g = make_lat(L);
    cd* f = reinterpret_cast<cd*>(F);
    for (long x = 0; x < g.V; ++x) {
        M2 m = field_strength(g, U, x, mu, nu);
        f[x * 4 + 0] = m.a[0][0]; f[x * 4 + 1] = m.a[0][1]; f[x * 4 + 2] = m.a[1][0]; f[x * 4 + 3] = m.a[1][1];
    }
    return 0;
}

// O5/O6: dense site matrices on lex sites [begin,end): A[x] = diag*1 + C(x), C = csw (i/2) sum_{mu<nu} sigma F^.
// diag = 4+m0 gives the clover block A of O6 (A10); diag = 0 gives the bare clover term C.
int orc_clover_dense(const int* L, double diag, double csw, const double* U, double* A, long begin, long end,
                     int nthreads) {
    Lat g = make_lat(L);
    cd* a = reinterpret_cast<cd*>(A);
    run_ranges(begin, end, nthreads, [=](long b, long e) {
        for (long x = b; x < e; ++x) clover_site(g, diag, csw, U, x, reinterpret_cast<cd(*)[8]>(a + x * 64));
    });
    return 0;
}

// generic inverse of nmat dense n x n complex matrices (Gauss-Jordan, partial pivoting)
int orc_invert(int n, long nmat, const double* A, double* Ainv) {
    const cd* a = reinterpret_cast<const cd*>(A);
    cd* b = reinterpret_cast<cd*>(Ainv);
    for (long k = 0; k < nmat; ++k)
        if (invert_dense(n, a + k * n * n, b + k * n * n)) return 1;
    return 0;
}

// out[x] = M[x] psi[x] for lex sites [begin,end) with parity in mask (bit0 even, bit1 odd); fund spinors (8 comps)
int orc_site_matvec(const int* L, int parity_mask, const double* M, const double* psi, double* out,
                    long begin, long end) {
    Lat g = make_lat(L);
    const cd* m = reinterpret_cast<const cd*>(M);
    const cd* p = reinterpret_cast<const cd*>(psi);
    cd* o = reinterpret_cast<cd*>(out);
    for (long x = begin; x < end; ++x) {
        if (!((parity_mask >> parity(g, x)) & 1)) continue;
        for (int r = 0; r < 8; ++r) {
            cd s = 0.0;
            for (int c = 0; c < 8; ++c) s += m[x * 64 + r * 8 + c] * p[x * 8 + c];
            o[x * 8 + r] = s;
        }
    }
    return 0;
}

// D_sw psi = D psi + C psi on all sites (O1 + O5), fundamental rep.  Cdense = bare clover term (diag = 0).
int orc_dirac_clover(const int* L, double m0, const double* U, const double* Cdense, const double* psi,
                     double* out, int nthreads) {
    Lat g = make_lat(L);
    orc_dirac(L, 0, m0, U, psi, out, 0, g.V, nthreads);
    std::vector<cd> c(g.V * 8);
    orc_site_matvec(L, 3, Cdense, psi, reinterpret_cast<double*>(c.data()), 0, g.V);
    cd* o = reinterpret_cast<cd*>(out);
    for (long i = 0; i < g.V * 8; ++i) o[i] += c[i];
    return 0;
}

// O7: D^ psi_e = A_ee psi_e - 1/4 H_eo A_oo^{-1} H_oe psi_e, fundamental rep.
// A, Ainv: dense 8x8 site matrices (from orc_clover_dense with diag = 4+m0, and orc_invert).
int orc_dirac_eo_clover(const int* L, const double* U, const double* A, const double* Ainv,
                        const double* psi, double* out, int nthreads) {
    Lat g = make_lat(L);
    const long n = g.V * 8;
    std::vector<cd> pe(n), t1(n, cd(0.0, 0.0)), t2(n, cd(0.0, 0.0)), t3(n, cd(0.0, 0.0)), ae(n, cd(0.0, 0.0));
    const cd* p = reinterpret_cast<const cd*>(psi);
    for (long x = 0; x < g.V; ++x)
        for (int k = 0; k < 8; ++k) pe[x * 8 + k] = parity(g, x) == 0 ? p[x * 8 + k] : cd(0.0, 0.0);
    const double* ped = reinterpret_cast<const double*>(pe.data());
    orc_hop(L, 0, 1, U, ped, reinterpret_cast<double*>(t1.data()), 0, g.V, nthreads);              // H_oe psi_e
    orc_site_matvec(L, 2, Ainv, reinterpret_cast<const double*>(t1.data()), reinterpret_cast<double*>(t2.data()), 0, g.V);  // A_oo^-1
    orc_hop(L, 0, 0, U, reinterpret_cast<const double*>(t2.data()), reinterpret_cast<double*>(t3.data()), 0, g.V, nthreads); // H_eo
    orc_site_matvec(L, 1, A, ped, reinterpret_cast<double*>(ae.data()), 0, g.V);                     // A_ee psi_e
    cd* o = reinterpret_cast<cd*>(out);
    for (long x = 0; x < g.V; ++x)
        for (int k = 0; k < 8; ++k) {
            long i = x * 8 + k;
            o[i] = parity(g, x) == 0 ? ae[i] - 0.25 * t3[i] : cd(0.0, 0.0);
        }
    return 0;
}

int orc_hardware_threads(void) { return (int)std::thread::hardware_concurrency(); }

}  // extern "C"
