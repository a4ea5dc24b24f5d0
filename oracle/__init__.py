"""CPU oracle — TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/oracle.cpp header).

ctypes marshalling around oracle/liboracle.so; every function here only converts numpy
arrays to pointers and back.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from
paper_2411_18511_b200.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """g++ -O2 the oracle into oracle/liboracle.so (plain C++, no intrinsics)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-pthread", "-o", _LIB, _SRC])
    return _LIB


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
    return _lib


def _p(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _L(L):
    return (ctypes.c_int * 4)(*[int(v) for v in L])


def _c(a):
    a = np.ascontiguousarray(a)
    assert a.dtype in (np.complex128, np.float64), a.dtype
    return a


REP_FUND, REP_ADJ, REP_SU3 = 0, 1, 2      # rep argument of dirac / hop / dirac_eo: link format of oracle.cpp link()


def _vol(L):
    return int(L[0]) * int(L[1]) * int(L[2]) * int(L[3])


def available_cores() -> int:
    try:
        return len(os.sched_getaffinity(0))
    except AttributeError:
        return os.cpu_count() or 1


def gamma() -> np.ndarray:
    """A2 gamma matrices, complex128 [4,4,4]."""
    g = np.empty((4, 4, 4), dtype=np.complex128)
    lib().orc_gamma(_p(g))
    return g


def dirac(L, rep, m0, U, psi, begin=0, end=None, nthreads=1, out=None):
    """O1: D psi on lex sites [begin,end) (other sites of `out` untouched / zero)."""
    U, psi = _c(U), _c(psi)
    V = _vol(L)
    end = V if end is None else end
    if out is None:
        out = np.zeros_like(psi)
    lib().orc_dirac(_L(L), int(rep), ctypes.c_double(m0), _p(U), _p(psi), _p(out),
                    ctypes.c_long(begin), ctypes.c_long(end), int(nthreads))
    return out


def dirac_sites(L, rep, m0, U, psi, sites):
    U, psi = _c(U), _c(psi)
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((len(sites),) + psi.shape[1:], dtype=np.complex128)
    lib().orc_dirac_sites(_L(L), int(rep), ctypes.c_double(m0), _p(U), _p(psi),
                          ctypes.c_long(len(sites)), _p(sites), _p(out))
    return out


def hop(L, rep, out_parity, U, psi, begin=0, end=None, nthreads=1, out=None):
    """O2: out[x] = H psi(x) on sites of parity out_parity, zero elsewhere."""
    U, psi = _c(U), _c(psi)
    V = _vol(L)
    end = V if end is None else end
    if out is None:
        out = np.zeros_like(psi)
    lib().orc_hop(_L(L), int(rep), int(out_parity), _p(U), _p(psi), _p(out),
                  ctypes.c_long(begin), ctypes.c_long(end), int(nthreads))
    return out


def hop_sites(L, rep, U, psi, sites):
    U, psi = _c(U), _c(psi)
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((len(sites),) + psi.shape[1:], dtype=np.complex128)
    lib().orc_hop_sites(_L(L), int(rep), _p(U), _p(psi), ctypes.c_long(len(sites)), _p(sites), _p(out))
    return out


def dirac_eo(L, rep, m0, U, psi, nthreads=1):
    """O3: even-odd preconditioned operator on the even entries of psi (odd output = 0)."""
    U, psi = _c(U), _c(psi)
    out = np.zeros_like(psi)
    lib().orc_dirac_eo(_L(L), int(rep), ctypes.c_double(m0), _p(U), _p(psi), _p(out), int(nthreads))
    return out


def represent(Ufund):
    """O4: adjoint links [...,3,3] float64 from fundamental links [...,2,2]; also max |imag|."""
    Ufund = _c(Ufund)
    n = Ufund.size // 4
    out = np.empty(Ufund.shape[:-2] + (3, 3), dtype=np.float64)
    mi = ctypes.c_double(0.0)
    lib().orc_represent(ctypes.c_long(n), _p(Ufund), _p(out), ctypes.byref(mi))
    return out, mi.value


def field_strength(L, U, mu, nu):
    """O5: F^_mu,nu(x), complex128 [V,2,2]."""
    U = _c(U)
    F = np.empty((_vol(L), 2, 2), dtype=np.complex128)
    lib().orc_field_strength(_L(L), _p(U), int(mu), int(nu), _p(F))
    return F


def clover_dense(L, diag, csw, U, begin=0, end=None, nthreads=1):
    """O5/O6: dense [V,8,8] site matrices diag*1 + C(x) (rows/cols = spin*2 + colour)."""
    U = _c(U)
    V = _vol(L)
    end = V if end is None else end
    A = np.zeros((V, 8, 8), dtype=np.complex128)
    lib().orc_clover_dense(_L(L), ctypes.c_double(diag), ctypes.c_double(csw), _p(U), _p(A),
                           ctypes.c_long(begin), ctypes.c_long(end), int(nthreads))
    return A


def invert(A):
    """Generic dense inverse of a stack of n x n complex matrices."""
    A = _c(A)
    n = A.shape[-1]
    out = np.empty_like(A)
    rc = lib().orc_invert(int(n), ctypes.c_long(A.size // (n * n)), _p(A), _p(out))
    if rc:
        raise ZeroDivisionError("singular matrix in oracle.invert")
    return out


def site_matvec(L, parity_mask, M, psi, begin=0, end=None):
    M, psi = _c(M), _c(psi)
    V = _vol(L)
    end = V if end is None else end
    out = np.zeros_like(psi)
    lib().orc_site_matvec(_L(L), int(parity_mask), _p(M), _p(psi), _p(out), ctypes.c_long(begin), ctypes.c_long(end))
    return out


def dirac_clover(L, m0, U, Cdense, psi, nthreads=1):
    """D_sw psi = D psi + C psi on all sites (Cdense built with diag = 0)."""
    U, Cdense, psi = _c(U), _c(Cdense), _c(psi)
    out = np.zeros_like(psi)
    lib().orc_dirac_clover(_L(L), ctypes.c_double(m0), _p(U), _p(Cdense), _p(psi), _p(out), int(nthreads))
    return out


def dirac_eo_clover(L, U, A, Ainv, psi, nthreads=1):
    """O7 on the even entries of psi (odd output = 0)."""
    U, A, Ainv, psi = _c(U), _c(A), _c(Ainv), _c(psi)
    out = np.zeros_like(psi)
    lib().orc_dirac_eo_clover(_L(L), _p(U), _p(A), _p(Ainv), _p(psi), _p(out), int(nthreads))
    return out


# ------------------------------------------------------------------ O8: conjugate gradient on the normal equations
def cg_normal(L, rep, m0, U, b, tol=1e-12, max_iter=2000, nthreads=1, A=None, Ainv=None, dhat=None):
    """O8 (the HMC inverts the even-odd operator): solve
        Dhat^dag Dhat x = b        on the even sites,   Dhat^dag = gamma5 Dhat gamma5  (pin P2),
    by the textbook conjugate-gradient iteration (Hestenes-Stiefel) from x = 0, in the order
        r = b, p = r;  loop:  q = Dhat^dag Dhat p;  alpha = <r,r>/<p,q>;  x += alpha p;  r -= alpha q;
                              stop when |r| <= tol |b|;  beta = <r,r>_new/<r,r>_old;  p = r + beta p.
    b, x: complex [V,4,N] with zero odd entries.  Returns (x, iterations, |r|/|b|).  Plain numpy on top of
    dirac_eo (dirac_eo_clover when A, Ainv are given); no preconditioning, no restarts, no reordering."""
    g5 = np.array([1.0, 1.0, -1.0, -1.0])[None, :, None]

    def Dhat(v):   # O3, or O7 when the dense clover matrices A, A^-1 are given (fundamental representation),
        if dhat is not None:   # or any even-odd operator handed in (e.g. dirac_eo_clover_adj)
            return dhat(v)
        if A is None:
            return dirac_eo(L, rep, m0, U, v, nthreads)
        return dirac_eo_clover(L, U, A, Ainv, v, nthreads)

    def M(v):
        return g5 * Dhat(g5 * Dhat(v))

    b = _c(b)
    x = np.zeros_like(b)
    r = b.copy()
    p = r.copy()
    rr = float(np.vdot(r, r).real)
    bb = rr
    it = 0
    while it < max_iter and rr > tol * tol * bb:
        q = M(p)
        alpha = rr / float(np.vdot(p, q).real)
        x += alpha * p
        r -= alpha * q
        rr_new = float(np.vdot(r, r).real)
        p = r + (rr_new / rr) * p
        rr = rr_new
        it += 1
    return x, it, float(np.sqrt(rr / bb))


# ------------------------------------------------------------------ O9: exponential clover term
def clover_exp_dense(L, diag, csw, U, nthreads=1, begin=0, end=None):
    """O9 ("exponential of the clover term ... the diagonal part of the Dirac operator and its inverse
    take the same time to execute", ref [6] at PAPER.md:123; reading B4 of DESIGN.md §3): the site-diagonal term of
    the exponential clover improvement,
        A_exp(x) = diag * exp( C(x) / diag ),     A_exp(x)^-1 = exp( -C(x) / diag ) / diag,     diag = 4 + m0,
    with C(x) = csw (i/4) sum_{mu,nu} sigma_mu,nu F^_mu,nu(x) the clover term of O5 (the regular term is diag + C,
    the first two orders of this exponential).  The exponential of the hermitian 8x8 matrix C/diag is taken from
    its eigendecomposition, exp(H) = V diag(e^lambda) V^dag.  Returns (A_exp, A_exp^-1), dense [V,8,8]."""
    # (begin, end: restrict to the lex sites [begin, end); the returned arrays then hold only those sites)
    end = _vol(L) if end is None else end
    A = clover_dense(L, diag, csw, U, begin, end, nthreads)[begin:end]
    C = A - diag * np.eye(8)[None]
    return _exp_hermitian_pair(C, diag)


def _exp_hermitian_pair(C, diag):
    """(diag exp(C/diag), exp(-C/diag)/diag) for a stack of hermitian matrices C, from the eigendecomposition
    exp(H) = V diag(e^lambda) V^dag."""
    lam, V = np.linalg.eigh(C / diag)
    Vh = np.conj(np.swapaxes(V, -1, -2))
    return diag * (V * np.exp(lam)[:, None, :]) @ Vh, (V * np.exp(-lam)[:, None, :]) @ Vh / diag


# ------------------------------------------------------------------ O10: clover term in the adjoint representation
def clover_dense_adj(L, diag, csw, R):
    """O10 (SURVEY.md §8(f) item 3 "adjoint-representation clover"): the clover term of O5 with the
    real 3x3 adjoint links R in place of U (dagger = transpose), acting on 4 spin x 3 colour:
        A(x) = diag + C(x),  C = csw (i/2) sum_{mu<nu} sigma_mu,nu (x) F^_mu,nu,  sigma_mu,nu = (i/2)[gamma_mu, gamma_nu],
        F^_mu,nu = (Q - Q^T)/8,  Q = P1 + P2 + P3 + P4 the four leaves of O5 that start and end at x (mu -> nu sense).
    R: real [V,4,3,3].  Returns dense [V,12,12] complex (row/col = spin*3 + colour).  Whole-lattice numpy shifts."""
    R = np.ascontiguousarray(R, dtype=np.float64)
    Lt = tuple(int(v) for v in L)
    V = _vol(L)
    Rg = R.reshape(Lt + (4, 3, 3))
    gam = gamma()

    def at(mu, shift):      # U_mu(x + shift), shift a dict {axis: displacement}
        a = Rg[..., mu, :, :]
        for ax, d in shift.items():
            a = np.roll(a, -d, axis=ax)
        return a

    def T(m):
        return np.swapaxes(m, -1, -2)

    A = np.zeros((V, 12, 12), dtype=np.complex128)
    A += diag * np.eye(12)[None]
    for mu in range(4):
        for nu in range(mu + 1, 4):
            P1 = at(mu, {}) @ at(nu, {mu: 1}) @ T(at(mu, {nu: 1})) @ T(at(nu, {}))
            P2 = at(nu, {}) @ T(at(mu, {mu: -1, nu: 1})) @ T(at(nu, {mu: -1})) @ at(mu, {mu: -1})
            P3 = T(at(mu, {mu: -1})) @ T(at(nu, {mu: -1, nu: -1})) @ at(mu, {mu: -1, nu: -1}) @ at(nu, {nu: -1})
            P4 = T(at(nu, {nu: -1})) @ at(mu, {nu: -1}) @ at(nu, {mu: 1, nu: -1}) @ T(at(mu, {}))
            Q = P1 + P2 + P3 + P4
            F = ((Q - T(Q)) / 8.0).reshape(V, 3, 3)
            sig = 0.5j * (gam[mu] @ gam[nu] - gam[nu] @ gam[mu])
            A += csw * 0.5j * np.einsum("st,xab->xsatb", sig, F).reshape(V, 12, 12)
    return A


def clover_exp_dense_adj(L, diag, csw, R):
    """O11 (PAPER.md:59-61 exponential clover, PAPER.md:21, 53 higher representations; readings B4 + B5 of DESIGN.md
    §3): the exponential site-diagonal term in the adjoint representation,
        A_exp(x) = diag * exp( C(x) / diag ),     A_exp(x)^-1 = exp( -C(x) / diag ) / diag,
    with C(x) = clover_dense_adj(L, 0, csw, R) the 12x12 hermitian clover term of O10; the exponential is taken from
    the eigendecomposition as in O9.  Returns (A_exp, A_exp^-1), dense [V,12,12].  Pinned by P19."""
    C = clover_dense_adj(L, 0.0, csw, R)
    return _exp_hermitian_pair(C, diag)


def site_matvec_n(M, psi, mask=None):
    """out[x] = M[x] psi[x] for dense [V,n,n] site matrices and spinors [V,4,N] (n = 4N); sites with mask False -> 0."""
    V = psi.shape[0]
    out = np.einsum("xij,xj->xi", M, psi.reshape(V, -1)).reshape(psi.shape)
    if mask is not None:
        out = np.where(mask[:, None, None], out, 0.0)
    return out


def dirac_eo_clover_adj(L, R, A, Ainv, psi, nthreads=1):
    """O7 in the adjoint representation: Dhat psi_e = A_ee psi_e - 1/4 H_eo A_oo^-1 H_oe psi_e (odd output = 0);
    A, Ainv dense [V,12,12] (clover_dense_adj with diag = 4 + m0 and its inverse)."""
    par = (np.indices(tuple(int(v) for v in L)).sum(axis=0) % 2).reshape(-1)     # (x0+x1+x2+x3) mod 2, lex order
    even, odd = par == 0, par == 1
    pe = np.where(even[:, None, None], psi, 0.0)
    t = hop(L, 1, 1, R, pe, nthreads=nthreads)              # H_oe psi_e on odd sites
    t = site_matvec_n(Ainv, t, odd)
    h = hop(L, 1, 0, R, t, nthreads=nthreads)               # H_eo (...) on even sites
    return site_matvec_n(A, pe, even) - 0.25 * h


# ------------------------------------------------------------------ O12: clover term for complex 3 x 3 links (HR_REP_SU3)
def clover_dense_su3(L, diag, csw, U):
    """O12 (SURVEY.md §8(f) item 4 "other groups"): the clover term of O5 for complex 3 x 3 links U
    (dagger = conjugate transpose), acting on 4 spin x 3 colour:
        A(x) = diag + C(x),  C = csw (i/2) sum_{mu<nu} sigma_mu,nu (x) F^_mu,nu,  sigma_mu,nu = (i/2)[gamma_mu, gamma_nu],
        F^_mu,nu = (Q - Q^dag)/8,  Q = P1 + P2 + P3 + P4 the four leaves of O5 that start and end at x (mu -> nu sense).
    U: complex [V,4,3,3].  Returns dense [V,12,12] complex (row/col = spin*3 + colour).  Whole-lattice numpy shifts; the
    same construction as O10 with the real adjoint links replaced by complex ones.  Pinned by P22."""
    U = np.ascontiguousarray(U, dtype=np.complex128)
    Lt = tuple(int(v) for v in L)
    V = _vol(L)
    Ug = U.reshape(Lt + (4, 3, 3))
    gam = gamma()

    def at(mu, shift):      # U_mu(x + shift), shift a dict {axis: displacement}
        a = Ug[..., mu, :, :]
        for ax, d in shift.items():
            a = np.roll(a, -d, axis=ax)
        return a

    def H(m):
        return np.conj(np.swapaxes(m, -1, -2))

    A = np.zeros((V, 12, 12), dtype=np.complex128)
    A += diag * np.eye(12)[None]
    for mu in range(4):
        for nu in range(mu + 1, 4):
            P1 = at(mu, {}) @ at(nu, {mu: 1}) @ H(at(mu, {nu: 1})) @ H(at(nu, {}))
            P2 = at(nu, {}) @ H(at(mu, {mu: -1, nu: 1})) @ H(at(nu, {mu: -1})) @ at(mu, {mu: -1})
            P3 = H(at(mu, {mu: -1})) @ H(at(nu, {mu: -1, nu: -1})) @ at(mu, {mu: -1, nu: -1}) @ at(nu, {nu: -1})
            P4 = H(at(nu, {nu: -1})) @ at(mu, {nu: -1}) @ at(nu, {mu: 1, nu: -1}) @ H(at(mu, {}))
            Q = P1 + P2 + P3 + P4
            F = ((Q - H(Q)) / 8.0).reshape(V, 3, 3)
            sig = 0.5j * (gam[mu] @ gam[nu] - gam[nu] @ gam[mu])
            A += csw * 0.5j * np.einsum("st,xab->xsatb", sig, F).reshape(V, 12, 12)
    return A


def clover_exp_dense_su3(L, diag, csw, U):
    """the exponential site-diagonal term (O9 / O11, reading B4) for complex 3 x 3 links: (diag exp(C/diag), exp(-C/diag)/diag) with
    C = clover_dense_su3(L, 0, csw, U); dense [V,12,12]."""
    return _exp_hermitian_pair(clover_dense_su3(L, 0.0, csw, U), diag)


def dirac_eo_clover_n(L, rep, U, A, Ainv, psi, nthreads=1):
    """O7 for any representation of link() with dense site matrices: Dhat psi_e = A_ee psi_e - 1/4 H_eo A_oo^-1 H_oe psi_e (odd
    output = 0); A, Ainv dense [V,4N,4N].  The construction of dirac_eo_clover_adj (pinned by P18) with the hop's representation
    as an argument; rep = 2 (complex 3 x 3 links) is pinned by P22."""
    par = (np.indices(tuple(int(v) for v in L)).sum(axis=0) % 2).reshape(-1)
    even, odd = par == 0, par == 1
    pe = np.where(even[:, None, None], psi, 0.0)
    t = hop(L, rep, 1, U, pe, nthreads=nthreads)
    t = site_matvec_n(Ainv, t, odd)
    h = hop(L, rep, 0, U, t, nthreads=nthreads)
    return site_matvec_n(A, pe, even) - 0.25 * h


# ------------------------------------------------------------------ O13: two-index antisymmetric representation of SU(3)
def represent_antisym_su3(U):
    """O13 (SURVEY.md §8(f) item 4 "symmetric/antisymmetric reps", "higher representations"; DESIGN.md §3 reading B9):
    the two-index antisymmetric representation of complex 3 x 3 links by its definition as the action U e U^T on antisymmetric
    matrices,
        R_ab(U) = tr( (e^a)^dag  U  e^b  U^T ),     e^a = (E_ij - E_ji) / sqrt(2)  for the pairs a = (i<j) = (0,1), (0,2), (1,2),
    written out with explicit basis matrices and one einsum (no minors, no cofactors).  U: complex [..., 3, 3]; returns complex
    [..., 3, 3].  For N = 3 the representation has dimension N(N-1)/2 = 3 and the result is again a special unitary 3 x 3 matrix, so
    the operators of link() rep 2 act on it unchanged.  Pinned by P23."""
    U = np.ascontiguousarray(U, dtype=np.complex128)
    pairs = [(0, 1), (0, 2), (1, 2)]
    e = np.zeros((3, 3, 3), dtype=np.complex128)
    for a, (i, j) in enumerate(pairs):
        e[a, i, j] = 1.0 / np.sqrt(2.0)
        e[a, j, i] = -1.0 / np.sqrt(2.0)
    # tr(e^a^dag U e^b U^T) = sum_{ijkl} conj(e^a_ij) U_ik e^b_kl U_jl
    return np.einsum("aij,...ik,bkl,...jl->...ab", np.conj(e), U, e, U)
