"""Pins P1-P20 (P15-P20 for the oracle pieces of the §8(f) rows): what holds the CPU oracle in place.

The paper (arXiv 2411.18511) prints no formula and no worked numeric example (PAPER.md:29-39,
51-61 describe kernels only), so the oracle is pinned to what physics and mathematics fix:
closed forms, invariants, special cases, brute force.  Everything on the right-hand side of an
assert here is typed in this file / tests/helpers.py / tests/golden, or computed by numpy —
never by the CUDA path.
"""
import numpy as np
import pytest

from paper_2411_18511_b200 import inputs
from helpers import (PAULI, bwd, dagger, flat, fwd, gauge_transform, golden_gamma, grid, rel_l2,
                     wilson_dirac_numpy)

GAM = golden_gamma()
G5 = np.diag([1.0, 1.0, -1.0, -1.0]).astype(np.complex128)


def inner(a, b):
    return np.vdot(a.ravel(), b.ravel())


# ---------------------------------------------------------------- gamma basis (A2)
def test_gamma_basis_is_the_golden_one(orc):
    g = orc.gamma()
    assert np.array_equal(g, GAM)
    for mu in range(4):
        assert np.array_equal(g[mu], dagger(g[mu]))
        for nu in range(4):
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.allclose(anti, 2.0 * np.eye(4) * (mu == nu), atol=0)
    assert np.array_equal(g[0] @ g[1] @ g[2] @ g[3], G5)


# ---------------------------------------------------------------- P1 plane wave
@pytest.mark.parametrize("rep,N", [(0, 2), (1, 3)])
@pytest.mark.parametrize("n", [(1, 0, 3, 2), (1, 0, 0, 0), (0, 2, 0, 0), (0, 0, 1, 0), (0, 0, 0, 3)])
def test_P1_plane_wave(orc, rep, N, n):
    L = (4, 6, 4, 8)
    m0 = -0.2
    V = inputs.volume(L)
    x = inputs.site_coords(L)
    p = 2.0 * np.pi * np.array(n) / np.array(L)
    phase = np.exp(1j * (x @ p))
    rng = np.random.default_rng(11)
    w = rng.normal(size=(4, N)) + 1j * rng.normal(size=(4, N))
    psi = phase[:, None, None] * w[None]
    if rep == 0:
        U = inputs.unit_gauge(L)
    else:
        U = np.tile(np.eye(3), (V, 4, 1, 1))
    out = orc.dirac(L, rep, m0, U, psi)
    M = (m0 + np.sum(1.0 - np.cos(p))) * np.eye(4) + 1j * sum(GAM[mu] * np.sin(p[mu]) for mu in range(4))
    expect = phase[:, None, None] * (M @ w)[None]
    assert rel_l2(out, expect) < 1e-14
    # eigenvalues (basis independent): m0 + sum(1 - cos p) +- i sqrt(sum sin^2 p), each twice
    ev = np.linalg.eigvals(M)
    lam = m0 + np.sum(1.0 - np.cos(p))
    s = np.sqrt(np.sum(np.sin(p) ** 2))
    ev = ev[np.argsort(ev.imag)]
    assert np.allclose(ev, np.array([lam - 1j * s] * 2 + [lam + 1j * s] * 2), atol=1e-14)


# ---------------------------------------------------------------- P14 brute force / independent restatement
@pytest.mark.parametrize("L", [(2, 2, 2, 2), (4, 4, 4, 4), (2, 4, 6, 4)])
def test_P14_independent_restatement_fund(orc, L):
    U = inputs.haar_gauge(L, seed=1)
    psi = inputs.gaussian_spinor(L, 2, seed=2)
    out = orc.dirac(L, 0, -0.2, U, psi)
    ref = wilson_dirac_numpy(L, U, psi, -0.2, GAM)
    assert rel_l2(out, ref) < 1e-14


def test_P14_independent_restatement_adj(orc):
    L = (4, 2, 4, 6)
    Ua, _ = orc.represent(inputs.haar_gauge(L, seed=1))
    psi = inputs.gaussian_spinor(L, 3, seed=2)
    out = orc.dirac(L, 1, -0.3, Ua, psi)
    ref = wilson_dirac_numpy(L, Ua, psi, -0.3, GAM)
    assert rel_l2(out, ref) < 1e-14


def test_P14_dense_matrix_columns(orc):
    """2^4: assemble D column by column from the oracle and from the numpy restatement."""
    L = (2, 2, 2, 2)
    V = 16
    U = inputs.haar_gauge(L, seed=1)
    n = V * 8
    Do = np.empty((n, n), dtype=np.complex128)
    Dn = np.empty((n, n), dtype=np.complex128)
    for k in range(n):
        e = np.zeros(n, dtype=np.complex128)
        e[k] = 1.0
        e = e.reshape(V, 4, 2)
        Do[:, k] = orc.dirac(L, 0, -0.2, U, e).ravel()
        Dn[:, k] = wilson_dirac_numpy(L, U, e, -0.2, GAM).ravel()
    assert np.abs(Do - Dn).max() < 1e-14


# ---------------------------------------------------------------- P2 gamma5-hermiticity
@pytest.mark.parametrize("rep,N", [(0, 2), (1, 3)])
def test_P2_gamma5_hermiticity(orc, rep, N):
    L = (4, 4, 4, 4)
    U = inputs.haar_gauge(L, seed=1)
    if rep == 1:
        U, _ = orc.represent(U)
    psi = inputs.gaussian_spinor(L, N, seed=2)
    chi = inputs.gaussian_spinor(L, N, seed=3, field=inputs.FIELD_SPINOR2)
    g5 = lambda v: np.einsum("st,xtc->xsc", G5, v)
    lhs = inner(chi, orc.dirac(L, rep, -0.2, U, psi))
    rhs = inner(g5(orc.dirac(L, rep, -0.2, U, g5(chi))), psi)
    assert abs(lhs - rhs) / abs(lhs) < 1e-14


def test_P2_gamma5_hermiticity_clover(orc):
    L = (4, 4, 4, 4)
    U = inputs.weak_gauge(L, 0.3, seed=1)
    C = orc.clover_dense(L, 0.0, 1.2, U)
    psi = inputs.gaussian_spinor(L, 2, seed=2)
    chi = inputs.gaussian_spinor(L, 2, seed=3, field=inputs.FIELD_SPINOR2)
    g5 = lambda v: np.einsum("st,xtc->xsc", G5, v)
    lhs = inner(chi, orc.dirac_clover(L, -0.25, U, C, psi))
    rhs = inner(g5(orc.dirac_clover(L, -0.25, U, C, g5(chi))), psi)
    assert abs(lhs - rhs) / abs(lhs) < 1e-14


# ---------------------------------------------------------------- P3 gauge covariance
def test_P3_gauge_covariance_fund(orc):
    L = (4, 6, 4, 4)
    U = inputs.haar_gauge(L, seed=1)
    g = inputs.haar_sites(L, seed=4)
    psi = inputs.gaussian_spinor(L, 2, seed=2)
    Ug = gauge_transform(U, g, L)
    gpsi = np.einsum("xcd,xsd->xsc", g, psi)
    lhs = orc.dirac(L, 0, -0.2, Ug, gpsi)
    rhs = np.einsum("xcd,xsd->xsc", g, orc.dirac(L, 0, -0.2, U, psi))
    assert rel_l2(lhs, rhs) < 1e-14


def test_P3_gauge_covariance_adj(orc):
    L = (4, 4, 6, 4)
    U = inputs.haar_gauge(L, seed=1)
    g = inputs.haar_sites(L, seed=4)
    psi = inputs.gaussian_spinor(L, 3, seed=2)
    Ra, _ = orc.represent(U)
    Rg, _ = orc.represent(gauge_transform(U, g, L))
    Rsite, _ = orc.represent(g)
    gpsi = np.einsum("xcd,xsd->xsc", Rsite, psi)
    lhs = orc.dirac(L, 1, -0.3, Rg, gpsi)
    rhs = np.einsum("xcd,xsd->xsc", Rsite, orc.dirac(L, 1, -0.3, Ra, psi))
    assert rel_l2(lhs, rhs) < 1e-14


# ---------------------------------------------------------------- P9 EO vs full on a parity-supported vector
@pytest.mark.parametrize("rep,N", [(0, 2), (1, 3)])
def test_P9_hop_is_offdiagonal_part_of_D(orc, rep, N):
    L = (4, 4, 2, 6)
    m0 = -0.2
    U = inputs.haar_gauge(L, seed=1)
    if rep == 1:
        U, _ = orc.represent(U)
    par = inputs.site_parity(L)
    psi = inputs.gaussian_spinor(L, N, seed=2)
    psi_e = psi * (par == 0)[:, None, None]
    Dpsi = orc.dirac(L, rep, m0, U, psi_e)
    H = orc.hop(L, rep, 1, U, psi_e)
    assert np.array_equal(H[par == 0], np.zeros_like(H[par == 0]))
    assert rel_l2(Dpsi[par == 1], -0.5 * H[par == 1]) < 1e-15
    assert rel_l2(Dpsi[par == 0], (4 + m0) * psi_e[par == 0]) < 1e-15
    # hop_sites agrees with hop on a list of sites
    sites = np.nonzero(par == 1)[0][::7]
    assert np.array_equal(orc.hop_sites(L, rep, U, psi_e, sites), H[sites])
    assert np.array_equal(orc.dirac_sites(L, rep, m0, U, psi_e, sites), Dpsi[sites])


# ---------------------------------------------------------------- P4 Schur identity (no solve)
@pytest.mark.parametrize("rep,N", [(0, 2), (1, 3)])
def test_P4_schur_identity(orc, rep, N):
    L = (4, 4, 4, 6)
    m0 = -0.1
    d = 4.0 + m0
    U = inputs.haar_gauge(L, seed=1)
    if rep == 1:
        U, _ = orc.represent(U)
    par = inputs.site_parity(L)
    even = (par == 0)[:, None, None]
    x = inputs.gaussian_spinor(L, N, seed=2)
    eta = orc.dirac(L, rep, m0, U, x)
    # D^ x_e = eta_e - D_eo D_oo^-1 eta_o,  D_eo = -1/2 H_eo, D_oo = (4+m0)
    rhs = eta * even + 0.5 / d * orc.hop(L, rep, 0, U, eta * ~even)
    lhs = orc.dirac_eo(L, rep, m0, U, x)
    assert rel_l2(lhs, rhs) < 1e-14
    # x_o = D_oo^-1 (eta_o - D_oe x_e)
    xo = (eta * ~even + 0.5 * orc.hop(L, rep, 1, U, x * even)) / d
    assert rel_l2(xo, x * ~even) < 1e-14


def test_P4_schur_identity_clover(orc):
    L = (4, 4, 4, 4)
    m0, csw = -0.25, 1.2
    U = inputs.weak_gauge(L, 0.3, seed=1)
    par = inputs.site_parity(L)
    even = (par == 0)[:, None, None]
    C = orc.clover_dense(L, 0.0, csw, U)
    A = orc.clover_dense(L, 4.0 + m0, csw, U)
    assert np.abs(A - C - (4.0 + m0) * np.eye(8)).max() < 1e-15
    Ainv = orc.invert(A)
    x = inputs.gaussian_spinor(L, 2, seed=2)
    eta = orc.dirac_clover(L, m0, U, C, x)
    Ainv_eta_o = orc.site_matvec(L, 2, Ainv, eta)
    rhs = eta * even + 0.5 * orc.hop(L, 0, 0, U, Ainv_eta_o)
    lhs = orc.dirac_eo_clover(L, U, A, Ainv, x)
    assert rel_l2(lhs, rhs) < 1e-14


# ---------------------------------------------------------------- P5 Schur complement vs full solve at 4^4
def test_P5_schur_vs_full_solve(orc):
    L = (4, 4, 4, 4)
    m0 = -0.2
    d = 4.0 + m0
    V = 256
    n = V * 8
    U = inputs.haar_gauge(L, seed=1)
    par = inputs.site_parity(L)
    even = (par == 0)[:, None, None]
    D = np.empty((n, n), dtype=np.complex128)
    Dhat = np.zeros((n, n), dtype=np.complex128)
    for k in range(n):
        e = np.zeros(n, dtype=np.complex128)
        e[k] = 1.0
        e = e.reshape(V, 4, 2)
        D[:, k] = orc.dirac(L, 0, m0, U, e).ravel()
        if par[k // 8] == 0:
            Dhat[:, k] = orc.dirac_eo(L, 0, m0, U, e).ravel()
    eta = inputs.gaussian_spinor(L, 2, seed=2)
    x = np.linalg.solve(D, eta.ravel()).reshape(V, 4, 2)
    assert np.linalg.cond(D) < 10.0
    ev = np.repeat(par == 0, 8)
    rhs_e = (eta * even + 0.5 / d * orc.hop(L, 0, 0, U, eta * ~even)).ravel()[ev]
    xe = np.linalg.solve(Dhat[np.ix_(ev, ev)], rhs_e)
    assert rel_l2(xe, x.ravel()[ev]) < 1e-12
    x_e_full = np.zeros(n, dtype=np.complex128)
    x_e_full[ev] = xe
    xo = (eta * ~even + 0.5 * orc.hop(L, 0, 1, U, x_e_full.reshape(V, 4, 2))) / d
    assert rel_l2(xo.ravel()[~ev], x.ravel()[~ev]) < 1e-12


# ---------------------------------------------------------------- P6-P8 adjoint links
def _quaternion(U):
    """U = a0 + i a.sigma  ->  a0 [n], a [n,3]  (A14)"""
    a0 = U[..., 0, 0].real
    a = np.stack([U[..., 0, 1].imag, U[..., 0, 1].real, U[..., 0, 0].imag], axis=-1)
    return a0, a


def test_P6_P7_P8_adjoint(orc):
    U1 = inputs.haar_su2(500, 1, inputs.FIELD_GAUGE)
    U2 = inputs.haar_su2(500, 7, inputs.FIELD_GAUGE)
    R1, mi = orc.represent(U1)
    R2, _ = orc.represent(U2)
    assert mi < 1e-15
    eye = np.eye(3)
    # P6 orthogonal, det +1
    assert np.abs(R1 @ np.swapaxes(R1, -1, -2) - eye).max() < 1e-14
    assert np.abs(np.linalg.det(R1) - 1.0).max() < 1e-14
    # P7 homomorphism
    R12, _ = orc.represent(U1 @ U2)
    assert np.abs(R12 - R1 @ R2).max() < 1e-14
    Rd, _ = orc.represent(dagger(U1))
    assert np.abs(Rd - np.swapaxes(R1, -1, -2)).max() < 1e-15
    Rm, _ = orc.represent(-U1)
    assert np.abs(Rm - R1).max() < 1e-15
    # P8 orientation: U sigma_b U^dag = sum_a sigma_a R_ab
    lhs = np.einsum("nij,bjk,nkl->nbil", U1, PAULI, dagger(U1))
    rhs = np.einsum("aij,nab->nbij", PAULI, R1)
    assert np.abs(lhs - rhs).max() < 1e-14
    # closed form (O4): R_ab = (a0^2 - |a|^2) d_ab + 2 a_a a_b + 2 a0 eps_abc a_c
    a0, a = _quaternion(U1)
    eps = np.zeros((3, 3, 3))
    eps[0, 1, 2] = eps[1, 2, 0] = eps[2, 0, 1] = 1.0
    eps[0, 2, 1] = eps[2, 1, 0] = eps[1, 0, 2] = -1.0
    cf = ((a0 ** 2 - (a * a).sum(-1))[:, None, None] * eye + 2.0 * a[:, :, None] * a[:, None, :]
          + 2.0 * a0[:, None, None] * np.einsum("abc,nc->nab", eps, a))
    assert np.abs(cf - R1).max() < 1e-14
    # identity and a rotation about axis 3 by angle 2*theta: U = exp(i theta sigma_3)
    Rid, _ = orc.represent(np.eye(2, dtype=np.complex128)[None])
    assert np.array_equal(Rid[0], eye)
    th = 0.37
    Rz, _ = orc.represent(np.diag([np.exp(1j * th), np.exp(-1j * th)])[None])
    c, s = np.cos(2 * th), np.sin(2 * th)
    assert np.abs(Rz[0] - np.array([[c, s, 0], [-s, c, 0], [0, 0, 1]])).max() < 1e-15


# ---------------------------------------------------------------- P10 clover structure
def test_P10_clover_structure(orc):
    L = (4, 4, 4, 4)
    U = inputs.haar_gauge(L, seed=1)
    g = inputs.haar_sites(L, seed=4)
    Ug = gauge_transform(U, g, L)
    for mu in range(4):
        for nu in range(4):
            if mu == nu:
                continue
            F = orc.field_strength(L, U, mu, nu)
            assert np.abs(F + dagger(F)).max() < 1e-15                       # anti-hermitian
            assert np.abs(np.trace(F, axis1=-1, axis2=-2)).max() < 1e-15       # traceless
            assert np.abs(F + orc.field_strength(L, U, nu, mu)).max() < 1e-15  # antisymmetric in mu,nu
            Fg = orc.field_strength(L, Ug, mu, nu)
            assert np.abs(Fg - g @ F @ dagger(g)).max() < 1e-14                # covariant at x
    C = orc.clover_dense(L, 0.0, 1.0, U)
    assert np.abs(C - dagger(C)).max() < 1e-15
    assert np.abs(np.trace(C, axis1=-1, axis2=-2)).max() < 1e-14
    g5 = np.kron(G5, np.eye(2))
    assert np.abs(C @ g5 - g5 @ C).max() < 1e-15
    assert np.abs(C[:, :4, 4:]).max() < 1e-15 and np.abs(C[:, 4:, :4]).max() < 1e-15
    # pure gauge links U_mu(x) = g(x) g(x+mu)^dag  =>  C = 0
    Upure = gauge_transform(inputs.unit_gauge(L), g, L)
    assert np.abs(orc.clover_dense(L, 0.0, 1.0, Upure)).max() < 1e-14


def test_O6_block_formula(orc):
    """A+- = (4+m0) + (csw/2)[tau1 x i(+-F01 - F23) + tau2 x i(+-F02 + F13) + tau3 x i(+-F03 - F12)]."""
    L = (4, 4, 4, 4)
    m0, csw = -0.25, 1.2
    U = inputs.weak_gauge(L, 0.3, seed=1)
    A = orc.clover_dense(L, 4.0 + m0, csw, U)
    F = {(m, n): orc.field_strength(L, U, m, n) for m in range(4) for n in range(m + 1, 4)}
    for sign, sl in ((+1, slice(0, 4)), (-1, slice(4, 8))):
        blk = (4.0 + m0) * np.eye(4)[None] + 0.5 * csw * (
            np.einsum("st,xcd->xsctd", PAULI[0], 1j * (sign * F[0, 1] - F[2, 3])).reshape(-1, 4, 4)
            + np.einsum("st,xcd->xsctd", PAULI[1], 1j * (sign * F[0, 2] + F[1, 3])).reshape(-1, 4, 4)
            + np.einsum("st,xcd->xsctd", PAULI[2], 1j * (sign * F[0, 3] - F[1, 2])).reshape(-1, 4, 4))
        assert np.abs(A[:, sl, sl] - blk).max() < 1e-15


# ---------------------------------------------------------------- P11 abelian closed form
def test_P11_abelian_closed_form(orc):
    L = (4, 6, 4, 4)
    V = inputs.volume(L)
    rng = np.random.default_rng(5)
    phi = rng.uniform(-np.pi, np.pi, size=(V, 4))
    U = np.zeros((V, 4, 2, 2), dtype=np.complex128)
    U[..., 0, 0] = np.exp(1j * phi)
    U[..., 1, 1] = np.exp(-1j * phi)
    ph = grid(phi, L)
    for mu in range(4):
        for nu in range(4):
            if mu == nu:
                continue
            P = ph[..., mu] + fwd(ph[..., nu], mu) - fwd(ph[..., mu], nu) - ph[..., nu]
            S = np.sin(P) + np.sin(bwd(P, mu)) + np.sin(bwd(bwd(P, mu), nu)) + np.sin(bwd(P, nu))
            expect = (0.25j * S)[..., None, None] * PAULI[2]
            F = orc.field_strength(L, U, mu, nu)
            assert np.abs(F - flat(expect, L)).max() < 1e-15


# ---------------------------------------------------------------- P12 sign of the clover term
def test_P12_clover_sign(orc):
    """Tree-level improvement identity: -1/2 sum_{mu!=nu} g_mu g_nu Dl_mu Dl_nu psi ~ C psi (c_sw = 1),
    Dl = symmetric covariant difference; residual is the O(k^2) lattice artefact."""
    L = (12, 12, 12, 12)
    V = inputs.volume(L)
    k = 2.0 * np.pi / 12.0
    x = inputs.site_coords(L).astype(np.float64)
    rng = np.random.default_rng(3)
    q = np.zeros((V, 4, 4))
    for mu in range(4):
        f = np.empty((V, 3))
        for c in range(3):
            n = rng.integers(0, 2, size=4)
            f[:, c] = 0.2 * np.cos(k * (x @ n) + rng.uniform(0, 2 * np.pi))
        r = np.sqrt((f * f).sum(-1))
        q[:, mu, 0] = np.cos(r)
        q[:, mu, 1:] = f * (np.sin(r) / r)[:, None]
    U = np.empty((V, 4, 2, 2), dtype=np.complex128)
    inputs._quaternion_to_su2(q, U)
    w = rng.normal(size=(4, 2)) + 1j * rng.normal(size=(4, 2))
    psi = (np.cos(k * x[:, 0] + 0.3) * np.sin(k * (x[:, 1] + x[:, 2])))[:, None, None] * w[None]

    Ug = grid(U, L)

    def cdiff(v, mu):
        u = Ug[..., mu, :, :]
        f = np.einsum("...cd,...sd->...sc", u, fwd(v, mu))
        b = bwd(np.einsum("...dc,...sd->...sc", np.conj(u), v), mu)
        return 0.5 * (f - b)

    p = grid(psi, L)
    lhs = np.zeros_like(p)
    for mu in range(4):
        for nu in range(4):
            if mu != nu:
                lhs += -0.5 * np.einsum("st,...tc->...sc", GAM[mu] @ GAM[nu], cdiff(cdiff(p, nu), mu))
    lhs = flat(lhs, L)
    C = orc.clover_dense(L, 0.0, 1.0, U)
    Cpsi = orc.site_matvec(L, 3, C, psi)
    nC = np.linalg.norm(Cpsi)
    assert np.linalg.norm(lhs - Cpsi) < 0.5 * nC
    assert np.linalg.norm(lhs + Cpsi) > 1.5 * nC


# ---------------------------------------------------------------- P13 inverse
def test_P13_clover_inverse(orc):
    L = (4, 4, 4, 4)
    U = inputs.weak_gauge(L, 0.3, seed=1)
    A = orc.clover_dense(L, 4.0 - 0.25, 1.2, U)
    Ainv = orc.invert(A)
    assert np.abs(A @ Ainv - np.eye(8)).max() < 1e-14
    assert np.abs(Ainv - np.linalg.inv(A)).max() < 1e-14
    ev = np.linalg.eigvalsh(A[:, :4, :4])
    # each chirality block of C is traceless (tr tau_k = 0): eigenvalues average to 4+m0 exactly;
    # SURVEY P13 saw [2.7, 4.8] with its own random field at these parameters: same scale here
    assert np.abs(ev.mean(axis=1) - 3.75).max() < 1e-14
    assert ev.min() > 2.4 and ev.max() < 5.1 and (ev.max(axis=1) / ev.min(axis=1)).max() < 2.0
    # the generic inverse on a matrix that needs pivoting
    M = np.array([[[0, 2], [3, 1]]], dtype=np.complex128)
    assert np.abs(orc.invert(M) - np.linalg.inv(M)).max() < 1e-15


# ---------------------------------------------------------------- threads give the same bits
def test_threads_bitwise_identical(orc):
    L = (4, 4, 4, 6)
    U = inputs.haar_gauge(L, seed=1)
    psi = inputs.gaussian_spinor(L, 2, seed=2)
    a = orc.dirac(L, 0, -0.2, U, psi, nthreads=1)
    b = orc.dirac(L, 0, -0.2, U, psi, nthreads=3)
    assert np.array_equal(a, b)
    assert np.array_equal(orc.dirac_eo(L, 0, -0.2, U, psi, 1), orc.dirac_eo(L, 0, -0.2, U, psi, 4))


def test_P15_cg_against_dense_solve(orc):
    """O8: the CG solution of Dhat^dag Dhat x = b equals the dense solve of the same system, whose matrix is
    assembled column by column from the oracle's Dhat (2 x 4 x 2 x 2 lattice: 256 even-site unknowns) and
    solved by LAPACK — a route that shares nothing with the iteration."""
    L, m0 = (2, 4, 2, 2), -0.2
    U = inputs.haar_gauge(L, 1)
    V = inputs.volume(L)
    even = inputs.site_parity(L) == 0
    n = int(even.sum()) * 8
    Dh = np.zeros((n, n), dtype=np.complex128)
    e = np.zeros((V, 4, 2), dtype=np.complex128)
    for j in range(n):
        col = np.zeros(n, dtype=np.complex128)
        col[j] = 1.0
        e[even] = col.reshape(-1, 4, 2)
        Dh[:, j] = orc.dirac_eo(L, 0, m0, U, e)[even].ravel()
    b = inputs.gaussian_spinor(L, 2, 2)
    b[~even] = 0
    x_dense = np.linalg.solve(Dh.conj().T @ Dh, b[even].ravel())
    x, it, relres = orc.cg_normal(L, 0, m0, U, b, tol=1e-13, max_iter=500)
    assert relres <= 1e-13 and 0 < it < 200
    assert not x[~even].any()
    assert np.linalg.norm(x[even].ravel() - x_dense) <= 1e-11 * np.linalg.norm(x_dense)
    # and Dhat^dag really is gamma5 Dhat gamma5 (used by O8): compare with the dense adjoint on a random vector
    v = inputs.gaussian_spinor(L, 2, 3, inputs.FIELD_SPINOR2)
    v[~even] = 0
    g5 = np.array([1.0, 1.0, -1.0, -1.0])[None, :, None]
    lhs = (g5 * orc.dirac_eo(L, 0, m0, U, g5 * v))[even].ravel()
    assert np.linalg.norm(lhs - Dh.conj().T @ v[even].ravel()) <= 1e-13 * np.linalg.norm(lhs)


def test_P16_exponential_clover(orc):
    """O9: A_exp = d exp(C/d).  Pins: the same matrix from scipy's Pade expm (another route); det A_exp = d^8 exactly
    because tr C = 0; A_exp A_exp^-1 = 1; hermitian, commuting with gamma5; A_exp - (d + C) = C^2/(2d) + O(C^3)
    (the regular clover term is its first two orders): the difference scales as csw^2 and matches C^2/(2d) to
    the next order; csw = 0 gives d * 1."""
    from scipy.linalg import expm
    L, m0 = (4, 4, 2, 2), -0.25
    d = 4.0 + m0
    U = inputs.weak_gauge(L, 0.3, 1)
    V = inputs.volume(L)
    eye = np.eye(8)[None]
    fwd, inv = orc.clover_exp_dense(L, d, 1.2, U)
    C = orc.clover_dense(L, d, 1.2, U) - d * eye
    for x in (0, 7, V - 1):
        assert np.abs(fwd[x] - d * expm(C[x] / d)).max() <= 1e-13
        assert np.abs(inv[x] - expm(-C[x] / d) / d).max() <= 1e-14
    assert np.abs(np.linalg.det(fwd) - d ** 8).max() <= 1e-9 * d ** 8
    assert np.abs(fwd @ inv - eye).max() <= 1e-14
    assert np.abs(fwd - np.conj(np.swapaxes(fwd, -1, -2))).max() <= 1e-14
    g5 = np.diag([1, 1, 1, 1, -1, -1, -1, -1]).astype(complex)
    assert np.abs(g5 @ fwd - fwd @ g5).max() <= 1e-14
    # series: A_exp - (d + C) - C^2/(2d) = O(C^3/d^2)
    rem2 = fwd - (d * eye + C)
    rem3 = rem2 - C @ C / (2 * d)
    nC = np.abs(C).max()
    assert np.abs(rem2).max() <= 2.0 * nC ** 2 / d and np.abs(rem3).max() <= 2.0 * nC ** 3 / d ** 2
    fwd_half, _ = orc.clover_exp_dense(L, d, 0.6, U)
    rem2_half = fwd_half - (d * eye + 0.5 * C)
    ratio = np.abs(rem2).max() / np.abs(rem2_half).max()
    assert 3.5 < ratio < 4.7          # quadratic in csw
    f0, i0 = orc.clover_exp_dense(L, d, 0.0, U)
    assert np.abs(f0 - d * eye).max() <= 1e-14 and np.abs(i0 - eye / d).max() <= 1e-15


def test_P17_adjoint_clover(orc):
    """O10.  (a) leaves: for every site of a 2x2x2x4 lattice and every plane, the sum of the four FUNDAMENTAL leaves,
    multiplied out here with explicit (x +- mu) mod L site arithmetic and mapped leaf by leaf through O4 (R is a
    homomorphism, pin P7), gives the adjoint Q whose antisymmetric part O10 uses — paths, orientation, transposes;
    (b) C hermitian, traceless, commuting with gamma5; (c) gauge covariance C[U^g](x) = R(g(x)) C(x) R(g(x))^T on
    colour; (d) abelian links exp(i phi sigma3): R is a rotation by 2 phi about axis 3 and
    F^_mu,nu = (1/4) J3 sum_leaves sin(2 P_leaf), J3 = [[0,-1,0],[1,0,0],[0,0,0]]... sign fixed by O4's orientation."""
    L = (2, 2, 2, 4)
    V = inputs.volume(L)
    U = inputs.haar_gauge(L, 1)
    R, _ = orc.represent(U)
    gam = orc.gamma()
    x_of = inputs.site_coords(L)

    def lex(x):
        return ((x[0] % L[0] * L[1] + x[1] % L[1]) * L[2] + x[2] % L[2]) * L[3] + x[3] % L[3]

    def u(x, mu, dag=False):
        m = U[lex(x), mu]
        return m.conj().T if dag else m

    def e(mu):
        v = np.zeros(4, dtype=int)
        v[mu] = 1
        return v

    d, csw = 3.7, 1.3
    A = orc.clover_dense_adj(L, d, csw, R)
    for s in range(0, V, 5):
        x = x_of[s]
        C = np.zeros((12, 12), dtype=complex)
        for mu in range(4):
            for nu in range(mu + 1, 4):
                m, n = e(mu), e(nu)
                leaves = [u(x, mu) @ u(x + m, nu) @ u(x + n, mu, True) @ u(x, nu, True),
                          u(x, nu) @ u(x - m + n, mu, True) @ u(x - m, nu, True) @ u(x - m, mu),
                          u(x - m, mu, True) @ u(x - m - n, nu, True) @ u(x - m - n, mu) @ u(x - n, nu),
                          u(x - n, nu, True) @ u(x - n, mu) @ u(x + m - n, nu) @ u(x, mu, True)]
                Q = sum(orc.represent(np.array([[[p]]]).reshape(1, 1, 2, 2))[0][0, 0] for p in leaves)
                F = (Q - Q.T) / 8.0
                sig = 0.5j * (gam[mu] @ gam[nu] - gam[nu] @ gam[mu])
                C += csw * 0.5j * np.kron(sig, F)
        assert np.abs(A[s] - d * np.eye(12) - C).max() <= 1e-13
    # (b)
    Cf = A - d * np.eye(12)[None]
    assert np.abs(Cf - np.conj(np.swapaxes(Cf, -1, -2))).max() <= 1e-15
    assert np.abs(np.trace(Cf, axis1=1, axis2=2)).max() <= 1e-14
    g5 = np.kron(np.diag([1, 1, -1, -1]), np.eye(3)).astype(complex)
    assert np.abs(g5 @ Cf - Cf @ g5).max() <= 1e-15
    # (c)
    g = inputs.haar_sites(L, 4)
    Rg_links, _ = orc.represent(gauge_transform(U, g, L))
    Rg = orc.represent(g.reshape(V, 1, 2, 2))[0][:, 0]
    big = np.einsum("st,xab->xsatb", np.eye(4), Rg).reshape(V, 12, 12)
    Cg = orc.clover_dense_adj(L, 0.0, csw, Rg_links)
    assert np.abs(Cg - big @ Cf @ np.swapaxes(big, -1, -2)).max() <= 1e-13
    # (d) abelian: U_mu(x) = exp(i phi_mu(x) sigma3)
    phi = 0.4 * inputs.normals(11, 9, 0, V * 4).reshape(L + (4,))
    Uab = np.zeros((V, 4, 2, 2), dtype=complex)
    Uab[:, :, 0, 0] = np.exp(1j * phi.reshape(V, 4))
    Uab[:, :, 1, 1] = np.exp(-1j * phi.reshape(V, 4))
    Rab, _ = orc.represent(Uab)
    Aab = orc.clover_dense_adj(L, 0.0, 1.0, Rab)
    # the rotation angle of R(exp(i t sigma3)) about axis 3: read it off O4 itself on one link, then use it for the sum
    t = 0.3
    R1 = orc.represent(np.diag([np.exp(1j * t), np.exp(-1j * t)]).reshape(1, 1, 2, 2))[0][0, 0]
    J = (R1 - R1.T) / (2 * np.sin(2 * t))           # = +-J3 with the sign O4's orientation gives
    assert np.abs(np.abs(J) - np.array([[0, 1, 0], [1, 0, 0], [0, 0, 0]])).max() <= 1e-14
    for mu in range(4):
        for nu in range(mu + 1, 4):
            P = phi[..., mu] + np.roll(phi[..., nu], -1, mu) - np.roll(phi[..., mu], -1, nu) - phi[..., nu]
            S = np.sin(2 * P) + np.sin(2 * np.roll(P, 1, mu)) + np.sin(2 * np.roll(np.roll(P, 1, mu), 1, nu)) + np.sin(2 * np.roll(P, 1, nu))
            Fcf = (S.reshape(V)[:, None, None] / 4.0) * J[None]
            # extract F^_mu,nu from the oracle: C = (i/2) sum sigma (x) F; project with sigma_mu,nu (tr sigma_a sigma_b = 4 delta)
            sig = 0.5j * (gam[mu] @ gam[nu] - gam[nu] @ gam[mu])
            Fo = np.einsum("ts,xsatb->xab", sig, Aab.reshape(V, 4, 3, 4, 3)) / 4.0 / 0.5j
            assert np.abs(Fo - Fcf).max() <= 1e-13, (mu, nu)


def _site_loop_matvec(M, psi):
    """out[x] = M[x] psi[x], one site at a time with the @ operator (row index of M first) — the plain definition the
    two oracle mat-vec routines are pinned to"""
    out = np.empty_like(psi)
    for x in range(psi.shape[0]):
        out[x] = (M[x] @ psi[x].reshape(-1)).reshape(psi.shape[1:])
    return out


def test_P20_site_matvec_orientation(orc):
    """orc_site_matvec (C++) and site_matvec_n (numpy): out[x]_i = sum_j M[x]_ij psi[x]_j with NON-hermitian random
    site matrices (a transposed mat-vec passes every identity that only uses hermitian matrices consistently; it
    fails here), the parity bit mask of orc_site_matvec (bit 0 even sites, bit 1 odd sites) and the mask of
    site_matvec_n"""
    L = (2, 4, 2, 4)
    V = inputs.volume(L)
    par = inputs.site_parity(L)
    for N, n in ((2, 8), (3, 12)):
        M = (inputs.normals(21, 5, 0, V * n * n) + 1j * inputs.normals(22, 5, 0, V * n * n)).reshape(V, n, n)
        psi = inputs.gaussian_spinor(L, N, 2)
        want = _site_loop_matvec(M, psi)
        got_n = orc.site_matvec_n(M, psi)
        assert np.abs(got_n - want).max() <= 1e-13
        assert np.abs(got_n - _site_loop_matvec(np.swapaxes(M, -1, -2), psi)).max() > 1.0     # the transpose is far away
        odd = par == 1
        got_odd = orc.site_matvec_n(M, psi, odd)
        assert np.abs(got_odd[odd] - want[odd]).max() <= 1e-13 and not got_odd[~odd].any()
        if N == 2:
            both = orc.site_matvec(L, 3, M, psi)
            assert np.abs(both - want).max() <= 1e-13
            for mask, sel in ((1, par == 0), (2, par == 1)):
                got = orc.site_matvec(L, mask, M, psi)
                assert np.abs(got[sel] - want[sel]).max() <= 1e-13 and not got[~sel].any()


def test_P18_adjoint_clover_schur_identity(orc):
    """O7 in the adjoint representation (oracle.dirac_eo_clover_adj), pinned by the Schur identity P4: with
    eta = D_sw x on all sites (D_sw = D[R] + C, the full operator O1 in the adjoint representation plus the O10
    clover term applied site by site here),
        Dhat x_e = eta_e - D_eo A_oo^-1 eta_o = eta_e + 1/2 H_eo A_oo^-1 eta_o        (D_eo = -1/2 H_eo).
    A wrong constant (-1/2 for -1/4), a swapped parity mask or A for A^-1 fails this; gamma5-hermiticity of Dhat
    (P2) and the equivalent full solve on a 2^4 lattice (P5) ride along."""
    L = (2, 4, 2, 4)
    m0, csw = -0.25, 1.2
    d = 4.0 + m0
    Uf = inputs.weak_gauge(L, 0.3, seed=1)
    R, _ = orc.represent(Uf)
    par = inputs.site_parity(L)
    even, odd = par == 0, par == 1
    A = orc.clover_dense_adj(L, d, csw, R)
    C = A - d * np.eye(12)[None]
    Ainv = np.linalg.inv(A)
    x = inputs.gaussian_spinor(L, 3, seed=2)
    eta = orc.dirac(L, 1, m0, R, x) + _site_loop_matvec(C, x)
    t = np.where(odd[:, None, None], _site_loop_matvec(Ainv, eta), 0.0)
    rhs = np.where(even[:, None, None], eta, 0.0) + 0.5 * orc.hop(L, 1, 0, R, t)
    lhs = orc.dirac_eo_clover_adj(L, R, A, Ainv, x)
    assert rel_l2(lhs, rhs) < 1e-14
    assert not lhs[odd].any()
    # the other half of the identity: x_o = A_oo^-1 (eta_o + 1/2 H_oe x_e)
    xe = np.where(even[:, None, None], x, 0.0)
    xo = _site_loop_matvec(Ainv, np.where(odd[:, None, None], eta + 0.5 * orc.hop(L, 1, 1, R, xe), 0.0))
    assert rel_l2(xo[odd], x[odd]) < 1e-14
    # P2: <chi, Dhat psi> = <gamma5 Dhat gamma5 chi, psi> on even-supported vectors
    g5 = np.array([1.0, 1.0, -1.0, -1.0])[None, :, None]
    chi = np.where(even[:, None, None], inputs.gaussian_spinor(L, 3, 3, inputs.FIELD_SPINOR2), 0.0)
    a = inner(chi, orc.dirac_eo_clover_adj(L, R, A, Ainv, xe))
    b = inner(g5 * orc.dirac_eo_clover_adj(L, R, A, Ainv, g5 * chi), xe)
    assert abs(a - b) <= 1e-13 * abs(a)
    # P5 on 2^4: dense D_sw (192 unknowns) solved by LAPACK; its even part solves the Schur system
    L2 = (2, 2, 2, 2)
    V2 = 16
    U2 = inputs.weak_gauge(L2, 0.3, seed=1)
    R2, _ = orc.represent(U2)
    A2 = orc.clover_dense_adj(L2, d, csw, R2)
    A2inv = np.linalg.inv(A2)
    C2 = A2 - d * np.eye(12)[None]
    n = V2 * 12
    Dsw = np.empty((n, n), dtype=np.complex128)
    for k in range(n):
        e = np.zeros(n, dtype=np.complex128)
        e[k] = 1.0
        e = e.reshape(V2, 4, 3)
        Dsw[:, k] = (orc.dirac(L2, 1, m0, R2, e) + _site_loop_matvec(C2, e)).ravel()
    eta2 = inputs.gaussian_spinor(L2, 3, seed=2)
    x2 = np.linalg.solve(Dsw, eta2.ravel()).reshape(V2, 4, 3)
    ev2 = (inputs.site_parity(L2) == 0)[:, None, None]
    t2 = np.where(~ev2, _site_loop_matvec(A2inv, eta2), 0.0)
    rhs2 = np.where(ev2, eta2, 0.0) + 0.5 * orc.hop(L2, 1, 0, R2, t2)
    assert rel_l2(orc.dirac_eo_clover_adj(L2, R2, A2, A2inv, x2), rhs2) < 1e-13


def test_P19_adjoint_exponential_clover(orc):
    """O11 (oracle.clover_exp_dense_adj): A_exp = d exp(C/d) on the 12x12 adjoint clover term.  Pins as P16: scipy's
    Pade expm on three sites (another route), det A_exp = d^12 exactly (tr C = 0), A_exp A_exp^-1 = 1, hermitian,
    commuting with gamma5, A_exp - (d + C) = C^2/(2d) + O(C^3) scaling as csw^2, and csw = 0 gives d * 1."""
    from scipy.linalg import expm
    L, m0 = (4, 2, 2, 2), -0.25
    d = 4.0 + m0
    R, _ = orc.represent(inputs.weak_gauge(L, 0.3, 1))
    V = inputs.volume(L)
    eye = np.eye(12)[None]
    fwd, inv = orc.clover_exp_dense_adj(L, d, 1.2, R)
    C = orc.clover_dense_adj(L, 0.0, 1.2, R)
    for x in (0, 5, V - 1):
        assert np.abs(fwd[x] - d * expm(C[x] / d)).max() <= 1e-13
        assert np.abs(inv[x] - expm(-C[x] / d) / d).max() <= 1e-14
    assert np.abs(np.linalg.det(fwd) - d ** 12).max() <= 1e-9 * d ** 12
    assert np.abs(fwd @ inv - eye).max() <= 1e-14
    assert np.abs(fwd - np.conj(np.swapaxes(fwd, -1, -2))).max() <= 1e-14
    g5 = np.kron(np.diag([1, 1, -1, -1]), np.eye(3)).astype(complex)
    assert np.abs(g5 @ fwd - fwd @ g5).max() <= 1e-14
    rem2 = fwd - (d * eye + C)
    rem3 = rem2 - C @ C / (2 * d)
    nC = np.abs(C).max()
    assert np.abs(rem2).max() <= 3.0 * nC ** 2 / d and np.abs(rem3).max() <= 4.0 * nC ** 3 / d ** 2
    fwd_half, _ = orc.clover_exp_dense_adj(L, d, 0.6, R)
    ratio = np.abs(rem2).max() / np.abs(fwd_half - (d * eye + 0.5 * C)).max()
    assert 3.5 < ratio < 4.7          # quadratic in csw
    f0, i0 = orc.clover_exp_dense_adj(L, d, 0.0, R)
    assert np.abs(f0 - d * eye).max() <= 1e-14 and np.abs(i0 - eye / d).max() <= 1e-15


# ---------------------------------------------------------------- P21: complex 3x3 links (rep 2, e.g. SU(3) fundamental)
def test_P21_complex_3x3_links(orc):
    """oracle rep 2 (complex 3 x 3 links, 3 complex colours): the same pins that hold
    O1-O3 for SU(2) — P1 plane wave at U = 1, P2 gamma5-hermiticity, P3 gauge covariance under a random local SU(3)
    transformation, P4 Schur identity, P9 hop = off-diagonal part of D, P14 an independent numpy restatement — and, as the
    special case that ties the new link format to the pinned one, SU(2) links embedded in the upper-left 2 x 2 block of a
    3 x 3 matrix (third colour decoupled): colours 0, 1 must reproduce the rep-0 operator, colour 2 the free one."""
    L = (4, 4, 2, 6)
    V = inputs.volume(L)
    m0 = -0.2
    d = 4.0 + m0
    U = inputs.haar_gauge_su3(L, 1)
    assert np.abs(U @ dagger(U) - np.eye(3)).max() < 1e-14 and np.abs(np.linalg.det(U) - 1.0).max() < 1e-13
    psi = inputs.gaussian_spinor(L, 3, 2)
    chi = inputs.gaussian_spinor(L, 3, 3, inputs.FIELD_SPINOR2)
    D = lambda v, links=U: orc.dirac(L, 2, m0, links, v)
    # P14: independent restatement (whole-lattice shifts, dense gamma matrices)
    assert rel_l2(D(psi), wilson_dirac_numpy(L, U, psi, m0, GAM)) < 1e-14
    # P2
    g5 = np.array([1.0, 1.0, -1.0, -1.0])[None, :, None]
    a, b = inner(chi, D(psi)), inner(g5 * D(g5 * chi), psi)
    assert abs(a - b) <= 1e-14 * abs(a)
    # P3: U^g_mu(x) = g(x) U_mu(x) g(x+mu)^dag, D[U^g](g psi) = g D[U] psi
    g = inputs.haar_sites_su3(L, 4)
    Ug = gauge_transform(U, g, L)
    gpsi = np.einsum("xab,xsb->xsa", g, psi)
    assert rel_l2(D(gpsi, Ug), np.einsum("xab,xsb->xsa", g, D(psi))) < 1e-14
    # P9 + P4
    par = inputs.site_parity(L)
    even = (par == 0)[:, None, None]
    eta = D(psi)
    H = orc.hop(L, 2, 0, U, psi)
    H = orc.hop(L, 2, 1, U, psi, out=H)
    assert rel_l2(eta, d * psi - 0.5 * H) < 1e-14
    rhs = eta * even + 0.5 / d * orc.hop(L, 2, 0, U, eta * ~even)
    assert rel_l2(orc.dirac_eo(L, 2, m0, U, psi), rhs) < 1e-14
    # P1: U = 1, plane wave
    n = np.array([1, 0, 1, 2])
    p = 2 * np.pi * n / np.array(L)
    x = inputs.site_coords(L)
    w = inputs.normals(5, 7, 0, 24).reshape(4, 3, 2)
    w = w[..., 0] + 1j * w[..., 1]
    wave = np.exp(1j * (x @ p))[:, None, None] * w[None]
    one = np.broadcast_to(np.eye(3, dtype=np.complex128), (V, 4, 3, 3)).copy()
    M = (m0 + np.sum(1 - np.cos(p))) * np.eye(4) + 1j * sum(np.sin(p[mu]) * GAM[mu] for mu in range(4))
    want = np.exp(1j * (x @ p))[:, None, None] * np.einsum("st,tc->sc", M, w)[None]
    assert rel_l2(orc.dirac(L, 2, m0, one, wave), want) < 1e-14
    # embedded SU(2): block-diagonal links diag(U2, 1)
    U2 = inputs.haar_gauge(L, 1)
    emb = np.zeros((V, 4, 3, 3), dtype=np.complex128)
    emb[..., :2, :2] = U2
    emb[..., 2, 2] = 1.0
    got = orc.dirac(L, 2, m0, emb, psi)
    assert rel_l2(got[..., :2], orc.dirac(L, 0, m0, U2, np.ascontiguousarray(psi[..., :2]))) < 1e-14
    free = orc.dirac(L, 2, m0, one, psi)
    assert rel_l2(got[..., 2], free[..., 2]) < 1e-14


def test_P22_su3_clover(orc):
    """O12 (clover term for complex 3 x 3 links) and dirac_eo_clover_n(rep = 2).  (a) SU(2) links embedded in the upper-left 2 x 2
    block of a 3 x 3 unit matrix: the colour-(0,1) sub-block of O12 must be the FUNDAMENTAL SU(2) clover term of the C++ oracle
    (O5/O6, explicit site loops — an independent implementation) and colour 2 must see the bare diagonal; (b) every site of a
    Haar SU(3) field against leaves multiplied out here with explicit (x +- mu) mod L site arithmetic; (c) C hermitian,
    traceless, commuting with gamma5; (d) gauge covariance under SU(3); (e) abelian links diag(e^{i a}, e^{i b}, e^{-i(a+b)}):
    F^_mu,nu = (i/4) diag(sum over the four leaves of sin(plaquette angle)) per colour; (f) the Schur identity P4 for
    dirac_eo_clover_n with D_sw = D[U] + C applied site by site here."""
    L = (2, 2, 2, 4)
    V = inputs.volume(L)
    gam = orc.gamma()
    d, csw = 3.7, 1.3
    # (a)
    U2 = inputs.haar_gauge(L, 1)
    U3 = np.zeros((V, 4, 3, 3), dtype=complex)
    U3[:, :, :2, :2] = U2
    U3[:, :, 2, 2] = 1.0
    A3 = orc.clover_dense_su3(L, d, csw, U3).reshape(V, 4, 3, 4, 3)
    A2 = orc.clover_dense(L, d, csw, U2).reshape(V, 4, 2, 4, 2)
    assert np.abs(A3[:, :, :2, :, :2] - A2).max() <= 1e-13
    assert np.abs(A3[:, :, 2, :, 2] - d * np.eye(4)[None]).max() <= 1e-14
    assert np.abs(A3[:, :, :2, :, 2]).max() == 0 and np.abs(A3[:, :, 2, :, :2]).max() == 0
    # (b)
    U = inputs.haar_gauge_su3(L, 1)
    x_of = inputs.site_coords(L)

    def lex(x):
        return ((x[0] % L[0] * L[1] + x[1] % L[1]) * L[2] + x[2] % L[2]) * L[3] + x[3] % L[3]

    def u(x, mu, dag=False):
        m = U[lex(x), mu]
        return m.conj().T if dag else m

    def e(mu):
        v = np.zeros(4, dtype=int)
        v[mu] = 1
        return v

    A = orc.clover_dense_su3(L, d, csw, U)
    for s_ in range(0, V, 3):
        x = x_of[s_]
        C = np.zeros((12, 12), dtype=complex)
        for mu in range(4):
            for nu in range(mu + 1, 4):
                m, n = e(mu), e(nu)
                Q = (u(x, mu) @ u(x + m, nu) @ u(x + n, mu, True) @ u(x, nu, True)
                     + u(x, nu) @ u(x - m + n, mu, True) @ u(x - m, nu, True) @ u(x - m, mu)
                     + u(x - m, mu, True) @ u(x - m - n, nu, True) @ u(x - m - n, mu) @ u(x - n, nu)
                     + u(x - n, nu, True) @ u(x - n, mu) @ u(x + m - n, nu) @ u(x, mu, True))
                F = (Q - Q.conj().T) / 8.0
                sig = 0.5j * (gam[mu] @ gam[nu] - gam[nu] @ gam[mu])
                C += csw * 0.5j * np.kron(sig, F)
        assert np.abs(A[s_] - d * np.eye(12) - C).max() <= 1e-13
    # (c)
    Cf = A - d * np.eye(12)[None]
    assert np.abs(Cf - np.conj(np.swapaxes(Cf, -1, -2))).max() <= 1e-15
    assert np.abs(np.trace(Cf, axis1=1, axis2=2)).max() <= 1e-14
    g5 = np.kron(np.diag([1, 1, -1, -1]), np.eye(3)).astype(complex)
    assert np.abs(g5 @ Cf - Cf @ g5).max() <= 1e-15
    # (d) U'_mu(x) = g(x) U_mu(x) g(x+mu)^dag  ->  C'(x) = g(x) C(x) g(x)^dag on colour
    g = inputs.haar_sites_su3(L, 4)
    Ug = np.empty_like(U)
    gl = g.reshape(L + (3, 3))
    for mu in range(4):
        gs = np.roll(gl, -1, axis=mu).reshape(V, 3, 3)
        Ug[:, mu] = g @ U[:, mu] @ np.conj(np.swapaxes(gs, -1, -2))
    big = np.einsum("st,xab->xsatb", np.eye(4), g).reshape(V, 12, 12)
    Cg = orc.clover_dense_su3(L, 0.0, csw, Ug)
    assert np.abs(Cg - big @ Cf @ np.conj(np.swapaxes(big, -1, -2))).max() <= 1e-13
    # (e)
    ph = 0.4 * inputs.normals(11, 9, 0, V * 8).reshape(L + (4, 2))
    ang = np.concatenate([ph, -ph.sum(axis=-1, keepdims=True)], axis=-1)          # three colour phases per link, sum 0
    Uab = np.zeros((V, 4, 3, 3), dtype=complex)
    for c in range(3):
        Uab[:, :, c, c] = np.exp(1j * ang[..., c].reshape(V, 4))
    Aab = orc.clover_dense_su3(L, 0.0, 1.0, Uab)
    for mu in range(4):
        for nu in range(mu + 1, 4):
            sig = 0.5j * (gam[mu] @ gam[nu] - gam[nu] @ gam[mu])
            Fo = np.einsum("ts,xsatb->xab", sig, Aab.reshape(V, 4, 3, 4, 3)) / 4.0 / 0.5j
            for c in range(3):
                a = ang[..., c]
                P = a[..., mu] + np.roll(a[..., nu], -1, mu) - np.roll(a[..., mu], -1, nu) - a[..., nu]
                S = np.sin(P) + np.sin(np.roll(P, 1, mu)) + np.sin(np.roll(np.roll(P, 1, mu), 1, nu)) + np.sin(np.roll(P, 1, nu))
                assert np.abs(Fo[:, c, c] - 0.25j * S.reshape(V)).max() <= 1e-13, (mu, nu, c)
            off = Fo.copy()
            off[:, range(3), range(3)] = 0
            assert np.abs(off).max() <= 1e-15
    # (f)
    L4 = (2, 4, 2, 4)
    m0 = -0.25
    dd = 4.0 + m0
    Uw = inputs.haar_gauge_su3(L4, 1)
    par = inputs.site_parity(L4)
    even, odd = par == 0, par == 1
    Aw = orc.clover_dense_su3(L4, dd, 1.2, Uw)
    Cw = Aw - dd * np.eye(12)[None]
    Awinv = np.linalg.inv(Aw)
    x = inputs.gaussian_spinor(L4, 3, seed=2)
    eta = orc.dirac(L4, 2, m0, Uw, x) + _site_loop_matvec(Cw, x)
    t = np.where(odd[:, None, None], _site_loop_matvec(Awinv, eta), 0.0)
    rhs = np.where(even[:, None, None], eta, 0.0) + 0.5 * orc.hop(L4, 2, 0, Uw, t)
    lhs = orc.dirac_eo_clover_n(L4, 2, Uw, Aw, Awinv, x)
    assert rel_l2(lhs, rhs) < 1e-14 and not lhs[odd].any()
    # the exponential pair: scipy's Pade expm on three sites, det = d^12
    import scipy.linalg
    Ae, Aei = orc.clover_exp_dense_su3(L4, dd, 1.2, Uw)
    for s_ in (0, 17, inputs.volume(L4) - 1):
        assert np.abs(Ae[s_] - dd * scipy.linalg.expm(Cw[s_] / dd)).max() <= 1e-12
        assert np.abs(Ae[s_] @ Aei[s_] - np.eye(12)).max() <= 1e-13
    assert np.abs(np.linalg.det(Ae) / dd ** 12 - 1).max() <= 1e-11
    # and the adjoint wrapper is this function
    Uf = inputs.weak_gauge(L4, 0.3, seed=1)
    R, _ = orc.represent(Uf)
    Ar = orc.clover_dense_adj(L4, dd, 1.2, R)
    xa = inputs.gaussian_spinor(L4, 3, seed=2)
    assert np.array_equal(orc.dirac_eo_clover_n(L4, 1, R, Ar, np.linalg.inv(Ar), xa), orc.dirac_eo_clover_adj(L4, R, Ar, np.linalg.inv(Ar), xa))


# ---------------------------------------------------------------- P23: two-index antisymmetric representation of SU(3) (O13)
def test_P23_antisymmetric_representation_su3(orc):
    """O13 against what the mathematics fixes, none of it through the oracle's own formula:
    (i) R(U) is unitary with det 1 and R(1) = 1; (ii) homomorphism R(UV) = R(U) R(V); (iii) character
    tr R(U) = ((tr U)^2 - tr U^2) / 2; (iv) for SU(3) the antisymmetric pair (i,j) is dual to the third index k (epsilon_ijk), so
    R(U) = P conj(U) P^T with the signed permutation P: (0,1) -> +2, (0,2) -> -1, (1,2) -> +0 — an exact closed form;
    (v) a diagonal U = diag(z0, z1, z2) gives diag(z0 z1, z0 z2, z1 z2); (vi) an SU(2) matrix V embedded in the upper-left block acts
    as 1 on the pair (0,1) and as V on the pairs ((0,2), (1,2)); (vii) a non-unitary matrix: the entries are the 2 x 2 minors
    (brute force), which catches a transposed operand that unitarity would hide."""
    rng = np.random.default_rng(23)
    U = inputs.haar_su3(64, 5, 0)
    Vm = inputs.haar_su3(64, 6, 0)
    R = orc.represent_antisym_su3(U)
    I3 = np.eye(3)
    assert np.abs(R @ np.conj(np.swapaxes(R, -1, -2)) - I3).max() < 1e-14
    assert np.abs(np.linalg.det(R) - 1.0).max() < 1e-13
    assert np.abs(orc.represent_antisym_su3(I3) - I3).max() < 1e-15
    assert np.abs(orc.represent_antisym_su3(U @ Vm) - R @ orc.represent_antisym_su3(Vm)).max() < 1e-14
    tr = np.trace(U, axis1=-2, axis2=-1)
    tr2 = np.trace(U @ U, axis1=-2, axis2=-1)
    assert np.abs(np.trace(R, axis1=-2, axis2=-1) - 0.5 * (tr * tr - tr2)).max() < 1e-14
    P = np.array([[0, 0, 1], [0, -1, 0], [1, 0, 0]], dtype=float)
    assert np.abs(R - P @ np.conj(U) @ P.T).max() < 1e-14
    ph = rng.uniform(0, 2 * np.pi, 2)
    z = np.exp(1j * np.array([ph[0], ph[1], -ph[0] - ph[1]]))
    assert np.abs(orc.represent_antisym_su3(np.diag(z)) - np.diag([z[0] * z[1], z[0] * z[2], z[1] * z[2]])).max() < 1e-15
    V2 = inputs.haar_su2(1, 7, 0)[0]
    E = np.eye(3, dtype=complex)
    E[:2, :2] = V2
    want = np.eye(3, dtype=complex)
    want[1:, 1:] = V2
    assert np.abs(orc.represent_antisym_su3(E) - want).max() < 1e-15
    M = rng.normal(size=(3, 3)) + 1j * rng.normal(size=(3, 3))      # not unitary: R_ab = minor(rows pair a, columns pair b)
    pairs = [(0, 1), (0, 2), (1, 2)]
    minors = np.array([[M[i, k] * M[j, l] - M[i, l] * M[j, k] for (k, l) in pairs] for (i, j) in pairs])
    assert np.abs(orc.represent_antisym_su3(M) - minors).max() < 1e-14
