"""numpy helpers for the tests: facts typed here independently of oracle/ and of the CUDA path."""
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))

PAULI = np.array([[[0, 1], [1, 0]], [[0, -1j], [1j, 0]], [[1, 0], [0, -1]]], dtype=np.complex128)


def golden_gamma():
    """The A2 gamma matrices as printed in tests/golden/gamma_chiral.txt -> complex [4,4,4]."""
    tok = {"0": 0, "1": 1, "-1": -1, "i": 1j, "-i": -1j}
    mats, rows = [], []
    with open(os.path.join(HERE, "golden", "gamma_chiral.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            if line.startswith("gamma"):
                if rows:
                    mats.append(rows)
                rows = []
                continue
            rows.append([tok[t] for t in line.split()])
    mats.append(rows)
    g = np.array(mats, dtype=np.complex128)
    assert g.shape == (4, 4, 4)
    return g


def grid(a, L):
    """[V, ...] -> [L0, L1, L2, L3, ...] (lex order has x3 fastest, so this is a plain reshape)."""
    return a.reshape(tuple(L) + a.shape[1:])


def flat(a, L):
    V = L[0] * L[1] * L[2] * L[3]
    return np.ascontiguousarray(a.reshape((V,) + a.shape[4:]))


def fwd(a, mu):
    """field at x + mu_hat, on the grid view"""
    return np.roll(a, -1, axis=mu)


def bwd(a, mu):
    """field at x - mu_hat, on the grid view"""
    return np.roll(a, +1, axis=mu)


def dagger(m):
    return np.conj(np.swapaxes(m, -1, -2))


def gauge_transform(U, g, L):
    """U^g_mu(x) = g(x) U_mu(x) g(x+mu)^dag;  U [V,4,2,2], g [V,2,2]"""
    Ug = grid(U, L).copy()
    gg = grid(g, L)
    for mu in range(4):
        Ug[..., mu, :, :] = gg @ Ug[..., mu, :, :] @ dagger(fwd(gg, mu))
    return flat(Ug, L)


def wilson_dirac_numpy(L, U, psi, m0, gam):
    """Independent restatement of O1 with whole-lattice shifts (np.roll) and einsum:
    D psi = (4+m0) psi - 1/2 sum_mu [(1-g_mu) U_mu(x) psi(x+mu) + (1+g_mu) (U_mu^dag psi)(x-mu)].
    U [V,4,N,N] complex (or real), psi [V,4,N]."""
    Ug = grid(U.astype(np.complex128), L)
    p = grid(psi, L)
    one = np.eye(4)
    H = np.zeros_like(p)
    for mu in range(4):
        u = Ug[..., mu, :, :]
        t = np.einsum("...cd,...sd->...sc", u, fwd(p, mu))
        H += np.einsum("st,...tc->...sc", one - gam[mu], t)
        t = bwd(np.einsum("...dc,...sd->...sc", np.conj(u), p), mu)
        H += np.einsum("st,...tc->...sc", one + gam[mu], t)
    return flat((4.0 + m0) * p - 0.5 * H, L)


def rel_l2(a, b):
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))
