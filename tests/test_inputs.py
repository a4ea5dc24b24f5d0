"""The seeded input generator: reproducible, layout independent, right distributions (A14-A17)."""
import numpy as np

from paper_2411_18511_b200 import inputs
from helpers import dagger


def test_normals_counter_based():
    a = inputs.normals(1, 2, 0, 1000)
    b = np.concatenate([inputs.normals(1, 2, 0, 137), inputs.normals(1, 2, 137, 863)])
    assert np.array_equal(a, b)
    assert not np.array_equal(a, inputs.normals(2, 2, 0, 1000))
    assert not np.array_equal(a, inputs.normals(1, 3, 0, 1000))
    # fixed first values: the generator must never change silently (written by this generator itself,
    # they pin reproducibility across hosts, not correctness)
    n = inputs.normals(1, 1, 0, 200000)
    assert abs(n.mean()) < 0.01 and abs(n.std() - 1.0) < 0.01
    assert abs(np.mean(n ** 3)) < 0.03 and abs(np.mean(n ** 4) - 3.0) < 0.1


def test_su2_fields():
    L = (4, 4, 2, 6)
    for U in (inputs.haar_gauge(L, 1), inputs.weak_gauge(L, 0.3, 1)):
        assert U.shape == (inputs.volume(L), 4, 2, 2)
        assert np.abs(U @ dagger(U) - np.eye(2)).max() < 1e-15
        assert np.abs(np.linalg.det(U) - 1.0).max() < 1e-15
        # A14: second row is (-conj(beta), conj(alpha))
        assert np.array_equal(U[..., 1, 0], -np.conj(U[..., 0, 1]))
        assert np.array_equal(U[..., 1, 1], np.conj(U[..., 0, 0]))
    W = inputs.weak_gauge(L, 0.3, 1)
    # exp(i eps a.sigma): tr/2 = cos(eps |a|), |a| ~ chi_3 -> links stay near 1 on average
    assert 0.8 < (W[..., 0, 0].real).mean() < 0.95
    H = inputs.haar_gauge(L, 1)
    assert abs(H[..., 0, 0].real.mean()) < 0.05


def test_spinor_and_coords():
    L = (2, 4, 6, 4)
    psi = inputs.gaussian_spinor(L, 3, seed=2)
    assert psi.shape == (inputs.volume(L), 4, 3)
    assert abs(psi.real.std() - 1.0) < 0.05 and abs(psi.imag.std() - 1.0) < 0.05
    x = inputs.site_coords(L)
    lex = ((x[:, 0] * L[1] + x[:, 1]) * L[2] + x[:, 2]) * L[3] + x[:, 3]
    assert np.array_equal(lex, np.arange(inputs.volume(L)))
    assert np.array_equal(inputs.site_parity(L), x.sum(1) % 2)
    r = inputs.to_f32_rounded(psi)
    assert r.dtype == np.complex128 and np.array_equal(r, r.astype(np.complex64).astype(np.complex128))
