"""Seeded synthetic inputs, canonical layout.

This module is the ONE thing shared by the CPU oracle's tests and the CUDA path:
it draws random numbers and shapes them into canonical arrays.  It holds none of
the method's arithmetic (no gamma matrices, no hopping term, no representation
map, no clover term) and imports neither `oracle/` nor the CUDA binding.

Generator (A17): counter-based and layout independent.  Every real number is
    normal(seed, field, e) with e = global element index in the canonical array,
produced by two SplitMix64-finalised 64-bit hashes feeding one Box-Muller draw in
double precision.  The same (seed, field, e) gives the same value whatever the
chunking, the host or the order of generation.

Canonical formats (A3/A4), V = L0*L1*L2*L3, lex(x) = ((x0*L1 + x1)*L2 + x2)*L3 + x3:
    spinor       complex128 [V, 4 spin, N colour]
    fund gauge   complex128 [V, 4 mu, 2 row, 2 col]
    site SU(2)   complex128 [V, 2, 2]                 (gauge transformations)

The paper's workloads are SU(2) gauge configurations from HiRep runs at local
volume 48^4 that are not published with it; BASELINE.json
`configs` replaces them with the seeded fields below (Haar-random links, or
U = exp(i eps a.sigma) links, Gaussian spinors).
"""
from __future__ import annotations

import numpy as np

FIELD_GAUGE = 1
FIELD_SPINOR = 2
FIELD_SPINOR2 = 3
FIELD_GAUGE_TRANSFORM = 4

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_TWO_PI = 6.283185307179586476925286766559


def _mix(z: np.ndarray) -> np.ndarray:
    """SplitMix64 output function on uint64 arrays (wrap-around arithmetic)."""
    z = (z ^ (z >> np.uint64(30))) * _M1
    z = (z ^ (z >> np.uint64(27))) * _M2
    return z ^ (z >> np.uint64(31))


def _stream_key(seed: int, field: int) -> np.uint64:
    s = np.array([(int(seed) & 0xFFFFFFFF) | ((int(field) & 0xFFFFFFFF) << 32)], dtype=np.uint64)
    return _mix(_mix(s) + _GOLDEN)[0]


def normals(seed: int, field: int, start: int, count: int) -> np.ndarray:
    """`count` N(0,1) doubles for global element indices start .. start+count-1."""
    with np.errstate(over="ignore"):
        key = _stream_key(seed, field)
        e = np.arange(start, start + count, dtype=np.uint64)
        h1 = _mix(key + _GOLDEN * (np.uint64(2) * e + np.uint64(1)))
        h2 = _mix(key + _GOLDEN * (np.uint64(2) * e + np.uint64(2)))
    # 53-bit uniforms in (0, 1): never 0, so the log is finite
    u1 = ((h1 >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)
    u2 = ((h2 >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(_TWO_PI * u2)


def volume(L) -> int:
    return int(L[0]) * int(L[1]) * int(L[2]) * int(L[3])


def _chunks(total: int, chunk: int):
    s = 0
    while s < total:
        n = min(chunk, total - s)
        yield s, n
        s += n


def gaussian_spinor(L, ncolour: int, seed: int = 2, field: int = FIELD_SPINOR) -> np.ndarray:
    """Spinor with independent N(0,1) real and imaginary parts (A15)."""
    V = volume(L)
    per_site = 4 * ncolour * 2
    out = np.empty((V, 4, ncolour), dtype=np.complex128)
    flat = out.view(np.float64).reshape(-1)
    for s, n in _chunks(V, 1 << 18):
        flat[s * per_site:(s + n) * per_site] = normals(seed, field, s * per_site, n * per_site)
    return out


def _quaternion_to_su2(q: np.ndarray, out: np.ndarray) -> None:
    """A14: U = a0 + i a.sigma = [[a0 + i a3, a2 + i a1], [-a2 + i a1, a0 - i a3]]."""
    a0, a1, a2, a3 = q[..., 0], q[..., 1], q[..., 2], q[..., 3]
    out[..., 0, 0] = a0 + 1j * a3
    out[..., 0, 1] = a2 + 1j * a1
    out[..., 1, 0] = -a2 + 1j * a1
    out[..., 1, 1] = a0 - 1j * a3


def haar_su2(n: int, seed: int, field: int) -> np.ndarray:
    """n Haar-random SU(2) matrices: unit quaternion from N(0,1)^4 (BASELINE.json configs[0])."""
    out = np.empty((n, 2, 2), dtype=np.complex128)
    for s, m in _chunks(n, 1 << 18):
        q = normals(seed, field, 4 * s, 4 * m).reshape(m, 4)
        q /= np.sqrt((q * q).sum(axis=1, keepdims=True))
        _quaternion_to_su2(q, out[s:s + m])
    return out


def weak_su2(n: int, eps: float, seed: int, field: int) -> np.ndarray:
    """n matrices U = exp(i eps a.sigma), a ~ N(0,1)^3 (A16): cos(th) + i sin(th) n.sigma."""
    out = np.empty((n, 2, 2), dtype=np.complex128)
    for s, m in _chunks(n, 1 << 18):
        a = normals(seed, field, 3 * s, 3 * m).reshape(m, 3)
        r = np.sqrt((a * a).sum(axis=1))
        th = eps * r
        q = np.empty((m, 4))
        q[:, 0] = np.cos(th)
        q[:, 1:] = a * (np.sin(th) / r)[:, None]
        _quaternion_to_su2(q, out[s:s + m])
    return out


def haar_gauge(L, seed: int = 1) -> np.ndarray:
    """Fundamental gauge field [V,4,2,2], Haar-random links."""
    V = volume(L)
    return haar_su2(4 * V, seed, FIELD_GAUGE).reshape(V, 4, 2, 2)


def weak_gauge(L, eps: float = 0.3, seed: int = 1) -> np.ndarray:
    """Fundamental gauge field [V,4,2,2], links exp(i eps a.sigma)."""
    V = volume(L)
    return weak_su2(4 * V, eps, seed, FIELD_GAUGE).reshape(V, 4, 2, 2)


def unit_gauge(L) -> np.ndarray:
    V = volume(L)
    u = np.zeros((V, 4, 2, 2), dtype=np.complex128)
    u[..., 0, 0] = 1.0
    u[..., 1, 1] = 1.0
    return u


def haar_su3(n: int, seed: int, field: int) -> np.ndarray:
    """n Haar-random SU(3) matrices: QR of a complex Gaussian 3x3 matrix with the phases of R's diagonal moved into Q (Haar
    on U(3)), then divided by a cube root of the determinant."""
    out = np.empty((n, 3, 3), dtype=np.complex128)
    for s, m in _chunks(n, 1 << 16):
        z = normals(seed, field, 18 * s, 18 * m).reshape(m, 3, 3, 2)
        q, r = np.linalg.qr(z[..., 0] + 1j * z[..., 1])
        d = np.diagonal(r, axis1=-2, axis2=-1)
        q = q * (d / np.abs(d))[:, None, :]
        det = np.linalg.det(q)
        out[s:s + m] = q / np.exp(1j * np.angle(det) / 3.0)[:, None, None]
    return out


def haar_gauge_su3(L, seed: int = 1) -> np.ndarray:
    """SU(3) fundamental gauge field [V,4,3,3], Haar-random links (the rep-2 link format: complex 3 x 3)."""
    V = volume(L)
    return haar_su3(4 * V, seed, FIELD_GAUGE).reshape(V, 4, 3, 3)


def haar_sites_su3(L, seed: int = 4) -> np.ndarray:
    """One Haar SU(3) matrix per site [V,3,3] (a local gauge transformation g)."""
    return haar_su3(volume(L), seed, FIELD_GAUGE_TRANSFORM)


def haar_sites(L, seed: int = 4) -> np.ndarray:
    """One Haar SU(2) matrix per site [V,2,2] (a local gauge transformation g)."""
    return haar_su2(volume(L), seed, FIELD_GAUGE_TRANSFORM)


def site_coords(L) -> np.ndarray:
    """int64 [V,4]: coordinates of every site in canonical (lex) order."""
    V = volume(L)
    s = np.arange(V, dtype=np.int64)
    x = np.empty((V, 4), dtype=np.int64)
    for mu in (3, 2, 1, 0):
        x[:, mu] = s % L[mu]
        s = s // L[mu]
    return x


def site_parity(L) -> np.ndarray:
    """int64 [V]: (x0+x1+x2+x3) mod 2, even = 0 (A3)."""
    return site_coords(L).sum(axis=1) % 2


def to_f32_rounded(a: np.ndarray) -> np.ndarray:
    """Round complex128/float64 to the nearest float and promote back (SURVEY §8(c):
    fp32 runs and the oracle see the same rounded inputs)."""
    if np.iscomplexobj(a):
        return a.astype(np.complex64).astype(np.complex128)
    return a.astype(np.float32).astype(np.float64)
