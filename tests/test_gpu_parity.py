"""GPU parity: libhr_dslash (through the C-ABI) against the CPU oracle on the same seeded inputs.

BASELINE.json `north_star` bar: relative L2 error over the compared outputs <= 1e-13 (fp64), <= 1e-5 (fp32);
for fp32 both sides see the inputs rounded to float.  The five BASELINE.json configs are
covered at full size; edge cases (extent 2, ragged extents, both kernels) at sizes the oracle does in
seconds.  Expected values always come from oracle/ or from identities — never from the CUDA path."""
import os

import numpy as np
import pytest

from paper_2411_18511_b200 import inputs

pytestmark = pytest.mark.gpu

TOL = {0: 1e-13, 1: 1e-5}   # hr.PREC_F64, hr.PREC_F32
NTHREADS = max(1, len(os.sched_getaffinity(0)))


@pytest.fixture(scope="module")
def hr():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2411_18511_b200 import build, hr as _hr
    build.build()
    _hr.lib()
    return _hr


def lattice(hr, L, rep=0, prec=0, kernel=0):
    from paper_2411_18511_b200.lattice import Lattice
    return Lattice(L, rep, prec, kernel)


def rel(a, b):
    return float(np.linalg.norm((a.astype(np.complex128) - b).ravel()) / np.linalg.norm(b.ravel()))


def site_err(a, b):
    """largest per-site error relative to the r.m.s. site norm of the expected field: the whole-field norm of rel()
    averages a defect confined to a few sites away (0.02 at one of 5.3 M sites is 1e-5 of the field norm); this
    companion does not.  Arrays are [sites, spin, colour]."""
    d = np.linalg.norm((a.astype(np.complex128) - b).reshape(b.shape[0], -1), axis=1)
    return float(d.max() / (np.linalg.norm(b.ravel()) / np.sqrt(b.shape[0])))


SITE_TOL = {0: 2e-13, 1: 2e-5}   # per-site companion of TOL (a single site may sit a few sigma above the r.m.s. error)


def rounded(a, prec):
    return inputs.to_f32_rounded(a) if prec == 1 else a


def kernels_for(hr, L, rep, prec):
    """kernel selectors to test on this lattice: generic always, tiled where the lattice fits it"""
    ks = [hr.KERNEL_GENERIC]
    if hr.hr_kernel_name(hr.geom(L, rep, prec, hr.LINKS_COMPRESSED, hr.KERNEL_TILED)) == "tiled":
        ks.append(hr.KERNEL_TILED)
    return ks


def dense_to_blocks(A):
    """oracle dense [n,8,8] -> canonical blocks [n,2,16]: 4 real diagonal entries, then the strictly-lower
    entries (1,0) (2,0) (3,0) (2,1) (3,1) (3,2) as re,im (include/hr_dslash.h)."""
    D = A.shape[-1] // 2          # 4 (fundamental) or 6 (adjoint): block = one chirality, index (spin mod 2)*N + colour
    out = np.empty((A.shape[0], 2, D * D))
    for chi in range(2):
        B = A[:, D * chi:D * chi + D, D * chi:D * chi + D]
        for i in range(D):
            out[:, chi, i] = B[:, i, i].real
        k = D
        for j in range(D):
            for i in range(j + 1, D):
                out[:, chi, k] = B[:, i, j].real
                out[:, chi, k + 1] = B[:, i, j].imag
                k += 2
    return out


def gpu_ops(hr, lat, U_dev, psi, m0):
    """run hop_oe, hop_eo, full D and Dhat on the GPU; return canonical arrays (untouched parity = 0)"""
    import torch
    psi_dev = lat.put_spinor(psi)
    res = {}
    out = torch.zeros_like(psi_dev)
    lat.hop(hr.EO_HOP_OE, U_dev, lat.even(psi_dev), lat.odd(out))
    lat.hop(hr.EO_HOP_EO, U_dev, lat.odd(psi_dev), lat.even(out))
    res["hop"] = lat.get_spinor(out)
    res["dirac"] = lat.get_spinor(lat.dirac(m0, U_dev, psi_dev))
    out2 = torch.zeros_like(psi_dev)
    lat.dhat(m0, U_dev, lat.even(psi_dev), lat.even(out2))
    res["dhat"] = lat.get_spinor(out2)
    torch.cuda.synchronize()
    return res


def oracle_ops(orc, L, rep, U, psi, m0):
    res = {}
    h = orc.hop(L, rep, 0, U, psi, nthreads=NTHREADS)
    res["hop"] = orc.hop(L, rep, 1, U, psi, nthreads=NTHREADS, out=h)
    res["dirac"] = orc.dirac(L, rep, m0, U, psi, nthreads=NTHREADS)
    res["dhat"] = orc.dirac_eo(L, rep, m0, U, psi, nthreads=NTHREADS)
    return res


# ------------------------------------------------------------------ layout permutations
@pytest.mark.parametrize("L", [(4, 4, 4, 4), (2, 4, 6, 8), (2, 2, 2, 2), (6, 4, 2, 10)])
@pytest.mark.parametrize("prec", [0, 1])
def test_pack_unpack_roundtrip_is_exact(hr, L, prec):
    U = rounded(inputs.haar_gauge(L, 1), prec)
    for rep, N in ((0, 2), (1, 3)):
        lat = lattice(hr, L, rep, prec)
        psi = rounded(inputs.gaussian_spinor(L, N, 2), prec)
        assert np.array_equal(lat.get_spinor(lat.put_spinor(psi)).astype(np.complex128), psi)
    lat = lattice(hr, L, 0, prec)
    assert np.array_equal(lat.get_gauge_fund(lat.put_gauge_fund(U)).astype(np.complex128), U)
    R = rounded(inputs.normals(7, 9, 0, lat.V * 36).reshape(lat.V, 4, 3, 3), prec)
    assert np.array_equal(lat.get_gauge_adj(lat.put_gauge_adj(R)).astype(np.float64), R)
    B = rounded(inputs.normals(8, 9, 0, lat.V * 32).reshape(lat.V, 2, 16), prec)
    assert np.array_equal(lat.get_clover(lat.put_clover(B)).astype(np.float64), B)


def test_device_layout_is_the_documented_one(hr):
    """chunk c of site (row,h) of parity p sits at 16-byte index p*Vh*NCH + (row*NCH + c)*L3h + h."""
    L = (2, 4, 6, 8)
    lat = lattice(hr, L, 0, 0)
    psi = inputs.gaussian_spinor(L, 2, 2)
    raw = lat.put_spinor(psi).cpu().numpy().view(np.complex128)
    x = inputs.site_coords(L)
    par = x.sum(1) % 2
    row = (x[:, 0] * L[1] + x[:, 1]) * L[2] + x[:, 2]
    h = x[:, 3] // 2
    L3h, Vh = L[3] // 2, lat.V // 2
    for c in (0, 3, 7):
        idx = par * Vh * 8 + (row * 8 + c) * L3h + h
        assert np.array_equal(raw[idx], psi.reshape(lat.V, 8)[:, c])


# ------------------------------------------------------------------ config 0 and the edge lattices
@pytest.mark.parametrize("L", [(4, 4, 4, 4), (2, 2, 2, 2), (2, 4, 6, 8), (4, 4, 4, 2), (6, 2, 4, 12), (8, 4, 4, 16), (4, 8, 8, 8), (4, 2, 4, 52), (2, 2, 2, 96)])
@pytest.mark.parametrize("prec", [0, 1])
def test_fundamental_small_lattices(hr, orc, L, prec):
    """configs[0] (4^4, Haar links, m0 = -0.2: full D and even-odd operator) plus degenerate and ragged extents"""
    m0 = -0.2
    U = rounded(inputs.haar_gauge(L, 1), prec)
    psi = rounded(inputs.gaussian_spinor(L, 2, 2), prec)
    want = oracle_ops(orc, L, 0, U, psi, m0)
    for kernel in kernels_for(hr, L, 0, prec):
        lat = lattice(hr, L, 0, prec, kernel)
        got = gpu_ops(hr, lat, lat.put_gauge_fund(U), psi, m0)
        for k in want:
            assert rel(got[k], want[k]) <= TOL[prec], (k, kernel)
        odd = inputs.site_parity(L) == 1
        assert not got["dhat"][odd].any()


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (2, 2, 2, 2), (2, 4, 6, 8), (4, 6, 4, 2)])
@pytest.mark.parametrize("prec", [0, 1])
def test_adjoint_small_lattices(hr, orc, L, prec):
    m0 = -0.3
    Uf = rounded(inputs.haar_gauge(L, 1), prec)
    R, _ = orc.represent(Uf)
    psi = rounded(inputs.gaussian_spinor(L, 3, 2), prec)
    lat = lattice(hr, L, 1, prec)
    R_dev = lat.represent(lat.put_gauge_fund(Uf))
    got_R = lat.get_gauge_adj(R_dev).astype(np.float64)
    assert np.abs(got_R - R).max() <= (1e-14 if prec == 0 else 1e-6)
    # the adjoint operator is compared on the links the oracle built (rounded for fp32), packed directly
    Rr = rounded(R, prec)
    want = oracle_ops(orc, L, 1, Rr, psi, m0)
    for kernel in kernels_for(hr, L, 1, prec):
        latk = lattice(hr, L, 1, prec, kernel)
        got = gpu_ops(hr, latk, latk.put_gauge_adj(Rr), psi, m0)
        for k in want:
            assert rel(got[k], want[k]) <= TOL[prec], (k, kernel)
    if prec == 0:   # and end to end on the links the GPU built
        got2 = gpu_ops(hr, lat, R_dev, psi, m0)
        for k in want:
            assert rel(got2[k], want[k]) <= TOL[prec], k


@pytest.mark.parametrize("L,seglen", [((8, 2, 8, 6), 1), ((8, 8, 32, 6), 2), ((8, 8, 40, 6), 4), ((8, 8, 80, 6), 8)])
@pytest.mark.parametrize("rep,N", [(0, 2), (1, 3)])
def test_tiled_kernel_segment_lengths(hr, orc, L, seglen, rep, N):
    """the x0-marching kernels with segments of 1, 2, 4 and 8 planes: the planner minimises waves x (L0/segments + 3),
    so the segment length follows from the number of tiles (2, 32, 40, 80 tiles of 2 x 4 rows on 148 SMs; the plan is
    read back through hr_kernel_plan and asserted); tiles that wrap onto themselves in x1 (L1 = T1) and many tiles in
    x2; all four operators against the oracle"""
    m0 = -0.2
    Uf = inputs.haar_gauge(L, 1)
    U = Uf if rep == 0 else orc.represent(Uf)[0]
    psi = inputs.gaussian_spinor(L, N, 2)
    want = oracle_ops(orc, L, rep, U, psi, m0)
    lat = lattice(hr, L, rep, 0, hr.KERNEL_TILED)
    assert hr.hr_kernel_name(lat.g) == "tiled"
    plan = hr.hr_kernel_plan(lat.g, hr.OP_HOP)
    assert plan["kernel"] == 1 and plan["nseg"] * plan["seglen"] == L[0]
    import torch
    if torch.cuda.get_device_properties(0).multi_processor_count == 148:
        assert plan["seglen"] == seglen, plan
    full = hr.hr_kernel_plan(lat.g, hr.OP_DIRAC)
    assert full["kernel"] == (2 if rep == 0 else 1), full
    got = gpu_ops(hr, lat, lat.put_gauge_fund(U) if rep == 0 else lat.put_gauge_adj(U), psi, m0)
    for k in want:
        assert rel(got[k], want[k]) <= TOL[0], (k, plan, full)


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (2, 2, 2, 2), (2, 4, 6, 8), (8, 2, 8, 6), (6, 2, 4, 12)])
@pytest.mark.parametrize("prec", [0, 1])
def test_adjoint_on_the_fly_links(hr, orc, L, prec):
    """the adjoint operators handed the FUNDAMENTAL gauge field (HR_LINKS_ONTHEFLY) rebuild
    R in registers; expected values = the oracle's adjoint operators on the oracle's R(U)"""
    m0 = -0.3
    Uf = rounded(inputs.haar_gauge(L, 1), prec)
    R, _ = orc.represent(Uf)
    psi = rounded(inputs.gaussian_spinor(L, 3, 2), prec)
    want = oracle_ops(orc, L, 1, R, psi, m0)
    from paper_2411_18511_b200.lattice import Lattice
    for kernel in kernels_for(hr, L, 1, prec):
        lat = Lattice(L, hr.REP_ADJ, prec, kernel, link_storage=hr.LINKS_ONTHEFLY)
        got = gpu_ops(hr, lat, lat.put_gauge_fund(Uf), psi, m0)
        for k in want:
            assert rel(got[k], want[k]) <= TOL[prec], (k, kernel)


# ------------------------------------------------------------------ config 1
@pytest.mark.parametrize("prec", [0, 1])
def test_config1_16to4_dhat_100_repetitions(hr, orc, prec):
    """configs[1]: 16^4, links exp(i 0.3 a.sigma), m0 = -0.1, Dhat on the even spinor, 100 repetitions of the
    same application; every repetition must give the same bits."""
    import torch
    L, m0 = (16, 16, 16, 16), -0.1
    U = rounded(inputs.weak_gauge(L, 0.3, 1), prec)
    psi = rounded(inputs.gaussian_spinor(L, 2, 2), prec)
    want = orc.dirac_eo(L, 0, m0, U, psi, nthreads=NTHREADS)
    for kernel in kernels_for(hr, L, 0, prec):
        lat = lattice(hr, L, 0, prec, kernel)
        U_dev, psi_dev = lat.put_gauge_fund(U), lat.put_spinor(psi)
        first = torch.zeros_like(psi_dev)
        last = torch.zeros_like(psi_dev)
        tmp = lat.empty_spinor(hr.ODD)
        lat.dhat(m0, U_dev, lat.even(psi_dev), lat.even(first), tmp)
        for _ in range(99):
            lat.dhat(m0, U_dev, lat.even(psi_dev), lat.even(last), tmp)
        torch.cuda.synchronize()
        assert torch.equal(first, last)
        assert rel(lat.get_spinor(last), want) <= TOL[prec], kernel


# ------------------------------------------------------------------ config 2
def test_config2_24to4_adjoint(hr, orc):
    """configs[2]: 24^4 adjoint fp64, links built from Haar fundamental links by hr_represent_gauge, m0 = -0.3"""
    L, m0 = (24, 24, 24, 24), -0.3
    Uf = inputs.haar_gauge(L, 1)
    psi = inputs.gaussian_spinor(L, 3, 2)
    R, max_imag = orc.represent(Uf)
    assert max_imag < 1e-15
    lat = lattice(hr, L, 1, 0)
    R_dev = lat.represent(lat.put_gauge_fund(Uf))
    got_R = lat.get_gauge_adj(R_dev)
    assert np.abs(got_R - R).max() <= 1e-14
    # P6 on the GPU's own output: real orthogonal with det +1
    RRt = np.einsum("xmab,xmcb->xmac", got_R, got_R)
    assert np.abs(RRt - np.eye(3)).max() < 1e-14
    assert np.abs(np.linalg.det(got_R) - 1.0).max() < 1e-14
    want = oracle_ops(orc, L, 1, R, psi, m0)
    got = gpu_ops(hr, lat, R_dev, psi, m0)
    for k in want:
        assert rel(got[k], want[k]) <= 1e-13, k
        assert site_err(got[k], want[k]) <= SITE_TOL[0], k
    # the same operators with the links rebuilt on the fly from the fundamental field, both kernels
    from paper_2411_18511_b200.lattice import Lattice
    for kernel in kernels_for(hr, L, 1, 0):
        fly = Lattice(L, hr.REP_ADJ, hr.PREC_F64, kernel, link_storage=hr.LINKS_ONTHEFLY)
        got = gpu_ops(hr, fly, fly.put_gauge_fund(Uf), psi, m0)
        for k in want:
            assert rel(got[k], want[k]) <= 1e-13, (k, kernel, "on the fly")


def test_48to4_adjoint_full_lattice_slab_order(hr, orc):
    """adjoint fermions at 48^4 (the paper's local volume): the full-lattice launch of the generic kernel walks the
    lattice in x1-slabs there (hr_hop_generic.cuh: generic_slab_w1).  Full D with stored and with on-the-fly links against the
    oracle's per-site operator on sampled sites that include both sides of every slab boundary and the lattice corners."""
    L, m0 = (48, 48, 48, 48), -0.3
    Uf = inputs.haar_gauge(L, 1)
    psi = inputs.gaussian_spinor(L, 3, 2)
    R, _ = orc.represent(Uf)
    V = inputs.volume(L)
    lex = lambda x0, x1, x2, x3: ((x0 * 48 + x1) * 48 + x2) * 48 + x3
    fixed = [lex(x0, x1, x2, x3) for x0 in (0, 17, 47) for x1 in (0, 5, 7, 8, 11, 12, 15, 16, 23, 24, 35, 36, 47) for (x2, x3) in ((0, 0), (47, 47), (20, 31))]
    sites = np.unique(np.concatenate([np.array(fixed), (inputs.normals(11, 9, 0, 60) * 1e9).astype(np.int64) % V]))
    want = orc.dirac_sites(L, 1, m0, R, psi, sites)
    from paper_2411_18511_b200.lattice import Lattice
    lat = Lattice(L, hr.REP_ADJ, hr.PREC_F64, hr.KERNEL_AUTO)
    assert hr.hr_kernel_plan(lat.g, hr.OP_DIRAC)["kernel"] == 0          # the generic kernel
    got = lat.get_spinor(lat.dirac(m0, lat.represent(lat.put_gauge_fund(Uf)), lat.put_spinor(psi)))
    assert rel(got[sites], want) <= 1e-13 and site_err(got[sites], want) <= SITE_TOL[0]
    fly = Lattice(L, hr.REP_ADJ, hr.PREC_F64, hr.KERNEL_AUTO, link_storage=hr.LINKS_ONTHEFLY)
    got = fly.get_spinor(fly.dirac(m0, fly.put_gauge_fund(Uf), fly.put_spinor(psi)))
    assert rel(got[sites], want) <= 1e-13 and site_err(got[sites], want) <= SITE_TOL[0]


# ------------------------------------------------------------------ config 3
@pytest.fixture(scope="module")
def big_inputs():
    L = (48, 48, 48, 48)
    return L, inputs.haar_gauge(L, 1), inputs.gaussian_spinor(L, 2, 2)


@pytest.mark.parametrize("prec", [0, 1])
def test_config3_48to4_fundamental(hr, orc, big_inputs, prec):
    """configs[3]: 48^4, Haar links, m0 = -0.2: bare hops, full D and Dhat against the oracle on the whole
    field, in the launch configuration bench.py times (kernel = AUTO), plus the forced generic kernel."""
    L, U, psi = big_inputs
    m0 = -0.2
    U, psi = rounded(U, prec), rounded(psi, prec)
    want = oracle_ops(orc, L, 0, U, psi, m0)
    kernels = [hr.KERNEL_AUTO]
    if hr.hr_kernel_name(hr.geom(L, 0, prec)) != "generic":
        kernels.append(hr.KERNEL_GENERIC)
    for kernel in kernels:
        lat = lattice(hr, L, 0, prec, kernel)
        got = gpu_ops(hr, lat, lat.put_gauge_fund(U), psi, m0)
        for k in want:
            assert rel(got[k], want[k]) <= TOL[prec], (k, kernel)
            assert site_err(got[k], want[k]) <= SITE_TOL[prec], (k, kernel)


def test_config3_invariants_on_the_gpu(hr, big_inputs):
    """P2 (gamma5-hermiticity) and P4 (Schur identity) hold at any size and need no oracle run: evaluated at 48^4
    on GPU outputs, in fp64."""
    import torch
    L, U, psi = big_inputs
    m0 = -0.2
    lat = lattice(hr, L, 0, 0)
    U_dev = lat.put_gauge_fund(U)
    chi = inputs.gaussian_spinor(L, 2, 3, inputs.FIELD_SPINOR2)
    g5 = np.array([1.0, 1.0, -1.0, -1.0])[None, :, None]
    Dpsi = lat.get_spinor(lat.dirac(m0, U_dev, lat.put_spinor(psi)))
    Dg5chi = lat.get_spinor(lat.dirac(m0, U_dev, lat.put_spinor(g5 * chi)))
    lhs = np.vdot(chi.ravel(), Dpsi.ravel())
    rhs = np.vdot((g5 * Dg5chi).ravel(), psi.ravel())
    assert abs(lhs - rhs) <= 1e-12 * abs(lhs)
    # P4: eta = D x  =>  Dhat x_e = eta_e - D_eo D_oo^-1 eta_o = eta_e + H_eo eta_o / (2 (4+m0))
    eta = Dpsi
    eta_dev = lat.put_spinor(eta)
    psi_dev = lat.put_spinor(psi)
    dh = torch.zeros_like(psi_dev)
    lat.dhat(m0, U_dev, lat.even(psi_dev), lat.even(dh))
    hop = torch.zeros_like(psi_dev)
    lat.hop(hr.EO_HOP_EO, U_dev, lat.odd(eta_dev), lat.even(hop))
    even = inputs.site_parity(L) == 0
    lhs = lat.get_spinor(dh)[even]
    rhs = eta[even] + lat.get_spinor(hop)[even] / (2.0 * (4.0 + m0))
    assert rel(lhs, rhs) <= 1e-13


# ------------------------------------------------------------------ clover (config 4)
def clover_oracle(orc, L, U, m0, csw):
    A = orc.clover_dense(L, 4.0 + m0, csw, U, nthreads=NTHREADS)
    return A, orc.invert(A)


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (2, 4, 6, 8), (8, 8, 8, 8), (2, 2, 2, 2)])
@pytest.mark.parametrize("prec", [0, 1])
def test_clover_small_lattices(hr, orc, L, prec):
    """C1 blocks and inverses, C2/C3 application, E2 (Dhat with clover) against the oracle's dense 8x8 route"""
    import torch
    m0, csw = -0.25, 1.2
    U = rounded(inputs.weak_gauge(L, 0.3, 1), prec)
    psi = rounded(inputs.gaussian_spinor(L, 2, 2), prec)
    A, Ainv = clover_oracle(orc, L, U, m0, csw)
    for kernel in kernels_for(hr, L, 0, prec):
        lat = lattice(hr, L, 0, prec, kernel)
        U_dev, psi_dev = lat.put_gauge_fund(U), lat.put_spinor(psi)
        fwd, inv = lat.clover_build(m0, csw, U_dev)
        tol_blk = 1e-13 if prec == 0 else 1e-6
        bf, bi = dense_to_blocks(A), dense_to_blocks(Ainv)
        assert np.linalg.norm(lat.get_clover(fwd) - bf) <= tol_blk * np.linalg.norm(bf)
        assert np.linalg.norm(lat.get_clover(inv) - bi) <= tol_blk * np.linalg.norm(bi)
        # C2 / C3 on both parities at once and on one parity
        got = lat.get_spinor(lat.clover_apply(hr.BOTH, fwd, psi_dev))
        assert rel(got, orc.site_matvec(L, 3, A, psi)) <= TOL[prec]
        got = lat.get_spinor(lat.clover_apply(hr.BOTH, inv, psi_dev))
        assert rel(got, orc.site_matvec(L, 3, Ainv, psi)) <= TOL[prec]
        half = torch.zeros_like(psi_dev)
        lat.clover_apply(hr.ODD, inv, lat.odd(psi_dev), lat.odd(half))
        assert rel(lat.get_spinor(half), orc.site_matvec(L, 2, Ainv, psi)) <= TOL[prec]
        # H3c: the clover-improved operator on all sites, D_sw psi = A psi - H psi / 2 (oracle: O1 + O5)
        dsw = lat.empty_spinor()
        hr.hr_dirac_clover_apply(lat.g, U_dev, fwd, psi_dev, dsw, hr.stream_ptr())
        C = A - (4.0 + m0) * np.eye(8)[None]
        assert rel(lat.get_spinor(dsw), orc.dirac_clover(L, m0, U, C, psi, nthreads=NTHREADS)) <= TOL[prec], kernel
        # E2 with the GPU's own blocks
        out = torch.zeros_like(psi_dev)
        lat.dhat(m0, U_dev, lat.even(psi_dev), lat.even(out), clover_fwd=fwd, clover_inv=inv)
        want = orc.dirac_eo_clover(L, U, A, Ainv, psi, nthreads=NTHREADS)
        assert rel(lat.get_spinor(out), want) <= TOL[prec], kernel
        # ... and with the oracle's blocks packed in (a pure mat-vec + hop check)
        if prec == 0:
            out2 = torch.zeros_like(psi_dev)
            lat.dhat(m0, U_dev, lat.even(psi_dev), lat.even(out2), clover_fwd=lat.put_clover(bf), clover_inv=lat.put_clover(bi))
            assert rel(lat.get_spinor(out2), want) <= TOL[prec]


def test_config4_48to4_clover(hr, orc):
    """configs[4]: 48^4 fp64, links exp(i 0.3 a.sigma), c_sw = 1.2, m0 = -0.25.  Blocks, C2/C3 and E2 are
    compared with the oracle on sampled sites (the dense 8x8 oracle field would need 11 GB at this size);
    the Schur identity with clover (P4) checks E2 on every even site."""
    import torch
    L, m0, csw = (48, 48, 48, 48), -0.25, 1.2
    V = inputs.volume(L)
    U = inputs.weak_gauge(L, 0.3, 1)
    psi = inputs.gaussian_spinor(L, 2, 2)
    lat = lattice(hr, L, 0, 0)
    U_dev, psi_dev = lat.put_gauge_fund(U), lat.put_spinor(psi)
    fwd, inv = lat.clover_build(m0, csw, U_dev)
    got_f, got_i = lat.get_clover(fwd), lat.get_clover(inv)
    got_Apsi = lat.get_spinor(lat.clover_apply(hr.BOTH, fwd, psi_dev))
    got_Aipsi = lat.get_spinor(lat.clover_apply(hr.BOTH, inv, psi_dev))
    # sampled ranges: lattice corners (wrap-around in every direction), the middle, a ragged interior stretch
    for b, e in [(0, 96), (V - 96, V), (V // 2 - 48, V // 2 + 48), (1234567, 1234567 + 101), (47 * 48 ** 3, 47 * 48 ** 3 + 64)]:
        A = orc.clover_dense(L, 4.0 + m0, csw, U, begin=b, end=e)[b:e]
        Ainv = orc.invert(A)
        bf, bi = dense_to_blocks(A), dense_to_blocks(Ainv)
        assert np.linalg.norm(got_f[b:e] - bf) <= 1e-13 * np.linalg.norm(bf)
        assert np.linalg.norm(got_i[b:e] - bi) <= 1e-13 * np.linalg.norm(bi)
        want = np.einsum("xij,xj->xi", A, psi[b:e].reshape(-1, 8)).reshape(-1, 4, 2)
        assert rel(got_Apsi[b:e], want) <= 1e-13
        want = np.einsum("xij,xj->xi", Ainv, psi[b:e].reshape(-1, 8)).reshape(-1, 4, 2)
        assert rel(got_Aipsi[b:e], want) <= 1e-13
    # E2 on sampled even sites, step by step with oracle calls: the 8 neighbours y of x, t(y) = A(y)^-1 (H psi)(y),
    # then one more hop at x of the field that is t on those neighbours
    out = torch.zeros_like(psi_dev)
    lat.dhat(m0, U_dev, lat.even(psi_dev), lat.even(out), clover_fwd=fwd, clover_inv=inv)
    got = lat.get_spinor(out)
    coords = inputs.site_coords(L)
    rng = np.random.default_rng(5)
    cand = np.concatenate([[0, V - 2, 47 * 48 ** 3 + 47 * 48 ** 2], rng.integers(0, V, 40)])
    sites = [int(s) for s in cand if coords[s].sum() % 2 == 0][:24]
    scratch = np.zeros_like(psi)
    Lv = np.array(L)
    strides = np.array([L[1] * L[2] * L[3], L[2] * L[3], L[3], 1])
    want, have = [], []
    for x in sites:
        nb = []
        for mu in range(4):
            for d in (+1, -1):
                y = coords[x].copy()
                y[mu] = (y[mu] + d) % Lv[mu]
                nb.append(int(y @ strides))
        nb = np.array(sorted(set(nb)), dtype=np.int64)
        t1 = orc.hop_sites(L, 0, U, psi, nb).reshape(-1, 8)
        for k, y in enumerate(nb):
            Ay = orc.clover_dense(L, 4.0 + m0, csw, U, begin=y, end=y + 1)[y]
            scratch[y] = (orc.invert(Ay[None])[0] @ t1[k]).reshape(4, 2)
        h = orc.hop_sites(L, 0, U, scratch, np.array([x]))[0]
        scratch[nb] = 0.0
        Ax = orc.clover_dense(L, 4.0 + m0, csw, U, begin=x, end=x + 1)[x]
        want.append((Ax @ psi[x].reshape(8)).reshape(4, 2) - 0.25 * h)
        have.append(got[x])
    assert rel(np.array(have), np.array(want)) <= 1e-13
    # P4 with clover on all even sites: eta = D_sw x = D x + (A - (4+m0)) x;
    #   Dhat x_e = eta_e - D_eo D_oo^-1 eta_o = eta_e + 1/2 H_eo A_oo^-1 eta_o
    Dx = lat.get_spinor(lat.dirac(m0, U_dev, psi_dev))
    eta = Dx + got_Apsi - (4.0 + m0) * psi
    eta_dev = lat.put_spinor(eta)
    t = torch.zeros_like(psi_dev)
    lat.clover_apply(hr.ODD, inv, lat.odd(eta_dev), lat.odd(t))
    hop = torch.zeros_like(psi_dev)
    lat.hop(hr.EO_HOP_EO, U_dev, lat.odd(t), lat.even(hop))
    even = inputs.site_parity(L) == 0
    assert rel(got[even], eta[even] + 0.5 * lat.get_spinor(hop)[even]) <= 1e-13


# ------------------------------------------------------------------ host-buffer path
@pytest.mark.parametrize("prec", [0, 1])
def test_host_entry_points(hr, orc, prec):
    import torch
    L, m0 = (4, 6, 8, 8), -0.2
    U = rounded(inputs.haar_gauge(L, 1), prec)
    psi = rounded(inputs.gaussian_spinor(L, 2, 2), prec)
    lat = lattice(hr, L, 0, prec)
    ws = hr.device_buffer(hr.hr_host_workspace_bytes(lat.g))
    Uh = torch.from_numpy(U.astype(lat.cplx)).pin_memory()
    ph = torch.from_numpy(psi.astype(lat.cplx)).pin_memory()
    oh = torch.empty_like(ph).pin_memory()
    hr.hr_dirac_apply_host(lat.g, m0, Uh, ph, oh, ws, hr.stream_ptr())
    assert rel(oh.numpy(), orc.dirac(L, 0, m0, U, psi)) <= TOL[prec]
    hr.hr_dirac_eo_apply_host(lat.g, hr.EO_DHAT, m0, Uh, ph, oh, ws, hr.stream_ptr())
    assert rel(oh.numpy(), orc.dirac_eo(L, 0, m0, U, psi)) <= TOL[prec]
    hr.hr_dirac_eo_apply_host(lat.g, hr.EO_HOP_OE, m0, Uh, ph, oh, ws, hr.stream_ptr())
    assert rel(oh.numpy(), orc.hop(L, 0, 1, U, psi)) <= TOL[prec]


@pytest.mark.parametrize("prec", [0, 1])
def test_host_batch_with_resident_gauge(hr, orc, prec):
    """hr_gauge_upload_host once, then hr_apply_host_batch on 5 right-hand sides (the double-buffered pipeline wraps
    around twice): full D, the bare hop, Dhat, and the clover-improved Dhat and D_sw, each result against the oracle"""
    import torch
    L, m0, csw = (4, 6, 8, 8), -0.25, 1.2
    U = rounded(inputs.weak_gauge(L, 0.3, 1), prec)
    lat = lattice(hr, L, 0, prec)
    g, st = lat.g, hr.stream_ptr()
    Uh = torch.from_numpy(U.astype(lat.cplx)).pin_memory()
    u_dev = lat.empty_gauge(hr.REP_FUND)
    hr.hr_gauge_upload_host(g, hr.REP_FUND, Uh, u_dev, hr.device_buffer(hr.hr_canonical_gauge_bytes(g, hr.REP_FUND)), st)
    assert torch.equal(u_dev, lat.put_gauge_fund(U))
    fwd, inv = lat.clover_build(m0, csw, u_dev)
    A = orc.clover_dense(L, 4.0 + m0, csw, U)
    Ainv = orc.invert(A)
    C = A - (4.0 + m0) * np.eye(8)[None]
    psis = [rounded(inputs.gaussian_spinor(L, 2, 2 + i), prec) for i in range(5)]
    ins = [torch.from_numpy(p.astype(lat.cplx)).pin_memory() for p in psis]
    outs = [torch.empty_like(a).pin_memory() for a in ins]
    ws = hr.device_buffer(hr.hr_host_batch_workspace_bytes(g))
    cases = [
        (hr.HOST_DIRAC, None, None, lambda p: orc.dirac(L, 0, m0, U, p)),
        (hr.EO_HOP_EO, None, None, lambda p: orc.hop(L, 0, 0, U, p)),
        (hr.EO_DHAT, None, None, lambda p: orc.dirac_eo(L, 0, m0, U, p)),
        (hr.EO_DHAT, fwd, inv, lambda p: orc.dirac_eo_clover(L, U, A, Ainv, p)),
        (hr.HOST_DIRAC, fwd, None, lambda p: orc.dirac_clover(L, m0, U, C, p)),
    ]
    for op, cf, ci, want in cases:
        for o in outs:
            o.fill_(7.0)
        hr.hr_apply_host_batch(g, op, m0, u_dev, cf, ci, ins, outs, ws, st)
        for p, o in zip(psis, outs):
            assert rel(o.numpy(), want(p)) <= TOL[prec], (op, cf is not None)
    hr.hr_apply_host_batch(g, hr.HOST_DIRAC, m0, u_dev, None, None, [], [], ws, st)      # empty batch: nothing to do
    with pytest.raises(hr.HrError):
        hr.hr_apply_host_batch(g, hr.HOST_DIRAC, m0, u_dev, fwd, inv, ins[:1], outs[:1], ws, st)
    # one pipeline across different operators (hr_apply_host_ops): item i applies ops[i]
    ops = [hr.EO_HOP_OE, hr.EO_HOP_EO, hr.HOST_DIRAC, hr.EO_DHAT, hr.HOST_DIRAC]
    wants = [lambda p: orc.hop(L, 0, 1, U, p), lambda p: orc.hop(L, 0, 0, U, p), lambda p: orc.dirac(L, 0, m0, U, p),
             lambda p: orc.dirac_eo(L, 0, m0, U, p), lambda p: orc.dirac(L, 0, m0, U, p)]
    for o in outs:
        o.fill_(7.0)
    hr.hr_apply_host_ops(g, ops, m0, u_dev, None, None, ins, outs, ws, st)
    for p_, o, w in zip(psis, outs, wants):
        assert rel(o.numpy(), w(p_)) <= TOL[prec]
    # with clover blocks: Dhat items use both block fields, full-D items the forward one
    for o in outs:
        o.fill_(7.0)
    hr.hr_apply_host_ops(g, [hr.EO_DHAT, hr.HOST_DIRAC], m0, u_dev, fwd, inv, ins[:2], outs[:2], ws, st)
    assert rel(outs[0].numpy(), orc.dirac_eo_clover(L, U, A, Ainv, psis[0])) <= TOL[prec]
    assert rel(outs[1].numpy(), orc.dirac_clover(L, m0, U, C, psis[1])) <= TOL[prec]
    with pytest.raises(hr.HrError):
        hr.hr_apply_host_ops(g, [9], m0, u_dev, None, None, ins[:1], outs[:1], ws, st)


def test_native_library_is_the_one_loaded(hr):
    """the product path is the in-tree shared object, and it counts its own launches"""
    import torch
    n0 = hr.hr_launch_count()
    lat = lattice(hr, (4, 4, 4, 4))
    lat.put_spinor(inputs.gaussian_spinor((4, 4, 4, 4), 2, 2))
    torch.cuda.synchronize()
    assert hr.hr_launch_count() == n0 + 1
    with open("/proc/self/maps") as f:
        assert "paper_2411_18511_b200/libhr_dslash.so" in f.read()


# ------------------------------------------------------------------ bounds (compute-sanitizer is closed on this pool)
@pytest.mark.parametrize("L,rep", [((8, 2, 8, 6), 0), ((8, 4, 4, 16), 0), ((6, 2, 4, 12), 1), ((2, 2, 2, 2), 0), ((2, 4, 6, 8), 1)])
@pytest.mark.parametrize("prec", [0, 1])
def test_operators_write_only_their_output(hr, L, rep, prec):
    """every output / temporary buffer sits between two guard regions holding a byte pattern; after all hop
    variants (both kernels, every epilogue) the guards are intact and bytes outside the output are unchanged"""
    import torch
    N = 2 if rep == 0 else 3
    U = inputs.haar_gauge(L, 1)
    psi = inputs.gaussian_spinor(L, N, 2)
    G = 1 << 16
    for kernel in kernels_for(hr, L, rep, prec):
        lat = lattice(hr, L, rep, prec, kernel)
        Uf = lat.put_gauge_fund(U)
        U_dev = Uf if rep == 0 else lat.represent(Uf)
        psi_dev = lat.put_spinor(psi)
        half = lat.half
        arena = torch.full((4 * G + 2 * half + half,), 0xA5, dtype=torch.uint8, device="cuda")
        out = arena[G:G + 2 * half]
        tmp = arena[3 * G + 2 * half:3 * G + 3 * half]
        st = hr.stream_ptr()

        def guards_ok():
            torch.cuda.synchronize()
            a = arena
            return bool((a[:G] == 0xA5).all() and (a[G + 2 * half:3 * G + 2 * half] == 0xA5).all() and (a[3 * G + 3 * half:] == 0xA5).all())

        hr.hr_dirac_apply(lat.g, -0.2, U_dev, psi_dev, out, st)
        assert guards_ok(), ("dirac", kernel)
        out.fill_(0xA5)
        hr.hr_dirac_eo_apply(lat.g, hr.EO_HOP_OE, 0.0, U_dev, None, None, lat.even(psi_dev), out[half:], None, st)
        assert guards_ok() and bool((out[:half] == 0xA5).all()), ("hop_oe", kernel)
        out.fill_(0xA5)
        hr.hr_dirac_eo_apply(lat.g, hr.EO_DHAT, -0.2, U_dev, None, None, lat.even(psi_dev), out[:half], tmp, st)
        assert guards_ok() and bool((out[half:] == 0xA5).all()), ("dhat", kernel)
        if rep == 0:
            fwd, inv = lat.clover_build(-0.25, 1.2, Uf)
            out.fill_(0xA5)
            tmp.fill_(0xA5)
            hr.hr_dirac_eo_apply(lat.g, hr.EO_DHAT, -0.25, U_dev, fwd, inv, lat.even(psi_dev), out[:half], tmp, st)
            assert guards_ok() and bool((out[half:] == 0xA5).all()), ("dhat clover", kernel)
            out.fill_(0xA5)
            hr.hr_clover_apply(lat.g, hr.ODD, inv, lat.odd(psi_dev), out[half:], st)
            assert guards_ok() and bool((out[:half] == 0xA5).all()), ("clover odd", kernel)


# ------------------------------------------------------------------ S1: CG on Dhat^dag Dhat
@pytest.mark.parametrize("L,rep", [((8, 4, 4, 8), 0), ((4, 4, 4, 4), 1), ((8, 2, 8, 6), 0)])
@pytest.mark.parametrize("prec", [0, 1])
def test_cg_solution_matches_the_oracle(hr, orc, L, rep, prec):
    """hr_cg_solve against the oracle's textbook CG (O8) on the same system: same solution up to the stopping
    tolerance times the conditioning, about the same iteration count, and a true residual (evaluated with the
    ORACLE's operator on the GPU's solution) at the requested level"""
    import torch
    m0 = -0.2
    N = 2 if rep == 0 else 3
    Uf = rounded(inputs.haar_gauge(L, 1), prec)
    U = Uf if rep == 0 else rounded(orc.represent(Uf)[0], prec)
    b = rounded(inputs.gaussian_spinor(L, N, 2), prec)
    even = inputs.site_parity(L) == 0
    b[~even] = 0
    tol = 1e-12 if prec == 0 else 2e-6
    x_orc, it_orc, _ = orc.cg_normal(L, rep, m0, U, b, tol=tol, max_iter=1000, nthreads=NTHREADS)
    g5 = np.array([1.0, 1.0, -1.0, -1.0])[None, :, None]
    for kernel in kernels_for(hr, L, rep, prec):
        lat = lattice(hr, L, rep, prec, kernel)
        U_dev = lat.put_gauge_fund(U) if rep == 0 else lat.put_gauge_adj(U)
        b_dev = lat.put_spinor(b)
        x_half, it, relres = lat.cg(m0, U_dev, lat.even(b_dev), tol, 1000, check_every=3)
        # the count may differ by the rounding of the residual norm at the threshold, plus the check interval
        assert relres <= tol and it_orc - 2 <= it <= it_orc + 6, (it, it_orc, relres)
        full = torch.zeros_like(b_dev)
        lat.even(full).copy_(x_half)
        x = lat.get_spinor(full).astype(np.complex128)
        assert not x[~even].any()
        assert rel(x, x_orc) <= (1e-9 if prec == 0 else 2e-3), kernel
        t = orc.dirac_eo(L, rep, m0, U, x, nthreads=NTHREADS)
        r = b - g5 * orc.dirac_eo(L, rep, m0, U, g5 * t, nthreads=NTHREADS)
        assert np.linalg.norm(r) <= (10 * tol if prec == 0 else 2e-5) * np.linalg.norm(b)


def test_cg_with_clover_and_repeatability(hr, orc):
    """the clover-improved system (E2 inside the solver) against the oracle, and two solves give the same bits"""
    import torch
    L, m0, csw = (4, 4, 4, 8), -0.25, 1.2
    U = inputs.weak_gauge(L, 0.3, 1)
    b = inputs.gaussian_spinor(L, 2, 2)
    even = inputs.site_parity(L) == 0
    b[~even] = 0
    A, Ainv = clover_oracle(orc, L, U, m0, csw)
    x_orc, it_orc, _ = orc.cg_normal(L, 0, m0, U, b, tol=1e-12, max_iter=500, nthreads=NTHREADS, A=A, Ainv=Ainv)
    lat = lattice(hr, L, 0, 0)
    U_dev, b_dev = lat.put_gauge_fund(U), lat.put_spinor(b)
    fwd, inv = lat.clover_build(m0, csw, U_dev)
    sols = []
    for _ in range(2):
        x_half, it, relres = lat.cg(m0, U_dev, lat.even(b_dev), 1e-12, 500, clover_fwd=fwd, clover_inv=inv, check_every=1)
        assert abs(it - it_orc) <= 2 and relres <= 1e-12, (it, it_orc)
        sols.append(x_half.clone())
    assert torch.equal(sols[0], sols[1])
    full = torch.zeros_like(b_dev)
    lat.even(full).copy_(sols[0])
    assert rel(lat.get_spinor(full), x_orc) <= 1e-9


# ------------------------------------------------------------------ C1x: exponential clover
@pytest.mark.parametrize("L", [(4, 4, 4, 4), (2, 4, 6, 8), (8, 2, 8, 6)])
@pytest.mark.parametrize("prec", [0, 1])
def test_exponential_clover(hr, orc, L, prec):
    """hr_clover_build_exp blocks and inverses against the oracle's O9 (eigendecomposition route), then C2/C3 and the
    even-odd operator E2 with those blocks"""
    import torch
    m0, csw = -0.25, 1.2
    U = rounded(inputs.weak_gauge(L, 0.3, 1), prec)
    psi = rounded(inputs.gaussian_spinor(L, 2, 2), prec)
    A, Ainv = orc.clover_exp_dense(L, 4.0 + m0, csw, U, nthreads=NTHREADS)
    bf, bi = dense_to_blocks(A), dense_to_blocks(Ainv)
    tol_blk = 1e-13 if prec == 0 else 1e-6
    for kernel in kernels_for(hr, L, 0, prec):
        lat = lattice(hr, L, 0, prec, kernel)
        U_dev, psi_dev = lat.put_gauge_fund(U), lat.put_spinor(psi)
        fwd, inv = lat.clover_build(m0, csw, U_dev, exponential=True)
        assert np.linalg.norm(lat.get_clover(fwd) - bf) <= tol_blk * np.linalg.norm(bf)
        assert np.linalg.norm(lat.get_clover(inv) - bi) <= tol_blk * np.linalg.norm(bi)
        got = lat.get_spinor(lat.clover_apply(hr.BOTH, fwd, psi_dev))
        assert rel(got, orc.site_matvec(L, 3, A, psi)) <= TOL[prec]
        got = lat.get_spinor(lat.clover_apply(hr.BOTH, inv, psi_dev))
        assert rel(got, orc.site_matvec(L, 3, Ainv, psi)) <= TOL[prec]
        out = torch.zeros_like(psi_dev)
        lat.dhat(m0, U_dev, lat.even(psi_dev), lat.even(out), clover_fwd=fwd, clover_inv=inv)
        want = orc.dirac_eo_clover(L, U, A, Ainv, psi, nthreads=NTHREADS)
        assert rel(lat.get_spinor(out), want) <= TOL[prec], kernel


@pytest.mark.parametrize("L,rep", [((8, 4, 4, 8), 0), ((4, 4, 4, 4), 1), ((8, 2, 8, 6), 0)])
def test_mixed_precision_cg(hr, orc, L, rep):
    """hr_cg_solve_mixed (fp64 defect correction around fp32 CG) reaches the oracle's fp64 solution: same x, a true
    residual (evaluated with the ORACLE's operator) at the requested 1e-12, in a handful of corrections"""
    import torch
    m0, tol = -0.2, 1e-12
    N = 2 if rep == 0 else 3
    Uf = inputs.haar_gauge(L, 1)
    U = Uf if rep == 0 else orc.represent(Uf)[0]
    b = inputs.gaussian_spinor(L, N, 2)
    even = inputs.site_parity(L) == 0
    b[~even] = 0
    x_orc, it_orc, _ = orc.cg_normal(L, rep, m0, U, b, tol=tol, max_iter=1000, nthreads=NTHREADS)
    g5 = np.array([1.0, 1.0, -1.0, -1.0])[None, :, None]
    for kernel in kernels_for(hr, L, rep, 0):
        l64, l32 = lattice(hr, L, rep, 0, kernel), lattice(hr, L, rep, 1, kernel)
        put = (lambda lat: lat.put_gauge_fund(U)) if rep == 0 else (lambda lat: lat.put_gauge_adj(U))
        U64, U32 = put(l64), put(l32)
        b_dev = l64.put_spinor(b)
        x_half = l64.empty_spinor(hr.EVEN)
        ws = hr.device_buffer(hr.hr_cg_mixed_workspace_bytes(l64.g))
        outer, inner, relres = hr.hr_cg_solve_mixed(l64.g, m0, U64, U32, l64.even(b_dev), x_half, ws, tol, 1e-4, 20, 1000, 5, hr.stream_ptr())
        assert relres <= tol and 2 <= outer <= 6, (outer, inner, relres)
        assert inner <= 3 * it_orc + 30, (inner, it_orc)
        full = torch.zeros_like(b_dev)
        l64.even(full).copy_(x_half)
        x = l64.get_spinor(full)
        assert not x[~even].any()
        assert rel(x, x_orc) <= 1e-9, kernel
        t = orc.dirac_eo(L, rep, m0, U, x, nthreads=NTHREADS)
        r = b - g5 * orc.dirac_eo(L, rep, m0, U, g5 * t, nthreads=NTHREADS)
        assert np.linalg.norm(r) <= 10 * tol * np.linalg.norm(b)


# ------------------------------------------------------------------ the widened rows at the bench size
def test_48to4_cg_and_exponential_clover(hr, orc, big_inputs):
    """at 48^4, in the launch configuration bench.py times: (i) hr_cg_solve and hr_cg_solve_mixed reach a TRUE residual
    (evaluated with the oracle's Dhat on the GPU's solution) at the requested level; (ii) hr_clover_build_exp
    blocks against the oracle's O9 on a slab of sites"""
    import torch
    L, U, psi = big_inputs
    m0 = -0.2
    even = inputs.site_parity(L) == 0
    b = psi.copy()
    b[~even] = 0
    l64, l32 = lattice(hr, L, 0, 0), lattice(hr, L, 0, 1)
    U64, U32 = l64.put_gauge_fund(U), l32.put_gauge_fund(U)
    b_dev = l64.put_spinor(b)
    g5 = np.array([1.0, 1.0, -1.0, -1.0])[None, :, None]

    def true_relres(x_half):
        full = torch.zeros_like(b_dev)
        l64.even(full).copy_(x_half)
        x = l64.get_spinor(full)
        t = orc.dirac_eo(L, 0, m0, U, x, nthreads=NTHREADS)
        r = b - g5 * orc.dirac_eo(L, 0, m0, U, g5 * t, nthreads=NTHREADS)
        return float(np.linalg.norm(r) / np.linalg.norm(b))

    x_half, it, relres = l64.cg(m0, U64, l64.even(b_dev), 1e-10, 500)
    assert relres <= 1e-10 and 10 < it < 200
    assert true_relres(x_half) <= 2e-10
    xm = l64.empty_spinor(hr.EVEN)
    ws = hr.device_buffer(hr.hr_cg_mixed_workspace_bytes(l64.g))
    outer, inner, rel_m = hr.hr_cg_solve_mixed(l64.g, m0, U64, U32, l64.even(b_dev), xm, ws, 1e-12, 1e-4, 20, 500, 5, hr.stream_ptr())
    assert rel_m <= 1e-12 and outer <= 6
    assert true_relres(xm) <= 1e-11
    # (ii) exponential clover blocks on the first 2 x 48^3 sites
    m0c, csw = -0.25, 1.2
    Uw = inputs.weak_gauge(L, 0.3, 1)
    fwd, inv = l64.clover_build(m0c, csw, l64.put_gauge_fund(Uw), exponential=True)
    n = 2 * 48 ** 3
    A, Ainv = orc.clover_exp_dense(L, 4.0 + m0c, csw, Uw, nthreads=NTHREADS, begin=0, end=n)
    bf, bi = dense_to_blocks(A), dense_to_blocks(Ainv)
    assert np.linalg.norm(l64.get_clover(fwd)[:n] - bf) <= 1e-13 * np.linalg.norm(bf)
    assert np.linalg.norm(l64.get_clover(inv)[:n] - bi) <= 1e-13 * np.linalg.norm(bi)


# ------------------------------------------------------------------ clover in the adjoint representation
@pytest.mark.parametrize("L", [(4, 4, 4, 4), (2, 4, 6, 8), (2, 2, 2, 2), (8, 2, 8, 6)])
@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("exponential", [False, True])
def test_adjoint_clover(hr, orc, L, prec, exponential):
    """6x6 blocks and inverses (regular and exponential) against the oracle's O10, C2/C3 on them, the even-odd
    operator with clover (E2) and the full clover-improved operator in the adjoint representation; stored links and
    links rebuilt on the fly"""
    import torch
    m0, csw = -0.25, 1.2
    d = 4.0 + m0
    Uf = rounded(inputs.weak_gauge(L, 0.3, 1), prec)
    R, _ = orc.represent(Uf)
    psi = rounded(inputs.gaussian_spinor(L, 3, 2), prec)
    if exponential:
        A, Ainv = orc.clover_exp_dense_adj(L, d, csw, R)      # O11, pinned by P19
    else:
        A = orc.clover_dense_adj(L, d, csw, R)
        Ainv = np.linalg.inv(A)
    bf, bi = dense_to_blocks(A), dense_to_blocks(Ainv)
    tol_blk = 1e-13 if prec == 0 else 1e-6
    want_dhat = orc.dirac_eo_clover_adj(L, R, A, Ainv, psi, nthreads=NTHREADS)
    H = orc.hop(L, 1, 0, R, psi, nthreads=NTHREADS)
    H = orc.hop(L, 1, 1, R, psi, nthreads=NTHREADS, out=H)
    want_dsw = orc.site_matvec_n(A, psi) - 0.5 * H
    from paper_2411_18511_b200.lattice import Lattice
    for storage in (hr.LINKS_COMPRESSED, hr.LINKS_ONTHEFLY):
        for kernel in kernels_for(hr, L, 1, prec):
            lat = Lattice(L, hr.REP_ADJ, prec, kernel, link_storage=storage)
            Uf_dev, psi_dev = lat.put_gauge_fund(Uf), lat.put_spinor(psi)
            U_dev = Uf_dev if storage == hr.LINKS_ONTHEFLY else lat.put_gauge_adj(rounded(R, prec))
            fwd, inv = lat.clover_build(m0, csw, Uf_dev, exponential=exponential)
            assert np.linalg.norm(lat.get_clover(fwd) - bf) <= tol_blk * np.linalg.norm(bf)
            assert np.linalg.norm(lat.get_clover(inv) - bi) <= tol_blk * np.linalg.norm(bi)
            got = lat.get_spinor(lat.clover_apply(hr.BOTH, fwd, psi_dev))
            assert rel(got, orc.site_matvec_n(A, psi)) <= TOL[prec]
            half = torch.zeros_like(psi_dev)
            lat.clover_apply(hr.ODD, inv, lat.odd(psi_dev), lat.odd(half))
            assert rel(lat.get_spinor(half), orc.site_matvec_n(Ainv, psi, inputs.site_parity(L) == 1)) <= TOL[prec]
            out = torch.zeros_like(psi_dev)
            lat.dhat(m0, U_dev, lat.even(psi_dev), lat.even(out), clover_fwd=fwd, clover_inv=inv)
            assert rel(lat.get_spinor(out), want_dhat) <= TOL[prec], (storage, kernel)
            assert rel(lat.get_spinor(lat.dirac_clover(U_dev, fwd, psi_dev)), want_dsw) <= TOL[prec], (storage, kernel)


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (2, 4, 6, 8)])
@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("exponential", [False, True])
@pytest.mark.parametrize("two_rows", [False, True])
def test_su3_clover(hr, orc, L, prec, exponential, two_rows):
    """complex 3 x 3 links (HR_REP_SU3): 6 x 6 blocks and inverses (regular and exponential) against the oracle's O12 (pinned by
    P22), C2/C3 on them, the even-odd operator with clover (E2), the full clover-improved operator and the CG solver on the
    clover-improved system; links stored in full and as two rows"""
    import torch
    from paper_2411_18511_b200.lattice import Lattice
    m0, csw = -0.25, 1.2
    d = 4.0 + m0
    U = rounded(inputs.haar_gauge_su3(L, 1), prec)
    psi = rounded(inputs.gaussian_spinor(L, 3, 2), prec)
    if exponential:
        A, Ainv = orc.clover_exp_dense_su3(L, d, csw, U)
    else:
        A = orc.clover_dense_su3(L, d, csw, U)
        Ainv = np.linalg.inv(A)
    bf, bi = dense_to_blocks(A), dense_to_blocks(Ainv)
    tol_blk = 1e-13 if prec == 0 else 2e-6
    want_dhat = orc.dirac_eo_clover_n(L, 2, U, A, Ainv, psi, nthreads=NTHREADS)
    H = orc.hop(L, 2, 0, U, psi, nthreads=NTHREADS)
    H = orc.hop(L, 2, 1, U, psi, nthreads=NTHREADS, out=H)
    want_dsw = orc.site_matvec_n(A, psi) - 0.5 * H
    lat = Lattice(L, hr.REP_SU3, prec, 0, link_storage=hr.LINKS_COMPRESSED if two_rows else hr.LINKS_FULL)
    U_dev, psi_dev = lat.put_gauge_su3(U), lat.put_spinor(psi)
    fwd, inv = lat.clover_build(m0, csw, U_dev, exponential=exponential)
    assert np.linalg.norm(lat.get_clover(fwd) - bf) <= tol_blk * np.linalg.norm(bf)
    assert np.linalg.norm(lat.get_clover(inv) - bi) <= tol_blk * np.linalg.norm(bi)
    got = lat.get_spinor(lat.clover_apply(hr.BOTH, fwd, psi_dev))
    assert rel(got, orc.site_matvec_n(A, psi)) <= TOL[prec]
    half = torch.zeros_like(psi_dev)
    lat.clover_apply(hr.ODD, inv, lat.odd(psi_dev), lat.odd(half))
    assert rel(lat.get_spinor(half), orc.site_matvec_n(Ainv, psi, inputs.site_parity(L) == 1)) <= TOL[prec]
    out = torch.zeros_like(psi_dev)
    lat.dhat(m0, U_dev, lat.even(psi_dev), lat.even(out), clover_fwd=fwd, clover_inv=inv)
    assert rel(lat.get_spinor(out), want_dhat) <= TOL[prec]
    assert rel(lat.get_spinor(lat.dirac_clover(U_dev, fwd, psi_dev)), want_dsw) <= TOL[prec]
    if prec == 0 and L == (4, 4, 4, 4) and not exponential:
        b = psi.copy()
        b[inputs.site_parity(L) == 1] = 0
        dh = lambda v: orc.dirac_eo_clover_n(L, 2, U, A, Ainv, v, nthreads=NTHREADS)
        x_orc, it_orc, _ = orc.cg_normal(L, 2, m0, U, b, tol=1e-12, max_iter=500, dhat=dh)
        b_dev = lat.put_spinor(b)
        x_half, it, relres = lat.cg(m0, U_dev, lat.even(b_dev), 1e-12, 500, clover_fwd=fwd, clover_inv=inv, check_every=1)
        full = torch.zeros_like(b_dev)
        lat.even(full).copy_(x_half)
        assert relres <= 1e-12 and abs(it - it_orc) <= 2 and rel(lat.get_spinor(full), x_orc) <= 1e-9


@pytest.mark.parametrize("rep", [0, 1])
def test_cg_with_clover_all_variants(hr, orc, rep):
    """hr_cg_solve and hr_cg_solve_mixed_clover on the clover-improved even-odd system, fundamental and adjoint,
    against the oracle's CG (O8) on the oracle's operators (O7 / its adjoint form)"""
    import torch
    L, m0, csw, tol = (4, 4, 4, 8), -0.25, 1.2, 1e-12
    d = 4.0 + m0
    N = 2 if rep == 0 else 3
    Uf = inputs.weak_gauge(L, 0.3, 1)
    b = inputs.gaussian_spinor(L, N, 2)
    even = inputs.site_parity(L) == 0
    b[~even] = 0
    if rep == 0:
        U = Uf
        A, Ainv = clover_oracle(orc, L, Uf, m0, csw)
        dhat = lambda v: orc.dirac_eo_clover(L, Uf, A, Ainv, v, nthreads=NTHREADS)
    else:
        U = orc.represent(Uf)[0]
        A = orc.clover_dense_adj(L, d, csw, U)
        Ainv = np.linalg.inv(A)
        dhat = lambda v: orc.dirac_eo_clover_adj(L, U, A, Ainv, v, nthreads=NTHREADS)
    x_orc, it_orc, _ = orc.cg_normal(L, rep, m0, U, b, tol=tol, max_iter=1000, dhat=dhat)
    l64, l32 = lattice(hr, L, rep, 0), lattice(hr, L, rep, 1)
    put = (lambda lat: lat.put_gauge_fund(U)) if rep == 0 else (lambda lat: lat.put_gauge_adj(U))
    U64, U32 = put(l64), put(l32)
    f64, i64 = l64.clover_build(m0, csw, l64.put_gauge_fund(Uf))
    f32, i32 = l32.clover_build(m0, csw, l32.put_gauge_fund(Uf))
    b_dev = l64.put_spinor(b)

    def solution(x_half):
        full = torch.zeros_like(b_dev)
        l64.even(full).copy_(x_half)
        return l64.get_spinor(full)

    x_half, it, relres = l64.cg(m0, U64, l64.even(b_dev), tol, 1000, clover_fwd=f64, clover_inv=i64, check_every=1)
    assert relres <= tol and abs(it - it_orc) <= 2
    assert rel(solution(x_half), x_orc) <= 1e-9
    xm = l64.empty_spinor(hr.EVEN)
    ws = hr.device_buffer(hr.hr_cg_mixed_workspace_bytes(l64.g))
    outer, inner, rel_m = hr.hr_cg_solve_mixed_clover(l64.g, m0, U64, U32, f64, i64, f32, i32, l64.even(b_dev), xm, ws, tol, 1e-4, 20, 1000, 5,
                                                      hr.stream_ptr())
    assert rel_m <= tol and 2 <= outer <= 6
    assert rel(solution(xm), x_orc) <= 1e-9


def test_tiled_kernel_soak_is_bitwise_repeatable(hr):
    """2 x 2000 launches of the tiled kernels (full D with both parities per CTA, and Dhat) on a small lattice: every
    output equals the first one bit for bit — a rare producer/consumer ordering slip in the mbarrier pipeline would show
    up here as a changed word (or a hang, caught by the test timeout)"""
    import torch
    for L, rep, prec in (((8, 2, 8, 6), 0, 0), ((8, 4, 4, 16), 1, 0), ((4, 2, 4, 52), 0, 1)):
        g = hr.geom(L, rep, prec, hr.LINKS_COMPRESSED, hr.KERNEL_TILED)
        assert hr.hr_kernel_name(g) == "tiled"
        U = torch.randn(hr.hr_gauge_bytes(g, rep) // 4, device="cuda").view(torch.uint8)
        psi = torch.randn(hr.hr_spinor_bytes(g, hr.BOTH) // 4, device="cuda").view(torch.uint8)
        out = torch.zeros_like(psi)
        half = psi.numel() // 2
        tmp = torch.empty(half, device="cuda", dtype=torch.uint8)
        st = hr.stream_ptr()
        ref = None
        for i in range(2000):
            hr.hr_dirac_apply(g, -0.2, U, psi, out, st)
            hr.hr_dirac_eo_apply(g, hr.EO_DHAT, -0.2, U, None, None, psi[:half], out[:half], tmp, st)
            if i % 250 == 0:
                if ref is None:
                    ref = out.clone()
                else:
                    assert torch.equal(ref, out), (L, rep, prec, i)
        torch.cuda.synchronize()


def test_clover_inverse_of_indefinite_blocks(hr, orc):
    """4 + m0 small against |csw F|: A(x) is indefinite and the unpivoted elimination would divide by tiny diagonal
    pivots; the build's Gauss-Jordan with partial pivoting must still reproduce the oracle's dense inverse, and
    hr_clover_count_nonfinite must report 0 non-finite entries"""
    import torch
    L, m0, csw = (4, 4, 4, 4), -3.95, 4.0
    U = inputs.weak_gauge(L, 0.6, 1)
    A = orc.clover_dense(L, 4.0 + m0, csw, U)
    ev = np.linalg.eigvalsh(A)
    assert ev.min() < -0.1 and ev.max() > 0.1 and np.abs(ev).min() > 1e-4     # indefinite, invertible
    Ainv = np.linalg.inv(A)
    lat = lattice(hr, L, 0, 0)
    fwd, inv = lat.clover_build(m0, csw, lat.put_gauge_fund(U))
    bf, bi = dense_to_blocks(A), dense_to_blocks(Ainv)
    assert np.linalg.norm(lat.get_clover(fwd) - bf) <= 1e-13 * np.linalg.norm(bf)
    assert np.linalg.norm(lat.get_clover(inv) - bi) <= 1e-11 * np.linalg.norm(bi)
    count = torch.full((1,), -1, dtype=torch.int64, device="cuda")
    for blocks in (fwd, inv):
        hr.hr_clover_count_nonfinite(lat.g, blocks, count, hr.stream_ptr())
        assert int(count.item()) == 0
    inv.view(torch.float64)[5] = float("nan")
    inv.view(torch.float64)[77] = float("inf")
    hr.hr_clover_count_nonfinite(lat.g, inv, count, hr.stream_ptr())
    assert int(count.item()) == 2


# ------------------------------------------------------------------ complex 3 x 3 links (HR_REP_SU3)
@pytest.mark.parametrize("L", [(4, 4, 4, 4), (2, 2, 2, 2), (2, 4, 6, 8), (6, 2, 4, 12)])
@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("two_rows", [False, True])
def test_su3_small_lattices(hr, orc, L, prec, two_rows):
    """Haar SU(3) links, 3 complex colours: pack/unpack round trip, bare hops, full D, Dhat and the CG solver against the
    oracle's rep-2 operators (pinned by P21); the clover calls refuse the representation.  two_rows: HR_LINKS_COMPRESSED — the
    device keeps the first two rows of a link and the kernels (and unpack) rebuild the third, row2 = conj(row0 x row1)."""
    import torch
    from paper_2411_18511_b200.lattice import Lattice
    m0 = -0.2
    U = rounded(inputs.haar_gauge_su3(L, 1), prec)
    psi = rounded(inputs.gaussian_spinor(L, 3, 2), prec)
    lat = Lattice(L, hr.REP_SU3, prec, 0, link_storage=hr.LINKS_COMPRESSED if two_rows else hr.LINKS_FULL)
    assert hr.hr_kernel_name(lat.g) == "generic"
    U_dev = lat.put_gauge_su3(U)
    assert hr.hr_gauge_bytes(lat.g, hr.REP_SU3) == inputs.volume(L) * 4 * (12 if two_rows else 18) * (8 if prec == 0 else 4)
    back = lat.get_gauge_su3(U_dev)
    if two_rows:      # rows 0 and 1 are a permutation, row 2 is recomputed from them
        assert np.array_equal(back[:, :, :2], U.astype(lat.cplx)[:, :, :2])
        assert np.abs(back[:, :, 2] - U[:, :, 2]).max() <= (1e-15 if prec == 0 else 5e-7)
    else:
        assert np.array_equal(back, U.astype(lat.cplx))
    want = oracle_ops(orc, L, 2, U, psi, m0)
    got = gpu_ops(hr, lat, U_dev, psi, m0)
    for k in want:
        assert rel(got[k], want[k]) <= TOL[prec], k
    f, bc, _ = hr.hr_dirac_flops_bytes(lat.g, hr.OP_HOP)
    w = 8 if prec == 0 else 4
    assert f == 1320.0 and bc == 2 * 24 * w + 8 * (12 if two_rows else 18) * w
    if prec == 0 and L == (4, 4, 4, 4):
        b = psi.copy()
        b[inputs.site_parity(L) == 1] = 0
        x_orc, it_orc, _ = orc.cg_normal(L, 2, m0, U, b, tol=1e-12, max_iter=500, nthreads=NTHREADS)
        b_dev = lat.put_spinor(b)
        x_half, it, relres = lat.cg(m0, U_dev, lat.even(b_dev), 1e-12, 500, check_every=1)
        full = torch.zeros_like(b_dev)
        lat.even(full).copy_(x_half)
        assert relres <= 1e-12 and abs(it - it_orc) <= 2 and rel(lat.get_spinor(full), x_orc) <= 1e-9


@pytest.mark.parametrize("L", [(4, 4, 4, 4), (2, 4, 6, 8), (6, 2, 4, 12)])
@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("two_rows", [False, True])
def test_su3_antisymmetric_representation(hr, orc, L, prec, two_rows):
    """hr_represent_gauge_antisym (the 2 x 2 minors of a link) against the oracle's O13 (trace definition, pinned by P23), link by
    link; the result is special unitary; and the operators of HR_REP_SU3 on the represented field against the oracle's rep-2
    operators on the oracle's represented field.  Wrong representation / aliased buffers are refused."""
    from paper_2411_18511_b200.lattice import Lattice
    m0 = -0.2
    U = rounded(inputs.haar_gauge_su3(L, 1), prec)
    psi = rounded(inputs.gaussian_spinor(L, 3, 2), prec)
    lat = Lattice(L, hr.REP_SU3, prec, 0, link_storage=hr.LINKS_COMPRESSED if two_rows else hr.LINKS_FULL)
    U_dev = lat.put_gauge_su3(U)
    R_dev = lat.represent_antisym(U_dev)
    R_want = orc.represent_antisym_su3(U)
    R_got = lat.get_gauge_su3(R_dev).astype(np.complex128)
    # entries are sums of two products of numbers of modulus <= 1; with two rows stored the third row of U (and of R) is rebuilt
    tol = (1e-15 if prec == 0 else 5e-7) * (4 if two_rows else 1)
    assert np.abs(R_got - R_want).max() <= tol
    eye = np.eye(3)
    assert np.abs(R_got @ np.conj(np.swapaxes(R_got, -1, -2)) - eye).max() <= 10 * tol
    assert np.abs(np.linalg.det(R_got) - 1).max() <= 10 * tol
    assert np.array_equal(lat.get_gauge_su3(U_dev)[:, :, :2], U.astype(lat.cplx)[:, :, :2])      # the input field is untouched
    want = oracle_ops(orc, L, 2, R_want, psi, m0)
    got = gpu_ops(hr, lat, R_dev, psi, m0)
    for k in want:
        assert rel(got[k], want[k]) <= TOL[prec], k
    with pytest.raises(hr.HrError) as e:
        hr.hr_represent_gauge_antisym(lat.g, U_dev, U_dev, hr.stream_ptr())
    assert e.value.status == hr.EINVAL
    with pytest.raises(hr.HrError) as e:
        hr.hr_represent_gauge_antisym(hr.geom(L, hr.REP_FUND, prec), U_dev, R_dev, hr.stream_ptr())
    assert e.value.status == hr.EUNSUPPORTED


def test_48to4_host_batch_on_sampled_sites(hr, orc, big_inputs):
    """the gauge-resident host path at the bench size: hr_gauge_upload_host + hr_apply_host_batch of 3 right-hand sides (full D
    and Dhat, fp64) at 48^4, checked on sampled sites against the oracle's per-site operator"""
    import torch
    L, U, psi = big_inputs
    m0 = -0.2
    lat = lattice(hr, L, 0, 0)
    g, st = lat.g, hr.stream_ptr()
    Uh = torch.from_numpy(U).pin_memory()
    u_dev = lat.empty_gauge(hr.REP_FUND)
    ws = hr.device_buffer(max(hr.hr_host_batch_workspace_bytes(g), hr.hr_canonical_gauge_bytes(g, hr.REP_FUND)))
    hr.hr_gauge_upload_host(g, hr.REP_FUND, Uh, u_dev, ws, st)
    V = inputs.volume(L)
    ins = [torch.from_numpy(psi).pin_memory(), torch.from_numpy(np.ascontiguousarray(psi[::-1])).pin_memory(), torch.from_numpy(1j * psi).pin_memory()]
    outs = [torch.empty_like(a).pin_memory() for a in ins]
    sites = np.unique(np.concatenate([np.array([0, 1, 47, 48, V - 1, V - 48, V // 2 + 5]), (inputs.normals(9, 9, 0, 40) * 1e9).astype(np.int64) % V]))
    hr.hr_apply_host_batch(g, hr.HOST_DIRAC, m0, u_dev, None, None, ins, outs, ws, st)
    for a, o in zip(ins, outs):
        want = orc.dirac_sites(L, 0, m0, U, a.numpy(), sites)
        assert rel(o.numpy()[sites], want) <= 1e-13
    hr.hr_apply_host_batch(g, hr.EO_HOP_OE, m0, u_dev, None, None, ins[:2], outs[:2], ws, st)
    odd = sites[inputs.site_parity(L)[sites] == 1]
    for a, o in zip(ins[:2], outs[:2]):
        assert rel(o.numpy()[odd], orc.hop_sites(L, 0, U, a.numpy(), odd)) <= 1e-13
        assert not o.numpy()[sites[inputs.site_parity(L)[sites] == 0]].any()
