"""hr_dhat_apply_static: the even-odd operator with its intermediate odd half field in the library's file-scope device array
(include/hr_dslash.h) — for callers that cannot call cudaMalloc.  The expected values are the EXISTING path's
(hr_dirac_eo_apply with a caller-owned tmp, itself checked against the oracle in test_gpu_parity.py) on the same inputs.

Named test_zz_* so that pytest collects it last: the suite runs with `pytest -x`."""
import numpy as np
import pytest

from paper_2411_18511_b200 import inputs

TOL = {0: 1e-13, 1: 1e-5}   # the bar of test_gpu_parity.py: relative L2 error, hr.PREC_F64 / hr.PREC_F32


@pytest.fixture(scope="module")
def hr():
    from paper_2411_18511_b200 import build, hr as _hr
    build.build()
    _hr.lib()
    return _hr


def rel(a, b):
    a, b = a.astype(np.complex128), b.astype(np.complex128)
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def test_lattice_beyond_the_static_scratch_is_refused(hr):
    """host logic only: the size check comes before any CUDA call, so no device is needed"""
    assert hr.STATIC_SCRATCH_BYTES == 8 << 20
    ok = hr.geom((16, 16, 16, 32), hr.REP_FUND, hr.PREC_F64)          # the largest fp64 SU(2)-fundamental lattice: exactly 8 MiB
    assert hr.hr_spinor_bytes(ok, hr.ODD) == hr.STATIC_SCRATCH_BYTES
    for L, rep, prec in (((16, 16, 16, 34), hr.REP_FUND, hr.PREC_F64), ((48, 48, 48, 48), hr.REP_FUND, hr.PREC_F32),
                         ((16, 16, 16, 32), hr.REP_ADJ, hr.PREC_F64), ((16, 16, 16, 32), hr.REP_SU3, hr.PREC_F64)):
        g = hr.geom(L, rep, prec)
        assert hr.hr_spinor_bytes(g, hr.ODD) > hr.STATIC_SCRATCH_BYTES
        with pytest.raises(hr.HrError) as e:
            hr.hr_dhat_apply_static(g, -0.2, 4096, None, None, 1 << 20, 1 << 30)
        assert e.value.status == 1                                       # HR_EINVAL
        assert "HR_STATIC_SCRATCH_BYTES" in str(e.value) and str(hr.hr_spinor_bytes(g, hr.ODD)) in str(e.value)


@pytest.mark.gpu
@pytest.mark.parametrize("L,prec,kernel", [((8, 8, 8, 16), 0, 1), ((8, 8, 8, 16), 1, 2), ((6, 2, 4, 12), 0, 1),
                                           ((16, 16, 16, 32), 0, 2), ((16, 16, 16, 32), 1, 0)])
def test_static_scratch_dhat_matches_the_existing_path_twice_in_a_row(hr, L, prec, kernel):
    """two calls in a row with DIFFERENT inputs (the array keeps the first call's odd half field: a second call that
    read stale entries would show), without and with clover; (16,16,16,32) in fp64 fills the array to its last byte"""
    import torch
    from paper_2411_18511_b200.lattice import Lattice
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    if kernel == hr.KERNEL_TILED and hr.hr_kernel_name(hr.geom(L, hr.REP_FUND, prec, hr.LINKS_COMPRESSED, kernel)) != "tiled":
        pytest.skip("lattice does not fit the tiled kernel")
    m0, csw = -0.25, 1.2
    lat = Lattice(L, hr.REP_FUND, prec, kernel)
    rnd = (lambda a: inputs.to_f32_rounded(a)) if prec == 1 else (lambda a: a)
    U_dev = lat.put_gauge_fund(rnd(inputs.weak_gauge(L, 0.3, 1)))
    fwd, inv = lat.clover_build(m0, csw, U_dev)
    psis = [lat.put_spinor(rnd(inputs.gaussian_spinor(L, 2, seed))) for seed in (2, 3)]
    calls = [(psis[0], None, None), (psis[1], fwd, inv)]

    want = []
    for psi_dev, cf, ci in calls:                                         # the existing path, caller-owned tmp
        out = torch.zeros_like(psi_dev)
        lat.dhat(m0, U_dev, lat.even(psi_dev), lat.even(out), clover_fwd=cf, clover_inv=ci)
        want.append(out)
    got = [torch.zeros_like(p) for p in psis]                             # outputs are the caller's, made before the calls
    torch.cuda.synchronize()

    lat.dhat_static(m0, U_dev, lat.even(calls[0][0]), lat.even(got[0]))   # first call: also the per-device set-up
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    lat.dhat_static(m0, U_dev, lat.even(calls[1][0]), lat.even(got[1]), clover_fwd=fwd, clover_inv=inv)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before, "the call took device memory"

    for k in range(2):
        g, w = lat.get_spinor(got[k]), lat.get_spinor(want[k])
        assert np.isfinite(g).all()
        assert np.linalg.norm(w.ravel()) > 0
        assert rel(g, w) <= TOL[prec], (k, rel(g, w))
        assert torch.equal(got[k], want[k]), "same kernels on the same inputs: the bits agree as well"
    # and once more, the first input again after the clover call: nothing of the previous call leaks into the result
    again = torch.zeros_like(psis[0])
    lat.dhat_static(m0, U_dev, lat.even(psis[0]), lat.even(again))
    torch.cuda.synchronize()
    assert rel(lat.get_spinor(again), lat.get_spinor(want[0])) <= TOL[prec]
