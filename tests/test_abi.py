"""CPU-only checks of the C-ABI boundary: libhr_dslash.so builds, loads and exports every symbol
include/hr_dslash.h declares; the host-only entry points (sizes, work model, argument checks) behave
as the header says.  No kernel is launched here."""
import ctypes
import os
import re

import pytest

from paper_2411_18511_b200 import build, hr

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    build.build()
    return hr.lib()


def header_symbols():
    src = open(os.path.join(ROOT, "include", "hr_dslash.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hr_[a-z0-9_]+)\s*\(", src)))


def test_header_and_binding_agree():
    assert header_symbols() == sorted(hr.SYMBOLS)


def test_every_symbol_is_exported(L):
    for name in header_symbols():
        assert getattr(L, name) is not None, name


def test_geom_struct_matches_header():
    assert ctypes.sizeof(hr.hr_geom) == 8 * 4
    src = open(os.path.join(ROOT, "include", "hr_dslash.h")).read()
    body = re.search(r"typedef struct hr_geom \{(.*?)\} hr_geom;", src, re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = re.findall(r"int\s+(\w+)", body)
    assert names == ["L", "rep", "prec", "link_storage", "kernel"]
    assert [f[0] for f in hr.hr_geom._fields_] == names


def test_sizes(L):
    g = hr.geom((48, 48, 48, 48), hr.REP_FUND, hr.PREC_F64)
    V = 48 ** 4
    assert hr.hr_spinor_bytes(g, hr.BOTH) == V * 128
    assert hr.hr_spinor_bytes(g, hr.EVEN) == V * 64 == hr.hr_spinor_bytes(g, hr.ODD)
    assert hr.hr_gauge_bytes(g, hr.REP_FUND) == 4 * V * 32        # compressed first row: 648 MiB
    assert hr.hr_gauge_bytes(g, hr.REP_ADJ) == 4 * V * 72
    assert hr.hr_clover_bytes(g) == V * 256
    assert hr.hr_canonical_spinor_bytes(g) == V * 128
    assert hr.hr_canonical_gauge_bytes(g, hr.REP_FUND) == 4 * V * 64
    assert hr.hr_canonical_clover_bytes(g) == V * 256
    g32 = hr.geom((4, 6, 8, 2), hr.REP_ADJ, hr.PREC_F32)
    V = 4 * 6 * 8 * 2
    assert hr.hr_spinor_bytes(g32, hr.BOTH) == V * 96
    assert hr.hr_gauge_bytes(g32, hr.REP_ADJ) == 4 * V * 36
    assert hr.hr_gauge_bytes(g32, hr.REP_FUND) == 4 * V * 16
    assert hr.hr_host_workspace_bytes(g32) > 0


@pytest.mark.parametrize("bad", [(3, 4, 4, 4), (4, 4, 4, 0), (4, 4, 5, 4), (4, 4, 4, -2), (2048, 2048, 2048, 2048)])
def test_invalid_geometry_is_rejected(L, bad):
    g = hr.geom(bad)
    assert hr.hr_spinor_bytes(g, hr.BOTH) == 0
    with pytest.raises(hr.HrError) as e:
        hr.hr_dirac_flops_bytes(g, hr.OP_HOP)
    assert e.value.status == hr.EINVAL
    with pytest.raises(hr.HrError) as e:
        hr.hr_dirac_apply(g, 0.0, 16, 32, 48)
    assert e.value.status == hr.EINVAL


def test_argument_checks_happen_before_any_cuda_call(L):
    g = hr.geom((4, 4, 4, 4))
    with pytest.raises(hr.HrError) as e:
        hr.hr_dirac_apply(g, 0.0, None, 4096, 8192)
    assert e.value.status == hr.EINVAL and "NULL" in str(e.value)
    with pytest.raises(hr.HrError) as e:
        hr.hr_dirac_apply(g, 0.0, 4096, 4096 * 1024 + 8, 8192 * 1024)
    assert e.value.status == hr.EALIGN
    with pytest.raises(hr.HrError) as e:   # out aliases psi: a gather cannot run in place
        hr.hr_dirac_apply(g, 0.0, 4096, 1 << 20, (1 << 20) + 1024)
    assert e.value.status == hr.EINVAL and "alias" in str(e.value)
    with pytest.raises(hr.HrError) as e:
        hr.hr_dirac_eo_apply(g, 7, 0.0, 4096, None, None, 1 << 20, 1 << 21, 1 << 22)
    assert e.value.status == hr.EINVAL
    with pytest.raises(hr.HrError) as e:   # 4+m0 = 0: D_oo singular
        hr.hr_dirac_eo_apply(g, hr.EO_DHAT, -4.0, 4096, None, None, 1 << 20, 1 << 21, 1 << 22)
    assert e.value.status == hr.EINVAL
    with pytest.raises(hr.HrError) as e:   # one clover field without the other
        hr.hr_dirac_eo_apply(g, hr.EO_DHAT, 0.0, 4096, 1 << 23, None, 1 << 20, 1 << 21, 1 << 22)
    assert e.value.status == hr.EINVAL
    gfull = hr.geom((4, 4, 4, 4), link_storage=hr.LINKS_FULL)
    with pytest.raises(hr.HrError) as e:
        hr.hr_dirac_apply(gfull, 0.0, 4096, 1 << 20, 1 << 21)
    assert e.value.status == hr.EUNSUPPORTED
    gadj = hr.geom((4, 4, 4, 4), rep=hr.REP_ADJ)
    with pytest.raises(hr.HrError) as e:   # adjoint clover exists (6x6 blocks); a bad parity is still caught first
        hr.hr_clover_apply(gadj, 7, 4096, 1 << 20, 1 << 21)
    assert e.value.status == hr.EINVAL
    assert hr.hr_clover_bytes(gadj) == 256 * 72 * 8 and hr.hr_canonical_clover_bytes(gadj) == 256 * 72 * 8
    with pytest.raises(hr.HrError) as e:   # hr_cg_solve: tol must be positive; checked before any CUDA call
        hr.hr_cg_solve(g, 0.0, 4096, None, None, 1 << 20, 1 << 21, 1 << 24, 0.0, 10)
    assert e.value.status == hr.EINVAL
    with pytest.raises(hr.HrError) as e:   # x aliases b
        hr.hr_cg_solve(g, 0.0, 4096, None, None, 1 << 20, 1 << 20, 1 << 24, 1e-8, 10)
    assert e.value.status == hr.EINVAL
    assert hr.hr_cg_workspace_bytes(g) >= 5 * hr.hr_spinor_bytes(g, hr.EVEN)
    with pytest.raises(hr.HrError) as e:   # hr_cg_solve_mixed: the geometry must describe the fp64 fields
        hr.hr_cg_solve_mixed(hr.geom((4, 4, 4, 4), prec=hr.PREC_F32), 0.0, 4096, 8192, 1 << 20, 1 << 21, 1 << 24, 1e-10)
    assert e.value.status == hr.EINVAL
    with pytest.raises(hr.HrError) as e:   # inner_tol must be below 1
        hr.hr_cg_solve_mixed(g, 0.0, 4096, 8192, 1 << 20, 1 << 21, 1 << 24, 1e-10, inner_tol=1.5)
    assert e.value.status == hr.EINVAL
    assert hr.hr_cg_mixed_workspace_bytes(g) > hr.hr_cg_workspace_bytes(hr.geom((4, 4, 4, 4), prec=hr.PREC_F32))
    assert hr.hr_cg_mixed_workspace_bytes(hr.geom((4, 4, 4, 4), prec=hr.PREC_F32)) == 0
    gt = hr.geom((4, 4, 4, 200), kernel=hr.KERNEL_TILED)   # rows of 100 sites per parity: no tile shape fits
    with pytest.raises(hr.HrError) as e:
        hr.hr_dirac_apply(gt, 0.0, 4096, 1 << 30, 1 << 31)
    assert e.value.status == hr.EUNSUPPORTED


def test_work_model_matches_survey_table(L):
    """SURVEY.md §8(d) table, typed here: F_hop = 8N(16N+7) fund / 8N(8N+7) adj; bytes in S, G, Bk."""
    f64 = hr.geom((48,) * 4, hr.REP_FUND, hr.PREC_F64, hr.LINKS_COMPRESSED)
    f64full = hr.geom((48,) * 4, hr.REP_FUND, hr.PREC_F64, hr.LINKS_FULL)
    f32 = hr.geom((48,) * 4, hr.REP_FUND, hr.PREC_F32, hr.LINKS_COMPRESSED)
    f32full = hr.geom((48,) * 4, hr.REP_FUND, hr.PREC_F32, hr.LINKS_FULL)
    adj = hr.geom((24,) * 4, hr.REP_ADJ, hr.PREC_F64)
    assert hr.hr_dirac_flops_bytes(f64, hr.OP_HOP) == (624.0, 512.0, 9 * 128 + 8 * 32)
    assert hr.hr_dirac_flops_bytes(f64full, hr.OP_HOP) == (624.0, 768.0, 1664.0)
    assert hr.hr_dirac_flops_bytes(f32, hr.OP_HOP)[:2] == (624.0, 256.0)
    assert hr.hr_dirac_flops_bytes(f32full, hr.OP_HOP) == (624.0, 384.0, 832.0)
    assert hr.hr_dirac_flops_bytes(adj, hr.OP_HOP) == (744.0, 960.0, 2304.0)
    adjfly = hr.geom((24,) * 4, hr.REP_ADJ, hr.PREC_F64, hr.LINKS_ONTHEFLY)
    assert hr.hr_dirac_flops_bytes(adjfly, hr.OP_HOP) == (744.0, 640.0, 9 * 192 + 8 * 32)   # 960 -> 640
    assert hr.hr_dirac_flops_bytes(adjfly, hr.OP_DIRAC)[:2] == (816.0, 2 * 192 + 4 * 32)
    assert hr.hr_spinor_bytes(hr.geom((4, 4, 4, 4), hr.REP_FUND, hr.PREC_F64, hr.LINKS_ONTHEFLY)) == 0   # adjoint only
    assert hr.hr_dirac_flops_bytes(f64, hr.OP_DIRAC)[:2] == (672.0, 384.0)
    assert hr.hr_dirac_flops_bytes(f64full, hr.OP_DIRAC)[:2] == (672.0, 512.0)
    assert hr.hr_dirac_flops_bytes(adj, hr.OP_DIRAC)[:2] == (816.0, 672.0)
    assert hr.hr_dirac_flops_bytes(f64, hr.OP_DHAT)[:2] == (1296.0, 1152.0)
    assert hr.hr_dirac_flops_bytes(f64full, hr.OP_DHAT)[:2] == (1296.0, 1664.0)
    assert hr.hr_dirac_flops_bytes(adj, hr.OP_DHAT)[:2] == (1560.0, 2112.0)
    assert hr.hr_dirac_flops_bytes(f64, hr.OP_CLOVER) == (208.0, 512.0, 512.0)
    assert hr.hr_dirac_flops_bytes(f32, hr.OP_CLOVER)[:2] == (208.0, 256.0)
    assert hr.hr_dirac_flops_bytes(f64, hr.OP_DHAT_CLOVER)[:2] == (1696.0, 1664.0)
    assert hr.hr_dirac_flops_bytes(f64full, hr.OP_DHAT_CLOVER)[:2] == (1696.0, 2176.0)
    assert hr.hr_dirac_flops_bytes(f64, hr.OP_REPRESENT)[1] == 416.0
    assert hr.hr_dirac_flops_bytes(f64full, hr.OP_REPRESENT)[1] == 544.0
    # adjoint clover: two hermitian 6x6 blocks per site = 72 reals; mat-vecs 2 (12 + 8*6*5) = 504 flops
    assert hr.hr_dirac_flops_bytes(adj, hr.OP_CLOVER) == (504.0, 2 * 192 + 576.0, 2 * 192 + 576.0)
    assert hr.hr_dirac_flops_bytes(adj, hr.OP_DHAT_CLOVER)[:2] == (2 * 744 + 2 * 504 + 2 * 24.0, 5 * 192 + 16 * 72 + 2 * 576.0)


def test_kernel_name_and_launch_counter(L):
    assert hr.hr_kernel_name(hr.geom((4, 4, 4, 4))) == "generic"
    assert hr.hr_kernel_name(hr.geom((4, 4, 4, 3))) == "invalid"
    assert hr.hr_launch_count() >= 0


def test_missing_library_fails_loudly(monkeypatch):
    monkeypatch.setattr(hr, "_lib", None)
    monkeypatch.setattr(hr, "LIB_PATH", "/nonexistent/libhr_dslash.so")
    with pytest.raises(ImportError):
        hr.lib()


def test_lattice_stages_on_its_own_device(monkeypatch):
    """every buffer a Lattice makes (canonical staging included) is requested on the Lattice's device, not on cuda:0:
    under `bench.py --gpus N` rank k packs on cuda:k and must not read a cuda:0 pointer (no GPU needed: the
    allocation and pack calls are recorded, not executed)"""
    import numpy as np
    from paper_2411_18511_b200 import hr as _hr, lattice
    seen = []
    monkeypatch.setattr(_hr, "upload", lambda a, device=None: seen.append(("upload", device)) or "canon")
    monkeypatch.setattr(_hr, "device_buffer", lambda n, device=None: seen.append(("buffer", device)) or "dev")
    monkeypatch.setattr(_hr, "stream_ptr", lambda stream=None: 0)
    for name in ("hr_pack_spinor", "hr_pack_gauge", "hr_pack_clover"):
        monkeypatch.setattr(_hr, name, lambda *a, **k: None)
    lat = lattice.Lattice((4, 4, 4, 4), _hr.REP_ADJ, _hr.PREC_F64, device="cuda:3")
    lat.put_spinor(np.zeros((256, 4, 3), dtype=np.complex128))
    lat.put_gauge_fund(np.zeros((256, 4, 2, 2), dtype=np.complex128))
    lat.put_gauge_adj(np.zeros((256, 4, 3, 3)))
    lat.put_clover(np.zeros((256, 2, 36)))
    assert len(seen) == 8 and all(dev == "cuda:3" for _, dev in seen), seen


def test_su3_geometry_and_sizes(L):
    """HR_REP_SU3: complex 3 x 3 links stored in full (18 reals per link) or as their first two rows (12 reals, HR_LINKS_COMPRESSED),
    3 complex colours; HR_LINKS_ONTHEFLY is rejected"""
    g = hr.geom((4, 4, 4, 8), hr.REP_SU3, hr.PREC_F64, hr.LINKS_FULL)
    V = 4 * 4 * 4 * 8
    assert hr.hr_spinor_bytes(g, hr.BOTH) == V * 24 * 8
    assert hr.hr_gauge_bytes(g, hr.REP_SU3) == hr.hr_canonical_gauge_bytes(g, hr.REP_SU3) == 4 * V * 18 * 8
    assert hr.hr_dirac_flops_bytes(g, hr.OP_DHAT) == (2 * 1320.0 + 72.0, 5 * 192.0 + 16 * 144.0, 19 * 192.0 + 16 * 144.0)
    g2 = hr.geom((4, 4, 4, 8), hr.REP_SU3, hr.PREC_F64, hr.LINKS_COMPRESSED)
    assert hr.hr_gauge_bytes(g2, hr.REP_SU3) == 4 * V * 12 * 8 and hr.hr_canonical_gauge_bytes(g2, hr.REP_SU3) == 4 * V * 18 * 8
    assert hr.hr_dirac_flops_bytes(g2, hr.OP_HOP)[1] == 2 * 192.0 + 8 * 96.0
    bad = hr.geom((4, 4, 4, 8), hr.REP_SU3, hr.PREC_F64, hr.LINKS_ONTHEFLY)
    assert hr.hr_spinor_bytes(bad, hr.BOTH) == 0
    assert hr.hr_dirac_flops_bytes(g, hr.OP_CLOVER)[1] == 2 * 192.0 + 2 * 36 * 8.0        # two hermitian 6 x 6 blocks per site
    with pytest.raises(hr.HrError):
        hr.hr_dirac_flops_bytes(g, hr.OP_REPRESENT)


def test_kernel_plan_of_the_bench_lattice(L):
    """hr_kernel_plan is host-only: the 48^4 launch plans DESIGN.md §5 describes (148 SMs assumed without a device)"""
    g64 = hr.geom((48,) * 4, hr.REP_FUND, hr.PREC_F64)
    g32 = hr.geom((48,) * 4, hr.REP_FUND, hr.PREC_F32)
    assert hr.hr_kernel_plan(g64, hr.OP_HOP) == {"kernel": 1, "t1": 2, "t2": 4, "nseg": 1, "seglen": 48, "threads": 224, "smem": 221312, "grid": 288}
    assert hr.hr_kernel_plan(g64, hr.OP_DIRAC) == {"kernel": 2, "t1": 2, "t2": 2, "nseg": 1, "seglen": 48, "threads": 224, "smem": 215168, "grid": 576}
    assert hr.hr_kernel_plan(g32, hr.OP_HOP)["grid"] == 144 and hr.hr_kernel_plan(g32, hr.OP_HOP)["t1"] == 4
    assert hr.hr_kernel_plan(g32, hr.OP_DIRAC) == {"kernel": 2, "t1": 2, "t2": 4, "nseg": 1, "seglen": 48, "threads": 416, "smem": 215168, "grid": 288}
    # the fp32 full-lattice kernel addresses its links by 32-bit offsets in 16-byte chunks: a gauge field of 2^32 chunks or more
    # (8 * L0*L1*L2 * L3/2 >= 2^32) falls back to the register-link form (no link slots: less shared memory); fp64 carries pointers
    assert hr.hr_kernel_plan(hr.geom((256, 256, 256, 48), hr.REP_FUND, hr.PREC_F32), hr.OP_DIRAC)["smem"] == 215168
    assert hr.hr_kernel_plan(hr.geom((512, 256, 256, 48), hr.REP_FUND, hr.PREC_F32), hr.OP_DIRAC)["smem"] == 172160
    assert hr.hr_kernel_plan(hr.geom((512, 256, 256, 48), hr.REP_FUND, hr.PREC_F64), hr.OP_DIRAC)["smem"] == 215168
    # below 32^4 and for adjoint / SU(3) fermions AUTO keeps the generic kernel
    assert hr.hr_kernel_plan(hr.geom((16,) * 4), hr.OP_HOP)["kernel"] == 0
    assert hr.hr_kernel_plan(hr.geom((48,) * 4, hr.REP_ADJ), hr.OP_HOP)["kernel"] == 0
    assert hr.hr_kernel_plan(hr.geom((48,) * 4, hr.REP_SU3, hr.PREC_F64, hr.LINKS_FULL), hr.OP_DIRAC)["kernel"] == 0
    with pytest.raises(hr.HrError):
        hr.hr_kernel_plan(g64, hr.OP_CLOVER)
