"""The sharded hop (include/hr_dslash.h "sharded hop"): a global lattice cut into sub-lattices that are held
as separate buffers on ONE device, faces exchanged by device-to-device copies, local operators applied, results stitched
together and compared with the oracle's GLOBAL operator — the oracle knows nothing about the decomposition.  Plus the
host-side plumbing without a GPU: block decomposition round trip and a world-size-2 gloo exchange of face buffers."""
import os
import socket
import subprocess
import sys
import textwrap

import numpy as np
import pytest

from paper_2411_18511_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
TOL = {0: 1e-13, 1: 1e-5}
NTHREADS = max(1, len(os.sched_getaffinity(0)))


def rel(a, b):
    return float(np.linalg.norm((a.astype(np.complex128) - b).ravel()) / np.linalg.norm(b.ravel()))


# ------------------------------------------------------------------ host side, no GPU
def test_block_decomposition_round_trip():
    from paper_2411_18511_b200 import halo
    Lg, P = (8, 4, 4, 12), (2, 1, 2, 3)
    a = np.arange(np.prod(Lg) * 3, dtype=np.float64).reshape(-1, 3)
    blocks = {c: halo.local_block(a, Lg, P, c) for c in halo.rank_coords(P)}
    assert len(blocks) == 12 and all(b.shape == (4 * 4 * 2 * 4, 3) for b in blocks.values())
    assert np.array_equal(halo.assemble(blocks, Lg, P), a)
    # the block of rank (1,0,1,2) starts at global site (4,0,2,8)
    x = ((4 * 4 + 0) * 4 + 2) * 12 + 8
    assert np.array_equal(blocks[(1, 0, 1, 2)][0], a[x])
    assert halo.rank_of((1, 0, 1, 2), P) == (1 * 1 + 0) * 2 * 3 + 1 * 3 + 2
    g = halo.RankGrid(P, (1, 0, 1, 2))
    assert g.split == (True, False, True, True) and g.neighbour(3, +1) == (1, 0, 1, 0) and g.neighbour(0, -1) == (0, 0, 1, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_ranks_exchange_faces_over_gloo():
    """world size 2, process grid (2,1,1,1) with direction 3 cut onto the rank itself: every face buffer ends up where
    hr_hop_local expects it (recv[2mu] = down face of the rank at +mu, recv[2mu+1] = up face of the rank at -mu)"""
    code = textwrap.dedent("""
        import os, sys
        sys.path.insert(0, %r)
        import torch
        import torch.distributed as dist
        from paper_2411_18511_b200 import halo
        from paper_2411_18511_b200.dist import Ranks
        r = Ranks(backend="gloo", device="cpu")
        P = (2, 1, 1, 1)
        grid = halo.RankGrid(P, halo.rank_coords(P)[r.rank], split=(True, False, False, True))
        def face(rank, f): return torch.full((64,), 16 * rank + f, dtype=torch.uint8)
        send = [face(r.rank, f) if grid.split[f // 2] else None for f in range(8)]
        recv = [torch.zeros(64, dtype=torch.uint8) if grid.split[f // 2] else None for f in range(8)]
        halo.exchange_distributed(grid, dist, send, recv)
        other = 1 - r.rank
        assert torch.equal(recv[0], face(other, 0)) and torch.equal(recv[1], face(other, 1))     # x0: the other rank on both sides
        assert torch.equal(recv[6], face(r.rank, 6)) and torch.equal(recv[7], face(r.rank, 7))   # x3: this rank is its own neighbour
        assert recv[2] is None and recv[4] is None
        r.barrier()
        r.close()
        print("rank", r.rank, "ok")
    """ % ROOT)
    port = _free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, WORLD_SIZE="2", RANK=str(rank), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, "-c", code], env=env, stdout=subprocess.PIPE, stderr=subprocess.STDOUT))
    for p in procs:
        out, _ = p.communicate(timeout=180)
        assert p.returncode == 0, out.decode()
        assert b"ok" in out


# ------------------------------------------------------------------ GPU: self-exchange parity against the global oracle
@pytest.fixture(scope="module")
def hr():
    import torch
    assert torch.cuda.is_available(), "the gpu tests need a CUDA device"
    from paper_2411_18511_b200 import build, hr as _hr
    build.build()
    _hr.lib()
    return _hr


def make_shards(hr, Lg, P, rep, prec, split=None, link_storage=None, kernel=None):
    from paper_2411_18511_b200 import halo
    from paper_2411_18511_b200.lattice import Lattice
    L = halo.local_extents(Lg, P)
    ls = hr.LINKS_COMPRESSED if link_storage is None else link_storage
    k = hr.KERNEL_AUTO if kernel is None else kernel
    return {c: halo.Shard(Lattice(L, rep, prec, k, link_storage=ls), P, c, split) for c in halo.rank_coords(P)}


CASES = [((8, 4, 4, 8), (2, 1, 1, 1), None),            # one cut direction, two ranks
         ((4, 4, 8, 8), (1, 1, 2, 2), None),            # two cut directions, 2 x 2 ranks
         ((8, 8, 4, 4), (2, 2, 1, 1), None),
         ((4, 4, 4, 4), (2, 2, 2, 2), None),            # all four cut, local lattice 2^4 (every site on every face)
         ((4, 6, 4, 8), (1, 1, 1, 1), (1, 1, 1, 1)),    # one rank that is its own neighbour in all four directions
         ((12, 4, 4, 4), (3, 1, 1, 1), None)]           # three ranks in a ring


@pytest.mark.gpu
@pytest.mark.parametrize("Lg,P,split", CASES)
@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("kernel", ["generic", "tiled"])
def test_sharded_fundamental_operators(hr, orc, Lg, P, split, prec, kernel):
    """bare hops, full D, Dhat and the clover-improved Dhat on a cut lattice against the oracle on the whole lattice, with
    both interior kernels (generic, and the x0-marching tiled kernel in its open-boundary instantiation)"""
    import torch
    from paper_2411_18511_b200 import halo
    from test_gpu_parity import dense_to_blocks
    m0, csw = -0.25, 1.2
    U = inputs.weak_gauge(Lg, 0.3, 1)
    psi = inputs.gaussian_spinor(Lg, 2, 2)
    if prec == 1:
        U, psi = inputs.to_f32_rounded(U), inputs.to_f32_rounded(psi)
    A = orc.clover_dense(Lg, 4.0 + m0, csw, U)
    Ainv = orc.invert(A)
    bf, bi = dense_to_blocks(A), dense_to_blocks(Ainv)
    kid = hr.KERNEL_GENERIC if kernel == "generic" else hr.KERNEL_TILED
    shards = make_shards(hr, Lg, P, hr.REP_FUND, prec, split, kernel=kid)
    assert all(hr.hr_kernel_name(sh.lat.g) == kernel for sh in shards.values())
    Ud, pd, od, td, cf, ci = {}, {}, {}, {}, {}, {}
    for c, sh in shards.items():
        lat = sh.lat
        Ud[c] = lat.put_gauge_fund(halo.local_block(U, Lg, P, c))
        pd[c] = lat.put_spinor(halo.local_block(psi, Lg, P, c))
        od[c] = torch.zeros_like(pd[c])
        td[c] = lat.empty_spinor(hr.ODD)
        cf[c] = lat.put_clover(halo.local_block(bf, Lg, P, c))
        ci[c] = lat.put_clover(halo.local_block(bi, Lg, P, c))
    ev = {c: sh.lat.even for c, sh in shards.items()}
    odd = {c: sh.lat.odd for c, sh in shards.items()}

    def gather():
        torch.cuda.synchronize()
        return halo.assemble({c: sh.lat.get_spinor(od[c]) for c, sh in shards.items()}, Lg, P)

    # bare hops into the two halves of one output field
    halo.hop_all(shards, halo.exchange_in_process, hr.ODD, Ud, {c: ev[c](pd[c]) for c in shards}, {c: odd[c](od[c]) for c in shards})
    halo.hop_all(shards, halo.exchange_in_process, hr.EVEN, Ud, {c: odd[c](pd[c]) for c in shards}, {c: ev[c](od[c]) for c in shards})
    want = orc.hop(Lg, 0, 0, U, psi, nthreads=NTHREADS)
    want = orc.hop(Lg, 0, 1, U, psi, nthreads=NTHREADS, out=want)
    assert rel(gather(), want) <= TOL[prec]
    # full D
    halo.dirac_all(shards, halo.exchange_in_process, m0, Ud, pd, od)
    assert rel(gather(), orc.dirac(Lg, 0, m0, U, psi, nthreads=NTHREADS)) <= TOL[prec]
    # Dhat without and with clover
    for c in shards:
        od[c].zero_()
    halo.dhat_all(shards, halo.exchange_in_process, m0, Ud, {c: ev[c](pd[c]) for c in shards}, {c: ev[c](od[c]) for c in shards}, td)
    assert rel(gather(), orc.dirac_eo(Lg, 0, m0, U, psi, nthreads=NTHREADS)) <= TOL[prec]
    want_e2 = orc.dirac_eo_clover(Lg, U, A, Ainv, psi, nthreads=NTHREADS)
    for overlap in (False, True):      # True: pack + transfer on a side stream while the interior kernels run
        for c in shards:
            od[c].zero_()
        halo.dhat_all(shards, halo.exchange_in_process, m0, Ud, {c: ev[c](pd[c]) for c in shards}, {c: ev[c](od[c]) for c in shards}, td,
                      clover_fwd=cf, clover_inv=ci, overlap=overlap)
        assert rel(gather(), want_e2) <= TOL[prec], overlap


@pytest.mark.gpu
@pytest.mark.parametrize("Lg,P,split", [CASES[1], CASES[3], CASES[4]])
@pytest.mark.parametrize("onfly", [False, True])
def test_sharded_adjoint_operators(hr, orc, Lg, P, split, onfly):
    """adjoint fermions on a cut lattice: stored 3x3 links, and links rebuilt on the fly from the fundamental field (the
    up faces are multiplied by the sender's rebuilt link)"""
    import torch
    from paper_2411_18511_b200 import halo
    m0 = -0.3
    Uf = inputs.haar_gauge(Lg, 1)
    R, _ = orc.represent(Uf)
    psi = inputs.gaussian_spinor(Lg, 3, 2)
    shards = make_shards(hr, Lg, P, hr.REP_ADJ, 0, split, hr.LINKS_ONTHEFLY if onfly else hr.LINKS_COMPRESSED)
    Ud, pd, od, td = {}, {}, {}, {}
    for c, sh in shards.items():
        lat = sh.lat
        Ud[c] = lat.put_gauge_fund(halo.local_block(Uf, Lg, P, c)) if onfly else lat.put_gauge_adj(halo.local_block(R, Lg, P, c))
        pd[c] = lat.put_spinor(halo.local_block(psi, Lg, P, c))
        od[c] = torch.zeros_like(pd[c])
        td[c] = lat.empty_spinor(hr.ODD)

    def gather():
        torch.cuda.synchronize()
        return halo.assemble({c: sh.lat.get_spinor(od[c]) for c, sh in shards.items()}, Lg, P)

    halo.dirac_all(shards, halo.exchange_in_process, m0, Ud, pd, od)
    assert rel(gather(), orc.dirac(Lg, 1, m0, R, psi, nthreads=NTHREADS)) <= 1e-13
    for c in shards:
        od[c].zero_()
    halo.dhat_all(shards, halo.exchange_in_process, m0, Ud, {c: sh.lat.even(pd[c]) for c, sh in shards.items()},
                  {c: sh.lat.even(od[c]) for c, sh in shards.items()}, td)
    assert rel(gather(), orc.dirac_eo(Lg, 1, m0, R, psi, nthreads=NTHREADS)) <= 1e-13


@pytest.mark.gpu
@pytest.mark.parametrize("Lg,P,split", [CASES[1], CASES[3], CASES[4]])
@pytest.mark.parametrize("prec", [0, 1])
@pytest.mark.parametrize("two_rows", [False, True])
def test_sharded_su3_operators(hr, orc, Lg, P, split, prec, two_rows):
    """complex 3 x 3 links (HR_REP_SU3) on a cut lattice: the up faces are multiplied by the sender's U^dag, the receiver applies its own
    U to the down faces; full D and Dhat stitched from the shards against the oracle's global operator (rep 2)"""
    import torch
    from paper_2411_18511_b200 import halo
    m0 = -0.3
    U = inputs.haar_gauge_su3(Lg, 1)
    psi = inputs.gaussian_spinor(Lg, 3, 2)
    if prec:
        U, psi = U.astype(np.complex64).astype(np.complex128), psi.astype(np.complex64).astype(np.complex128)
    shards = make_shards(hr, Lg, P, hr.REP_SU3, prec, split, hr.LINKS_COMPRESSED if two_rows else hr.LINKS_FULL)
    Ud, pd, od, td = {}, {}, {}, {}
    for c, sh in shards.items():
        lat = sh.lat
        Ud[c] = lat.put_gauge_su3(halo.local_block(U, Lg, P, c))
        pd[c] = lat.put_spinor(halo.local_block(psi, Lg, P, c))
        od[c] = torch.zeros_like(pd[c])
        td[c] = lat.empty_spinor(hr.ODD)

    def gather():
        torch.cuda.synchronize()
        return halo.assemble({c: sh.lat.get_spinor(od[c]) for c, sh in shards.items()}, Lg, P)

    halo.dirac_all(shards, halo.exchange_in_process, m0, Ud, pd, od)
    assert rel(gather(), orc.dirac(Lg, 2, m0, U, psi, nthreads=NTHREADS)) <= TOL[prec]
    for c in shards:
        od[c].zero_()
    halo.dhat_all(shards, halo.exchange_in_process, m0, Ud, {c: sh.lat.even(pd[c]) for c, sh in shards.items()},
                  {c: sh.lat.even(od[c]) for c, sh in shards.items()}, td)
    assert rel(gather(), orc.dirac_eo(Lg, 2, m0, U, psi, nthreads=NTHREADS)) <= TOL[prec]
    # Dhat with clover (E2) through the clover epilogues of the interior and boundary kernels
    m0c, csw = -0.25, 1.2
    A = orc.clover_dense_su3(Lg, 4.0 + m0c, csw, U)
    Ainv = np.linalg.inv(A)
    from test_gpu_parity import dense_to_blocks
    bf, bi = dense_to_blocks(A), dense_to_blocks(Ainv)
    fw, iv = {}, {}
    for c, sh in shards.items():
        fw[c] = sh.lat.put_clover(halo.local_block(bf, Lg, P, c))
        iv[c] = sh.lat.put_clover(halo.local_block(bi, Lg, P, c))
        od[c].zero_()
    halo.dhat_all(shards, halo.exchange_in_process, m0c, Ud, {c: sh.lat.even(pd[c]) for c, sh in shards.items()},
                  {c: sh.lat.even(od[c]) for c, sh in shards.items()}, td, clover_fwd=fw, clover_inv=iv)
    assert rel(gather(), orc.dirac_eo_clover_n(Lg, 2, U, A, Ainv, psi, nthreads=NTHREADS)) <= TOL[prec]


@pytest.mark.gpu
def test_uncut_hop_local_is_the_single_gpu_hop(hr):
    """with no cut direction hr_hop_local is hr_dirac_eo_apply bit for bit (same kernel, no boundary pass)"""
    import torch
    from paper_2411_18511_b200.lattice import Lattice
    L = (4, 4, 6, 8)
    lat = Lattice(L, hr.REP_FUND, hr.PREC_F64, hr.KERNEL_GENERIC)
    U = lat.put_gauge_fund(inputs.haar_gauge(L, 1))
    psi = lat.put_spinor(inputs.gaussian_spinor(L, 2, 2))
    a, b = torch.zeros_like(psi), torch.zeros_like(psi)
    lat.hop(hr.EO_HOP_OE, U, lat.even(psi), lat.odd(a))
    hr.hr_hop_local(lat.g, hr.decomp((0, 0, 0, 0)), hr.ODD, hr.EPI_NONE, 0.0, 1.0, U, None, lat.even(psi), None, lat.odd(b), [None] * 8, hr.stream_ptr())
    torch.cuda.synchronize()
    assert torch.equal(a, b)
    with pytest.raises(hr.HrError):      # a cut direction without its faces
        hr.hr_hop_local(lat.g, hr.decomp((1, 0, 0, 0)), hr.ODD, hr.EPI_NONE, 0.0, 1.0, U, None, lat.even(psi), None, lat.odd(b), [None] * 8, hr.stream_ptr())
