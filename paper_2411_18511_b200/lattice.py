"""Convenience wrapper used by the tests, bench.py and smoke(): owns torch-allocated device buffers
for one geometry and moves canonical numpy arrays in and out through hr_pack_* / hr_unpack_*.

Marshalling only — every operator call goes straight to the C-ABI (hr.py); nothing is computed here.
"""
from __future__ import annotations

import numpy as np

from . import hr


class Lattice:
    def __init__(self, L, rep=hr.REP_FUND, prec=hr.PREC_F64, kernel=hr.KERNEL_AUTO, device=None,
                 link_storage=None):
        self.L = tuple(int(v) for v in L)
        self.V = int(np.prod(self.L))
        self.N = 2 if rep == hr.REP_FUND else 3
        if link_storage is None:      # SU(2): first-row compressed fundamental links; SU(3): complex 3 x 3 links in full
            link_storage = hr.LINKS_FULL if rep == hr.REP_SU3 else hr.LINKS_COMPRESSED
        self.g = hr.geom(self.L, rep, prec, link_storage, kernel)
        self.device = hr.current_device() if device is None else device     # every buffer of this object lives here
        self.real = hr.np_real(self.g)
        self.cplx = hr.np_complex(self.g)
        self.half = hr.hr_spinor_bytes(self.g, hr.EVEN)

    # ---- buffers
    def empty_spinor(self, parity=hr.BOTH):
        return hr.device_buffer(hr.hr_spinor_bytes(self.g, parity), self.device)

    def empty_gauge(self, rep=None):
        return hr.device_buffer(hr.hr_gauge_bytes(self.g, self.g.rep if rep is None else rep), self.device)

    def empty_clover(self):
        return hr.device_buffer(hr.hr_clover_bytes(self.g), self.device)

    def even(self, full):
        return full[: self.half]

    def odd(self, full):
        return full[self.half:]

    # ---- canonical numpy <-> device layout
    def put_spinor(self, psi):
        """complex [V,4,N] -> packed full-lattice device field"""
        assert psi.shape == (self.V, 4, self.N), psi.shape
        canon = hr.upload(psi.astype(self.cplx), self.device)
        dev = self.empty_spinor()
        hr.hr_pack_spinor(self.g, canon, dev, hr.stream_ptr())
        return dev

    def get_spinor(self, dev):
        canon = hr.device_buffer(hr.hr_canonical_spinor_bytes(self.g), self.device)
        hr.hr_unpack_spinor(self.g, dev, canon, hr.stream_ptr())
        return hr.download(canon, self.cplx, (self.V, 4, self.N))

    def put_gauge_fund(self, U):
        """complex [V,4,2,2] -> packed (compressed) fundamental gauge field"""
        assert U.shape == (self.V, 4, 2, 2), U.shape
        canon = hr.upload(U.astype(self.cplx), self.device)
        dev = self.empty_gauge(hr.REP_FUND)
        hr.hr_pack_gauge(self.g, hr.REP_FUND, canon, dev, hr.stream_ptr())
        return dev

    def get_gauge_fund(self, dev):
        canon = hr.device_buffer(hr.hr_canonical_gauge_bytes(self.g, hr.REP_FUND), self.device)
        hr.hr_unpack_gauge(self.g, hr.REP_FUND, dev, canon, hr.stream_ptr())
        return hr.download(canon, self.cplx, (self.V, 4, 2, 2))

    def put_gauge_adj(self, R):
        assert R.shape == (self.V, 4, 3, 3), R.shape
        canon = hr.upload(R.astype(self.real), self.device)
        dev = self.empty_gauge(hr.REP_ADJ)
        hr.hr_pack_gauge(self.g, hr.REP_ADJ, canon, dev, hr.stream_ptr())
        return dev

    def put_gauge_su3(self, U):
        """complex [V,4,3,3] -> device layout of HR_REP_SU3 links (all three rows, or the first two with LINKS_COMPRESSED)"""
        assert U.shape == (self.V, 4, 3, 3), U.shape
        canon = hr.upload(U.astype(self.cplx), self.device)
        dev = self.empty_gauge(hr.REP_SU3)
        hr.hr_pack_gauge(self.g, hr.REP_SU3, canon, dev, hr.stream_ptr())
        return dev

    def get_gauge_su3(self, dev):
        canon = hr.device_buffer(hr.hr_canonical_gauge_bytes(self.g, hr.REP_SU3), self.device)
        hr.hr_unpack_gauge(self.g, hr.REP_SU3, dev, canon, hr.stream_ptr())
        return hr.download(canon, self.cplx, (self.V, 4, 3, 3))

    def get_gauge_adj(self, dev):
        canon = hr.device_buffer(hr.hr_canonical_gauge_bytes(self.g, hr.REP_ADJ), self.device)
        hr.hr_unpack_gauge(self.g, hr.REP_ADJ, dev, canon, hr.stream_ptr())
        return hr.download(canon, self.real, (self.V, 4, 3, 3))

    def put_clover(self, blocks):
        """real [V,2,(2N)^2] -> packed block field (16 reals per block for the fundamental, 36 for the adjoint rep)"""
        assert blocks.shape == (self.V, 2, 4 * self.N * self.N), blocks.shape
        canon = hr.upload(blocks.astype(self.real), self.device)
        dev = self.empty_clover()
        hr.hr_pack_clover(self.g, canon, dev, hr.stream_ptr())
        return dev

    def get_clover(self, dev):
        canon = hr.device_buffer(hr.hr_canonical_clover_bytes(self.g), self.device)
        hr.hr_unpack_clover(self.g, dev, canon, hr.stream_ptr())
        return hr.download(canon, self.real, (self.V, 2, 4 * self.N * self.N))

    # ---- operators (direct C-ABI calls on torch's current stream)
    def represent(self, u_fund):
        u_adj = self.empty_gauge(hr.REP_ADJ)
        hr.hr_represent_gauge(self.g, u_fund, u_adj, hr.stream_ptr())
        return u_adj

    def represent_antisym(self, u_fund):
        """two-index antisymmetric representation of HR_REP_SU3 links (same layout and size as the input field)"""
        u_rep = self.empty_gauge(hr.REP_SU3)
        hr.hr_represent_gauge_antisym(self.g, u_fund, u_rep, hr.stream_ptr())
        return u_rep

    def dirac(self, m0, u, psi, out=None):
        out = self.empty_spinor() if out is None else out
        hr.hr_dirac_apply(self.g, m0, u, psi, out, hr.stream_ptr())
        return out

    def dirac_clover(self, u, clover_fwd, psi, out=None):
        out = self.empty_spinor() if out is None else out
        hr.hr_dirac_clover_apply(self.g, u, clover_fwd, psi, out, hr.stream_ptr())
        return out

    def hop(self, op, u, inp, out=None):
        """op EO_HOP_OE: inp even half -> odd half;  EO_HOP_EO: odd half -> even half"""
        out = self.empty_spinor(hr.EVEN) if out is None else out
        hr.hr_dirac_eo_apply(self.g, op, 0.0, u, None, None, inp, out, None, hr.stream_ptr())
        return out

    def dhat(self, m0, u, inp, out=None, tmp=None, clover_fwd=None, clover_inv=None):
        out = self.empty_spinor(hr.EVEN) if out is None else out
        tmp = self.empty_spinor(hr.ODD) if tmp is None else tmp
        hr.hr_dirac_eo_apply(self.g, hr.EO_DHAT, m0, u, clover_fwd, clover_inv, inp, out, tmp, hr.stream_ptr())
        return out

    def dhat_static(self, m0, u, inp, out, clover_fwd=None, clover_inv=None):
        """dhat() with the intermediate odd half field in the library's static scratch array: allocates nothing
        (out is the caller's), lattices up to hr.STATIC_SCRATCH_BYTES per odd half field"""
        hr.hr_dhat_apply_static(self.g, m0, u, clover_fwd, clover_inv, inp, out, hr.stream_ptr())
        return out

    def clover_build(self, m0, csw, u_fund, exponential=False):
        fwd, inv = self.empty_clover(), self.empty_clover()
        build = hr.hr_clover_build_exp if exponential else hr.hr_clover_build
        build(self.g, m0, csw, u_fund, fwd, inv, hr.stream_ptr())
        return fwd, inv

    def clover_apply(self, parity, blocks, inp, out=None):
        out = self.empty_spinor(parity) if out is None else out
        hr.hr_clover_apply(self.g, parity, blocks, inp, out, hr.stream_ptr())
        return out

    def cg(self, m0, u, b, tol, max_iter, clover_fwd=None, clover_inv=None, check_every=5):
        """b: even half field -> (x even half field, iterations, |r|/|b|)"""
        x = self.empty_spinor(hr.EVEN)
        ws = hr.device_buffer(hr.hr_cg_workspace_bytes(self.g), self.device)
        it, rel = hr.hr_cg_solve(self.g, m0, u, clover_fwd, clover_inv, b, x, ws, tol, max_iter, check_every, hr.stream_ptr())
        return x, it, rel
