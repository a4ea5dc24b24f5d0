"""Thin ctypes binding of libhr_dslash (include/hr_dslash.h): same names, argument marshalling only.

Every step of the path runs in the library's CUDA kernels; this module converts Python objects to
pointers and raises on a non-zero status.  PyTorch is used by callers only to allocate device memory
and streams (`device_buffer`, `stream_ptr`).  There is no CPU fallback: if the shared library is
missing, importing `lib()` fails loudly.
"""
from __future__ import annotations

import ctypes
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libhr_dslash.so")

OK, EINVAL, EUNSUPPORTED, EALIGN, ECUDA = 0, 1, 2, 3, 4
REP_FUND, REP_ADJ, REP_SU3 = 0, 1, 2
PREC_F64, PREC_F32 = 0, 1
LINKS_FULL, LINKS_COMPRESSED, LINKS_ONTHEFLY = 0, 1, 2
KERNEL_AUTO, KERNEL_GENERIC, KERNEL_TILED = 0, 1, 2
EVEN, ODD, BOTH = 0, 1, 2
EO_HOP_OE, EO_HOP_EO, EO_DHAT = 0, 1, 2
HOST_DIRAC = 3
EPI_NONE, EPI_AXPY, EPI_CLOVER_INV, EPI_CLOVER_AXPY = 0, 1, 2, 3
OP_HOP, OP_DIRAC, OP_DHAT, OP_CLOVER, OP_DHAT_CLOVER, OP_REPRESENT = 0, 1, 2, 3, 4, 5
STATIC_SCRATCH_BYTES = 8 << 20   # HR_STATIC_SCRATCH_BYTES of include/hr_dslash.h

# every symbol include/hr_dslash.h declares (tests/test_abi.py checks the header against this list)
SYMBOLS = [
    "hr_spinor_bytes", "hr_gauge_bytes", "hr_clover_bytes", "hr_canonical_spinor_bytes",
    "hr_canonical_gauge_bytes", "hr_canonical_clover_bytes", "hr_pack_spinor", "hr_unpack_spinor",
    "hr_pack_gauge", "hr_unpack_gauge", "hr_pack_clover", "hr_unpack_clover", "hr_represent_gauge", "hr_represent_gauge_antisym",
    "hr_dirac_apply", "hr_dirac_clover_apply", "hr_dirac_eo_apply", "hr_dhat_apply_static", "hr_clover_build", "hr_clover_build_exp", "hr_clover_apply", "hr_clover_count_nonfinite", "hr_dirac_flops_bytes",
    "hr_host_workspace_bytes", "hr_dirac_apply_host", "hr_dirac_eo_apply_host", "hr_gauge_upload_host",
    "hr_host_batch_workspace_bytes", "hr_apply_host_batch", "hr_apply_host_ops", "hr_halo_face_bytes", "hr_halo_pack", "hr_hop_local",
    "hr_hop_local_interior", "hr_hop_local_boundary", "hr_last_error",
    "hr_launch_count", "hr_kernel_name", "hr_kernel_plan", "hr_cg_workspace_bytes", "hr_cg_solve",
    "hr_cg_mixed_workspace_bytes", "hr_cg_solve_mixed", "hr_cg_solve_mixed_clover",
]


class hr_geom(ctypes.Structure):
    _fields_ = [("L", ctypes.c_int * 4), ("rep", ctypes.c_int), ("prec", ctypes.c_int),
                ("link_storage", ctypes.c_int), ("kernel", ctypes.c_int)]


class hr_decomp(ctypes.Structure):
    _fields_ = [("split", ctypes.c_int * 4)]


class HrError(RuntimeError):
    def __init__(self, status, text):
        super().__init__("libhr_dslash status %d: %s" % (status, text))
        self.status = status


_lib = None


def lib():
    """Load libhr_dslash.so (built in-tree by paper_2411_18511_b200.build).  No fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s is missing: run `python -m paper_2411_18511_b200.build` "
                              "(there is no CPU fallback)" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        G, V, I, D, S = ctypes.POINTER(hr_geom), ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
        PD = ctypes.POINTER(ctypes.c_double)
        sig = {
            "hr_spinor_bytes": (S, [G, I]), "hr_gauge_bytes": (S, [G, I]), "hr_clover_bytes": (S, [G]),
            "hr_canonical_spinor_bytes": (S, [G]), "hr_canonical_gauge_bytes": (S, [G, I]),
            "hr_canonical_clover_bytes": (S, [G]),
            "hr_pack_spinor": (I, [G, V, V, V]), "hr_unpack_spinor": (I, [G, V, V, V]),
            "hr_pack_gauge": (I, [G, I, V, V, V]), "hr_unpack_gauge": (I, [G, I, V, V, V]),
            "hr_pack_clover": (I, [G, V, V, V]), "hr_unpack_clover": (I, [G, V, V, V]),
            "hr_represent_gauge": (I, [G, V, V, V]),
            "hr_represent_gauge_antisym": (I, [G, V, V, V]),
            "hr_dirac_apply": (I, [G, D, V, V, V, V]),
            "hr_dirac_clover_apply": (I, [G, V, V, V, V, V]),
            "hr_dirac_eo_apply": (I, [G, I, D, V, V, V, V, V, V, V]),
            "hr_dhat_apply_static": (I, [G, D, V, V, V, V, V, V]),
            "hr_clover_build": (I, [G, D, D, V, V, V, V]),
            "hr_clover_build_exp": (I, [G, D, D, V, V, V, V]),
            "hr_clover_apply": (I, [G, I, V, V, V, V]),
            "hr_clover_count_nonfinite": (I, [G, V, V, V]),
            "hr_dirac_flops_bytes": (I, [G, I, PD, PD, PD]),
            "hr_host_workspace_bytes": (S, [G]),
            "hr_dirac_apply_host": (I, [G, D, V, V, V, V, V]),
            "hr_dirac_eo_apply_host": (I, [G, I, D, V, V, V, V, V]),
            "hr_gauge_upload_host": (I, [G, I, V, V, V, V]),
            "hr_host_batch_workspace_bytes": (S, [G]),
            "hr_apply_host_batch": (I, [G, I, D, V, V, V, I, ctypes.POINTER(V), ctypes.POINTER(V), V, V]),
            "hr_apply_host_ops": (I, [G, ctypes.POINTER(ctypes.c_int), D, V, V, V, I, ctypes.POINTER(V), ctypes.POINTER(V), V, V]),
            "hr_halo_face_bytes": (S, [G, I]),
            "hr_halo_pack": (I, [G, ctypes.POINTER(hr_decomp), I, V, V, ctypes.POINTER(V), V]),
            "hr_hop_local": (I, [G, ctypes.POINTER(hr_decomp), I, I, D, D, V, V, V, V, V, ctypes.POINTER(V), V]),
            "hr_hop_local_interior": (I, [G, ctypes.POINTER(hr_decomp), I, I, D, D, V, V, V, V, V, V]),
            "hr_hop_local_boundary": (I, [G, ctypes.POINTER(hr_decomp), I, I, D, V, V, V, ctypes.POINTER(V), V]),
            "hr_last_error": (S, [ctypes.c_char_p, S]),
            "hr_launch_count": (ctypes.c_ulonglong, []),
            "hr_kernel_name": (ctypes.c_char_p, [G]),
            "hr_kernel_plan": (I, [G, I, ctypes.POINTER(ctypes.c_int)]),
            "hr_cg_workspace_bytes": (S, [G]),
            "hr_cg_mixed_workspace_bytes": (S, [G]),
            "hr_cg_solve_mixed": (I, [G, D, V, V, V, V, V, D, D, I, I, I, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int), PD, V]),
            "hr_cg_solve_mixed_clover": (I, [G, D, V, V, V, V, V, V, V, V, V, D, D, I, I, I, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_int), PD, V]),
            "hr_cg_solve": (I, [G, D, V, V, V, V, V, V, D, I, I, ctypes.POINTER(ctypes.c_int), PD, V]),
        }
        for name, (res, args) in sig.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def geom(L, rep=REP_FUND, prec=PREC_F64, link_storage=LINKS_COMPRESSED, kernel=KERNEL_AUTO) -> hr_geom:
    g = hr_geom()
    for i in range(4):
        g.L[i] = int(L[i])
    g.rep, g.prec, g.link_storage, g.kernel = int(rep), int(prec), int(link_storage), int(kernel)
    return g


def _ptr(x):
    """torch tensor / numpy array / int / None -> integer address (or None)"""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    raise TypeError("cannot take the address of %r" % type(x))


def stream_ptr(stream=None):
    """cudaStream_t of a torch.cuda.Stream (None: torch's current stream)."""
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def last_error() -> str:
    buf = ctypes.create_string_buffer(512)
    lib().hr_last_error(buf, 512)
    return buf.value.decode()


def _check(status):
    if status != OK:
        raise HrError(status, last_error())


# ------------------------------------------------------------------ sizes
def hr_spinor_bytes(g, parity=BOTH): return lib().hr_spinor_bytes(ctypes.byref(g), parity)
def hr_gauge_bytes(g, rep): return lib().hr_gauge_bytes(ctypes.byref(g), rep)
def hr_clover_bytes(g): return lib().hr_clover_bytes(ctypes.byref(g))
def hr_canonical_spinor_bytes(g): return lib().hr_canonical_spinor_bytes(ctypes.byref(g))
def hr_canonical_gauge_bytes(g, rep): return lib().hr_canonical_gauge_bytes(ctypes.byref(g), rep)
def hr_canonical_clover_bytes(g): return lib().hr_canonical_clover_bytes(ctypes.byref(g))
def hr_host_workspace_bytes(g): return lib().hr_host_workspace_bytes(ctypes.byref(g))


# ------------------------------------------------------------------ layout
def hr_pack_spinor(g, canon, dev, stream=0): _check(lib().hr_pack_spinor(ctypes.byref(g), _ptr(canon), _ptr(dev), stream))
def hr_unpack_spinor(g, dev, canon, stream=0): _check(lib().hr_unpack_spinor(ctypes.byref(g), _ptr(dev), _ptr(canon), stream))
def hr_pack_gauge(g, rep, canon, dev, stream=0): _check(lib().hr_pack_gauge(ctypes.byref(g), rep, _ptr(canon), _ptr(dev), stream))
def hr_unpack_gauge(g, rep, dev, canon, stream=0): _check(lib().hr_unpack_gauge(ctypes.byref(g), rep, _ptr(dev), _ptr(canon), stream))
def hr_pack_clover(g, canon, dev, stream=0): _check(lib().hr_pack_clover(ctypes.byref(g), _ptr(canon), _ptr(dev), stream))
def hr_unpack_clover(g, dev, canon, stream=0): _check(lib().hr_unpack_clover(ctypes.byref(g), _ptr(dev), _ptr(canon), stream))


# ------------------------------------------------------------------ operators
def hr_represent_gauge(g, u_fund, u_adj, stream=0):
    _check(lib().hr_represent_gauge(ctypes.byref(g), _ptr(u_fund), _ptr(u_adj), stream))


def hr_represent_gauge_antisym(g, u_fund, u_rep, stream=0):
    _check(lib().hr_represent_gauge_antisym(ctypes.byref(g), _ptr(u_fund), _ptr(u_rep), stream))


def hr_dirac_apply(g, m0, u, psi, out, stream=0):
    _check(lib().hr_dirac_apply(ctypes.byref(g), float(m0), _ptr(u), _ptr(psi), _ptr(out), stream))


def hr_dirac_clover_apply(g, u, clover_fwd, psi, out, stream=0):
    _check(lib().hr_dirac_clover_apply(ctypes.byref(g), _ptr(u), _ptr(clover_fwd), _ptr(psi), _ptr(out), stream))


def hr_dirac_eo_apply(g, op, m0, u, clover_fwd, clover_inv, inp, out, tmp, stream=0):
    _check(lib().hr_dirac_eo_apply(ctypes.byref(g), int(op), float(m0), _ptr(u), _ptr(clover_fwd), _ptr(clover_inv),
                                   _ptr(inp), _ptr(out), _ptr(tmp), stream))


def hr_dhat_apply_static(g, m0, u, clover_fwd, clover_inv, inp, out, stream=0):
    """Dhat with the odd half field between the two hops in the library's static device array (no allocation;
    lattices up to STATIC_SCRATCH_BYTES per odd half field)."""
    _check(lib().hr_dhat_apply_static(ctypes.byref(g), float(m0), _ptr(u), _ptr(clover_fwd), _ptr(clover_inv),
                                      _ptr(inp), _ptr(out), stream))


def hr_clover_build(g, m0, csw, u_fund, clover_fwd, clover_inv, stream=0):
    _check(lib().hr_clover_build(ctypes.byref(g), float(m0), float(csw), _ptr(u_fund), _ptr(clover_fwd), _ptr(clover_inv), stream))


def hr_clover_build_exp(g, m0, csw, u_fund, clover_fwd, clover_inv, stream=0):
    _check(lib().hr_clover_build_exp(ctypes.byref(g), float(m0), float(csw), _ptr(u_fund), _ptr(clover_fwd), _ptr(clover_inv), stream))


def hr_clover_apply(g, parity, blocks, inp, out, stream=0):
    _check(lib().hr_clover_apply(ctypes.byref(g), int(parity), _ptr(blocks), _ptr(inp), _ptr(out), stream))


def hr_clover_count_nonfinite(g, blocks, count_dev, stream=0):
    _check(lib().hr_clover_count_nonfinite(ctypes.byref(g), _ptr(blocks), _ptr(count_dev), stream))


def hr_dirac_flops_bytes(g, op):
    """-> (flops per output site, compulsory bytes per site, requested bytes per site)"""
    f, bc, br = ctypes.c_double(), ctypes.c_double(), ctypes.c_double()
    _check(lib().hr_dirac_flops_bytes(ctypes.byref(g), int(op), ctypes.byref(f), ctypes.byref(bc), ctypes.byref(br)))
    return f.value, bc.value, br.value


def hr_dirac_apply_host(g, m0, u_canon_host, psi_canon_host, out_canon_host, workspace, stream=0):
    _check(lib().hr_dirac_apply_host(ctypes.byref(g), float(m0), _ptr(u_canon_host), _ptr(psi_canon_host),
                                     _ptr(out_canon_host), _ptr(workspace), stream))


def hr_dirac_eo_apply_host(g, op, m0, u_canon_host, in_canon_host, out_canon_host, workspace, stream=0):
    _check(lib().hr_dirac_eo_apply_host(ctypes.byref(g), int(op), float(m0), _ptr(u_canon_host), _ptr(in_canon_host),
                                        _ptr(out_canon_host), _ptr(workspace), stream))


def hr_gauge_upload_host(g, rep, u_canon_host, u_dev, workspace, stream=0):
    _check(lib().hr_gauge_upload_host(ctypes.byref(g), int(rep), _ptr(u_canon_host), _ptr(u_dev), _ptr(workspace), stream))


def hr_host_batch_workspace_bytes(g): return lib().hr_host_batch_workspace_bytes(ctypes.byref(g))


def hr_apply_host_batch(g, op, m0, u_dev, clover_fwd, clover_inv, ins, outs, workspace, stream=0):
    """ins / outs: sequences of canonical host arrays (torch pinned tensors or numpy arrays), one per right-hand side"""
    n = len(ins)
    assert len(outs) == n
    pin = (ctypes.c_void_p * n)(*[_ptr(a) for a in ins])
    pout = (ctypes.c_void_p * n)(*[_ptr(a) for a in outs])
    _check(lib().hr_apply_host_batch(ctypes.byref(g), int(op), float(m0), _ptr(u_dev), _ptr(clover_fwd), _ptr(clover_inv), n, pin, pout,
                                     _ptr(workspace), stream))


def hr_apply_host_ops(g, ops, m0, u_dev, clover_fwd, clover_inv, ins, outs, workspace, stream=0):
    """one operator per item (ops[i]): the pipeline of hr_apply_host_batch across a sequence of different operators"""
    n = len(ins)
    assert len(outs) == n and len(ops) == n
    pin = (ctypes.c_void_p * n)(*[_ptr(a) for a in ins])
    pout = (ctypes.c_void_p * n)(*[_ptr(a) for a in outs])
    pops = (ctypes.c_int * n)(*[int(o) for o in ops])
    _check(lib().hr_apply_host_ops(ctypes.byref(g), pops, float(m0), _ptr(u_dev), _ptr(clover_fwd), _ptr(clover_inv), n, pin, pout,
                                   _ptr(workspace), stream))


def decomp(split) -> hr_decomp:
    d = hr_decomp()
    for i in range(4):
        d.split[i] = int(bool(split[i]))
    return d


def hr_halo_face_bytes(g, mu): return lib().hr_halo_face_bytes(ctypes.byref(g), int(mu))


def _faces(faces):
    """8 device buffers (or None) -> C array of 8 pointers"""
    assert len(faces) == 8
    return (ctypes.c_void_p * 8)(*[_ptr(f) for f in faces])


def hr_halo_pack(g, d, in_parity, u, in_half, face_out, stream=0):
    _check(lib().hr_halo_pack(ctypes.byref(g), ctypes.byref(d), int(in_parity), _ptr(u), _ptr(in_half), _faces(face_out), stream))


def hr_hop_local(g, d, out_parity, epi, a, c, u, clover, in_half, phi_half, out_half, face_in, stream=0):
    _check(lib().hr_hop_local(ctypes.byref(g), ctypes.byref(d), int(out_parity), int(epi), float(a), float(c), _ptr(u), _ptr(clover),
                              _ptr(in_half), _ptr(phi_half), _ptr(out_half), _faces(face_in), stream))


def hr_hop_local_interior(g, d, out_parity, epi, a, c, u, clover, in_half, phi_half, out_half, stream=0):
    _check(lib().hr_hop_local_interior(ctypes.byref(g), ctypes.byref(d), int(out_parity), int(epi), float(a), float(c), _ptr(u), _ptr(clover),
                                       _ptr(in_half), _ptr(phi_half), _ptr(out_half), stream))


def hr_hop_local_boundary(g, d, out_parity, epi, c, u, clover, out_half, face_in, stream=0):
    _check(lib().hr_hop_local_boundary(ctypes.byref(g), ctypes.byref(d), int(out_parity), int(epi), float(c), _ptr(u), _ptr(clover),
                                       _ptr(out_half), _faces(face_in), stream))


def hr_cg_workspace_bytes(g): return lib().hr_cg_workspace_bytes(ctypes.byref(g))


def hr_cg_solve(g, m0, u, clover_fwd, clover_inv, b, x, workspace, tol, max_iter, check_every=5, stream=0):
    """-> (iterations, |r|/|b|)"""
    it, rel = ctypes.c_int(), ctypes.c_double()
    _check(lib().hr_cg_solve(ctypes.byref(g), float(m0), _ptr(u), _ptr(clover_fwd), _ptr(clover_inv), _ptr(b), _ptr(x),
                             _ptr(workspace), float(tol), int(max_iter), int(check_every), ctypes.byref(it), ctypes.byref(rel), stream))
    return it.value, rel.value


def hr_cg_mixed_workspace_bytes(g): return lib().hr_cg_mixed_workspace_bytes(ctypes.byref(g))


def hr_cg_solve_mixed(g, m0, u_f64, u_f32, b, x, workspace, tol, inner_tol=1e-3, max_outer=30, max_inner=1000, check_every=5, stream=0):
    """-> (outer corrections, total fp32 iterations, true |r|/|b|)"""
    no, ni, rel = ctypes.c_int(), ctypes.c_int(), ctypes.c_double()
    _check(lib().hr_cg_solve_mixed(ctypes.byref(g), float(m0), _ptr(u_f64), _ptr(u_f32), _ptr(b), _ptr(x), _ptr(workspace), float(tol),
                                   float(inner_tol), int(max_outer), int(max_inner), int(check_every), ctypes.byref(no), ctypes.byref(ni),
                                   ctypes.byref(rel), stream))
    return no.value, ni.value, rel.value


def hr_cg_solve_mixed_clover(g, m0, u_f64, u_f32, cf64, ci64, cf32, ci32, b, x, workspace, tol, inner_tol=1e-3, max_outer=30,
                             max_inner=1000, check_every=5, stream=0):
    """-> (outer corrections, total fp32 iterations, true |r|/|b|)"""
    no, ni, rel = ctypes.c_int(), ctypes.c_int(), ctypes.c_double()
    _check(lib().hr_cg_solve_mixed_clover(ctypes.byref(g), float(m0), _ptr(u_f64), _ptr(u_f32), _ptr(cf64), _ptr(ci64), _ptr(cf32), _ptr(ci32),
                                          _ptr(b), _ptr(x), _ptr(workspace), float(tol), float(inner_tol), int(max_outer), int(max_inner),
                                          int(check_every), ctypes.byref(no), ctypes.byref(ni), ctypes.byref(rel), stream))
    return no.value, ni.value, rel.value


def hr_launch_count() -> int: return int(lib().hr_launch_count())
def hr_kernel_name(g) -> str: return lib().hr_kernel_name(ctypes.byref(g)).decode()


def hr_kernel_plan(g, op=OP_HOP) -> dict:
    """launch plan of the kernel behind a parity hop (OP_HOP) or the full operator (OP_DIRAC); needs a CUDA device"""
    info = (ctypes.c_int * 8)()
    _check(lib().hr_kernel_plan(ctypes.byref(g), int(op), info))
    keys = ("kernel", "t1", "t2", "nseg", "seglen", "threads", "smem", "grid")
    return dict(zip(keys, (int(v) for v in info)))


# ------------------------------------------------------------------ plumbing: device memory via torch
def current_device() -> str:
    """the calling thread's current CUDA device as a torch device string (one process per GPU sets it once)"""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("libhr_dslash needs a CUDA device; there is no CPU fallback")
    return "cuda:%d" % torch.cuda.current_device()


def device_buffer(nbytes: int, device=None):
    """A torch uint8 buffer of nbytes on `device` (default: the current device; 256-byte aligned by the caching allocator)."""
    import torch
    return torch.empty(int(nbytes), dtype=torch.uint8, device=current_device() if device is None else device)


def np_real(g):
    import numpy as np
    return np.float64 if g.prec == PREC_F64 else np.float32


def np_complex(g):
    import numpy as np
    return np.complex128 if g.prec == PREC_F64 else np.complex64


def upload(array, device=None):
    """numpy array -> uint8 buffer on `device` (default: the current device) holding the same bytes"""
    import numpy as np
    import torch
    a = np.ascontiguousarray(array)
    return torch.from_numpy(a.view(np.uint8).reshape(-1)).to(current_device() if device is None else device)


def download(buf, dtype, shape):
    """device uint8 buffer -> numpy array of dtype/shape"""
    import numpy as np
    return buf.cpu().numpy().view(dtype).reshape(shape)
