"""The sharded operator: composition and transport around hr_halo_pack / hr_hop_local (include/hr_dslash.h,
DESIGN.md §8).  Marshalling and data movement only — every arithmetic step (face projection, link multiply, interior and
boundary terms, epilogues) runs in the library's kernels.

One `Shard` = one rank's local lattice of a P0 x P1 x P2 x P3 domain decomposition (Fig. 4: "all four
dimensions parallelized"): ordinary device-layout fields plus, per cut direction, two send and two receive face buffers.
Transport is pluggable:
  * `exchange_in_process(shards)`     all shards live in this process (one GPU): device-to-device copies — the
                                      single-GPU self-exchange the parity tests use;
  * `exchange_distributed(shard, ..)` one shard per process: torch.distributed batched isend/irecv (NCCL over NVLink on
                                      GPUs, gloo on CPU tensors in the plumbing test).
With peer-mapped receive buffers the pack kernel can store straight into the neighbour's memory (pass those pointers as
`face_out`); then the "exchange" is only a synchronisation.
"""
from __future__ import annotations

import itertools

import numpy as np

from . import hr


# ------------------------------------------------------------------ decomposition of canonical arrays (indexing only)
def rank_coords(P):
    """all rank coordinates of a P0 x P1 x P2 x P3 process grid, rank index = lexicographic (last fastest)"""
    return list(itertools.product(*[range(int(p)) for p in P]))


def rank_of(coords, P):
    r = 0
    for c, p in zip(coords, P):
        r = r * int(p) + (int(c) % int(p))
    return r


def local_extents(Lg, P):
    L = tuple(int(l) // int(p) for l, p in zip(Lg, P))
    assert all(l * int(p) == int(lg) and l % 2 == 0 for l, p, lg in zip(L, P, Lg)), "every local extent must be even"
    return L


def local_block(a, Lg, P, coords):
    """the block of a canonical array [V_global, ...] that rank `coords` owns, as a canonical array [V_local, ...]"""
    L = local_extents(Lg, P)
    g = a.reshape(tuple(Lg) + a.shape[1:])
    sl = tuple(slice(c * l, (c + 1) * l) for c, l in zip(coords, L))
    return np.ascontiguousarray(g[sl]).reshape((-1,) + a.shape[1:])


def assemble(blocks, Lg, P):
    """inverse of local_block: {coords: [V_local, ...]} -> [V_global, ...]"""
    L = local_extents(Lg, P)
    first = next(iter(blocks.values()))
    out = np.empty(tuple(Lg) + first.shape[1:], dtype=first.dtype)
    for coords, b in blocks.items():
        sl = tuple(slice(c * l, (c + 1) * l) for c, l in zip(coords, L))
        out[sl] = b.reshape(L + first.shape[1:])
    return out.reshape((-1,) + first.shape[1:])


# ------------------------------------------------------------------ one rank
class RankGrid:
    """a rank's place in the process grid: which directions are cut and who the neighbours are (no device state)"""

    def __init__(self, P, coords, split=None):
        self.P, self.coords = tuple(int(p) for p in P), tuple(int(c) for c in coords)
        self.split = tuple(int(p) > 1 for p in P) if split is None else tuple(bool(s) for s in split)

    def neighbour(self, mu, sign):
        c = list(self.coords)
        c[mu] = (c[mu] + sign) % self.P[mu]
        return tuple(c)


class Shard(RankGrid):
    def __init__(self, lattice, P, coords, split=None):
        """lattice: a paper_2411_18511_b200.lattice.Lattice of the LOCAL extents; P: process grid; coords: this rank's
        position in it; split: which directions are cut (default: those with more than one rank)"""
        super().__init__(P, coords, split)
        self.lat = lattice
        self.d = hr.decomp(self.split)
        g = lattice.g
        self.send = [None] * 8
        self.recv = [None] * 8
        for mu in range(4):
            if self.split[mu]:
                n = hr.hr_halo_face_bytes(g, mu)
                for s in (0, 1):
                    self.send[2 * mu + s] = hr.device_buffer(n, lattice.device)
                    self.recv[2 * mu + s] = hr.device_buffer(n, lattice.device)

    def pack(self, in_parity, u, in_half, stream=None):
        hr.hr_halo_pack(self.lat.g, self.d, in_parity, u, in_half, self.send, hr.stream_ptr() if stream is None else stream)

    def hop(self, out_parity, u, in_half, out_half, epi=hr.EPI_NONE, a=0.0, c=1.0, clover=None, phi=None, stream=None):
        hr.hr_hop_local(self.lat.g, self.d, out_parity, epi, a, c, u, clover, in_half, phi, out_half, self.recv,
                        hr.stream_ptr() if stream is None else stream)

    def hop_interior(self, out_parity, u, in_half, out_half, epi=hr.EPI_NONE, a=0.0, c=1.0, clover=None, phi=None, stream=None):
        hr.hr_hop_local_interior(self.lat.g, self.d, out_parity, epi, a, c, u, clover, in_half, phi, out_half,
                                 hr.stream_ptr() if stream is None else stream)

    def hop_boundary(self, out_parity, u, out_half, epi=hr.EPI_NONE, c=1.0, clover=None, stream=None):
        hr.hr_hop_local_boundary(self.lat.g, self.d, out_parity, epi, c, u, clover, out_half, self.recv,
                                 hr.stream_ptr() if stream is None else stream)


# ------------------------------------------------------------------ transport
def exchange_in_process(shards):
    """shards: {coords: Shard}, all on this process's device.  Down faces go to the rank at -mu, up faces to +mu
    (stream-ordered device-to-device copies on torch's current stream)."""
    for sh in shards.values():
        for mu in range(4):
            if not sh.split[mu]:
                continue
            shards[sh.neighbour(mu, -1)].recv[2 * mu].copy_(sh.send[2 * mu], non_blocking=True)
            shards[sh.neighbour(mu, +1)].recv[2 * mu + 1].copy_(sh.send[2 * mu + 1], non_blocking=True)


def exchange_distributed(shard, dist, send=None, recv=None):
    """one shard per process: batched isend / irecv of the faces (NCCL: over NVLink; gloo: CPU tensors).  A rank that is
    its own neighbour in a direction copies locally.  send / recv default to the shard's own buffers."""
    send = shard.send if send is None else send
    recv = shard.recv if recv is None else recv
    ops = []
    me = rank_of(shard.coords, shard.P)
    for mu in range(4):
        if not shard.split[mu]:
            continue
        lo, hi = rank_of(shard.neighbour(mu, -1), shard.P), rank_of(shard.neighbour(mu, +1), shard.P)
        if lo == me and hi == me:
            recv[2 * mu].copy_(send[2 * mu])
            recv[2 * mu + 1].copy_(send[2 * mu + 1])
            continue
        # same order on every rank, so that messages between one pair of ranks match up (P_mu = 2: lo == hi)
        ops += [dist.P2POp(dist.isend, send[2 * mu], lo, tag=2 * mu), dist.P2POp(dist.irecv, recv[2 * mu], hi, tag=2 * mu),
                dist.P2POp(dist.isend, send[2 * mu + 1], hi, tag=2 * mu + 1), dist.P2POp(dist.irecv, recv[2 * mu + 1], lo, tag=2 * mu + 1)]
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()


# ------------------------------------------------------------------ operators on a set of shards in one process
_comm_streams = {}


def comm_stream(device):
    """the side stream pack + transfer run on when they overlap the interior kernel (one per device, made on first use)"""
    import torch
    if device not in _comm_streams:
        _comm_streams[device] = torch.cuda.Stream(device=device)
    return _comm_streams[device]


def hop_all(shards, exchange, out_parity, U, inp, out, overlap=False, **kw):
    """out[c] (half field of parity out_parity) = epilogue(H inp[c]) on every shard c; U, inp, out: {coords: buffer}.
    overlap=True: pack and transfer run on a side stream while the interior kernels run on the current one,
    the boundary kernels follow once the faces have arrived."""
    def per_shard(c):
        return {k: (v[c] if isinstance(v, dict) else v) for k, v in kw.items()}
    if not overlap:
        for c, sh in shards.items():
            sh.pack(1 - out_parity, U[c], inp[c])
        exchange(shards)
        for c, sh in shards.items():
            sh.hop(out_parity, U[c], inp[c], out[c], **per_shard(c))
        return
    import torch
    main = torch.cuda.current_stream()
    side = comm_stream(next(iter(shards.values())).lat.device)
    side.wait_stream(main)                       # the input (and the face buffers' last readers) are ready
    with torch.cuda.stream(side):
        for c, sh in shards.items():
            sh.pack(1 - out_parity, U[c], inp[c])
        exchange(shards)
    for c, sh in shards.items():
        sh.hop_interior(out_parity, U[c], inp[c], out[c], **per_shard(c))
    main.wait_stream(side)
    for c, sh in shards.items():
        kwc = per_shard(c)
        sh.hop_boundary(out_parity, U[c], out[c], epi=kwc.get("epi", hr.EPI_NONE), c=kwc.get("c", 1.0), clover=kwc.get("clover"))


def dhat_all(shards, exchange, m0, U, in_e, out_e, tmp_o, clover_fwd=None, clover_inv=None, overlap=False):
    """the even-odd operator on the global lattice: hop o<-e, exchange, hop e<-o with its epilogue (E1 / E2)"""
    if clover_fwd is None:
        d = 4.0 + m0
        hop_all(shards, exchange, hr.ODD, U, in_e, tmp_o, overlap=overlap)
        hop_all(shards, exchange, hr.EVEN, U, tmp_o, out_e, overlap=overlap, epi=hr.EPI_AXPY, a=d, c=-1.0 / (4.0 * d), phi=in_e)
    else:
        hop_all(shards, exchange, hr.ODD, U, in_e, tmp_o, overlap=overlap, epi=hr.EPI_CLOVER_INV, clover=clover_inv)
        hop_all(shards, exchange, hr.EVEN, U, tmp_o, out_e, overlap=overlap, epi=hr.EPI_CLOVER_AXPY, c=-0.25, clover=clover_fwd, phi=in_e)


def dirac_all(shards, exchange, m0, U, psi, out):
    """full D on the global lattice: the two parity hops, each with the axpy epilogue on its own half of psi"""
    for p in (hr.EVEN, hr.ODD):
        half_in = {c: (sh.lat.odd(psi[c]) if p == hr.EVEN else sh.lat.even(psi[c])) for c, sh in shards.items()}
        half_phi = {c: (sh.lat.even(psi[c]) if p == hr.EVEN else sh.lat.odd(psi[c])) for c, sh in shards.items()}
        half_out = {c: (sh.lat.even(out[c]) if p == hr.EVEN else sh.lat.odd(out[c])) for c, sh in shards.items()}
        hop_all(shards, exchange, p, U, half_in, half_out, epi=hr.EPI_AXPY, a=4.0 + m0, c=-0.5, phi=half_phi)
