"""z-slab decomposition of one periodic domain over several GPUs ("halo regions ...
exchanged between neighbouring subdomains", L126 "each GPU handles a slab").

One process per GPU owns ``nz_global / P`` consecutive z planes plus ``h`` halo planes on either side.  Every step is the
unchanged single-GPU step of the library on the padded box (a context created with ``halo_z = h``), followed by ONE
nearest-neighbour exchange: the byte ranges ``accLB_halo_chunks`` lists (whole planes of consecutive populations are
contiguous in the [z][i][y][x] layout, so nothing is packed) go to the two z-neighbours with NCCL send / recv over
NVLink -- ``torch.distributed`` point-to-point, nothing else.  With one rank both neighbours are the rank itself and the
exchange is two device copies; that is how the path is tested on one GPU (tests/test_gpu_slabs.py), next to the
world_size-2 ``gloo`` test of the message pairing on CPU buffers (tests/test_slabs_host.py).

This module holds no arithmetic of the method: plane bookkeeping and message pairing only.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

HALO_TWO_PHASE = 3  # WENO5 radius (R12); curvature of plane h-1 reaches phi of plane h-3
HALO_SINGLE = 1


@dataclass(frozen=True)
class Slab:
    """Planes [z0, z1) of the whole domain belong to `rank`; the local box adds `halo` planes on either side."""
    rank: int
    world: int
    nz_global: int
    z0: int
    z1: int
    halo: int

    @property
    def nz_own(self):
        return self.z1 - self.z0

    @property
    def nz_local(self):
        return self.nz_own + 2 * self.halo

    @property
    def z_origin(self):  # global coordinate of local plane 0
        return self.z0 - self.halo

    @property
    def below(self):  # rank that owns the planes under z0 (periodic)
        return (self.rank - 1) % self.world

    @property
    def above(self):
        return (self.rank + 1) % self.world

    def own(self, a, axis=0):
        """The slab's own planes of a local array (halo planes cut off)."""
        idx = [slice(None)] * a.ndim
        idx[axis] = slice(self.halo, self.halo + self.nz_own)
        return a[tuple(idx)]

    def take(self, a, axis=0):
        """The local box (own planes + halos, periodic wrap) out of an array of the whole domain."""
        assert a.shape[axis] == self.nz_global
        planes = np.arange(self.z_origin, self.z_origin + self.nz_local) % self.nz_global
        return np.ascontiguousarray(np.take(a, planes, axis=axis))


def make_slab(nz_global, world, rank, halo):
    """Equal slabs (nz_global divisible by world): what the paper's weak-scaling runs use."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError(f"rank {rank} of {world}")
    if nz_global % world:
        raise ValueError(f"nz_global = {nz_global} is not divisible by {world} ranks")
    own = nz_global // world
    if own < halo:
        raise ValueError(f"{own} planes per rank < halo {halo}: a neighbour's halo would reach past the next slab")
    return Slab(rank, world, nz_global, rank * own, (rank + 1) * own, halo)


def message_plan(chunks, slab):
    """Pair the ranges of ``accLB_halo_chunks`` with peers: (sends, recvs), each a list of (view, peer rank) in the order
    the messages must be posted.

    A range sent DOWN is received by the lower neighbour from ABOVE, so between one pair of ranks messages flow in two
    independent sequences.  With world = 2 both neighbours are the same rank: the peer posts its sends as [down..., up...],
    and what it sends down arrives here from above -- so receives are posted [from above..., from below...], which keeps
    the k-th message of the pair matched with the k-th receive for every world size.
    """
    sends = [(v, slab.below) for v, side, d in chunks if d == 0 and side < 0]
    sends += [(v, slab.above) for v, side, d in chunks if d == 0 and side > 0]
    recvs = [(v, slab.above) for v, side, d in chunks if d == 1 and side > 0]
    recvs += [(v, slab.below) for v, side, d in chunks if d == 1 and side < 0]
    assert len(sends) == len(recvs)
    return sends, recvs


def exchange(chunks, slab, group=None):
    """One halo exchange.  `chunks`: (uint8 tensor view, side, dir) as AccLB.halo_chunks() returns them."""
    sends, recvs = message_plan(chunks, slab)
    if slab.world == 1:
        # both neighbours are this rank: what goes down comes back in from above
        down = [v for v, side, d in chunks if d == 0 and side < 0]
        up = [v for v, side, d in chunks if d == 0 and side > 0]
        from_above = [v for v, side, d in chunks if d == 1 and side > 0]
        from_below = [v for v, side, d in chunks if d == 1 and side < 0]
        for src, dst in list(zip(down, from_above)) + list(zip(up, from_below)):
            assert src.numel() == dst.numel()
            dst.copy_(src)
        return
    import torch.distributed as dist

    ops = [dist.P2POp(dist.isend, v, peer, group=group) for v, peer in sends]
    ops += [dist.P2POp(dist.irecv, v, peer, group=group) for v, peer in recvs]
    for w in dist.batch_isend_irecv(ops):
        w.wait()


def exchange_in_process(parts):
    """The halo exchange between all the slabs of a domain held by ONE process: `parts[r]` = (chunks, slab) of rank r,
    ranks 0 .. world-1.  Plain tensor copies (peer copies over NVLink when the slabs live on different GPUs); also how the
    multi-slab path is tested on a single GPU."""
    world = len(parts)
    pick = lambda r, side, d: [v for v, sd, dd in parts[r][0] if sd == side and dd == d]
    for r, (_, slab) in enumerate(parts):
        assert slab.rank == r and slab.world == world
        for src, dst in list(zip(pick(r, -1, 0), pick(slab.below, +1, 1))) + list(zip(pick(r, +1, 0), pick(slab.above, -1, 1))):
            assert src.numel() == dst.numel()
            dst.copy_(src)


class SlabAccLB:
    """One z-slab of a periodic nx x ny x nz_global domain on this rank's GPU.

    Fields passed to ``init`` and returned by ``moments`` are LOCAL boxes [nz_local][ny][nx] (own planes + halos, see
    ``Slab.take`` / ``Slab.own``)."""

    def __init__(self, nx, ny, nz_global, *, rank=0, world=1, group=None, full_halo=False, device=0, **params):
        from . import binding

        halo = HALO_TWO_PHASE if params.get("two_phase") else HALO_SINGLE
        self.slab = make_slab(nz_global, world, rank, halo)
        self.group = group
        self.full_halo = bool(full_halo)
        self.sim = binding.AccLB(nx, ny, self.slab.nz_local, device=device, halo_z=halo, z_origin=self.slab.z_origin,
                                 nz_global=nz_global, **params)
        self.device = self.sim.device
        self.shape = self.sim.shape

    def close(self):
        self.sim.close()

    def exchange(self):
        exchange(self.sim.halo_chunks(self.full_halo), self.slab, self.group)

    def halo_bytes_per_step(self):
        """Bytes this rank sends per step (= bytes it receives)."""
        return sum(v.numel() for v, _, d in self.sim.halo_chunks(self.full_halo) if d == 0)

    def init(self, rho, u, phi=None):
        self.sim.init(rho, u, phi)  # the local fields carry their halos: nothing to exchange

    def step(self, nsteps=1):
        for _ in range(int(nsteps)):
            self.sim.step(1)
            self.exchange()

    def moments(self):
        """(rho, u, phi) of the slab's own planes."""
        rho, u, phi = self.sim.moments()
        s = self.slab
        return s.own(rho), s.own(u, axis=1), (s.own(phi) if phi is not None else None)

    def diagnostics(self):
        """R21 over the whole domain: sums added, means averaged (equal slabs), maximum taken over the ranks."""
        d = self.sim.diagnostics()
        if self.slab.world == 1:
            return d
        import torch
        import torch.distributed as dist

        dev = self.device if dist.get_backend(self.group) == "nccl" else "cpu"
        sums = torch.tensor([d[k] for k in ("ke", "dissipation", "sum_phi", "sum_pstar", "sum_mx", "sum_my", "sum_mz")],
                            dtype=torch.float64, device=dev)
        umax = torch.tensor([d["umax"]], dtype=torch.float64, device=dev)
        dist.all_reduce(sums, op=dist.ReduceOp.SUM, group=self.group)
        dist.all_reduce(umax, op=dist.ReduceOp.MAX, group=self.group)
        out = dict(d)
        for j, k in enumerate(("ke", "dissipation", "sum_phi", "sum_pstar", "sum_mx", "sum_my", "sum_mz")):
            out[k] = float(sums[j]) / (self.slab.world if j < 2 else 1)
        out["umax"] = float(umax[0])
        return out
