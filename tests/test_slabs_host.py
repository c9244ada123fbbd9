"""Host logic of the z-slab decomposition, on CPU: plane bookkeeping, and the message pairing of the halo
exchange over torch.distributed with the gloo backend, world_size 2 (both neighbours are the same peer) and 3, on fake
state buffers laid out like the library's ([z][i] planes of populations, [z] planes of phi) with the ranges that
include/acclb.h documents for accLB_halo_chunks."""
import socket
import subprocess
import sys
from pathlib import Path

import numpy as np
import pytest

from paper_2505_01126_b200 import slabs

ROOT = Path(__file__).resolve().parents[1]


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("world,nz,halo", [(1, 12, 3), (2, 12, 3), (4, 32, 1), (3, 9, 3)])
def test_slabs_tile_the_domain_and_take_wraps(world, nz, halo):
    a = np.arange(nz * 5, dtype=np.float64).reshape(nz, 5)
    own = []
    for r in range(world):
        s = slabs.make_slab(nz, world, r, halo)
        assert s.nz_local == nz // world + 2 * halo and s.z_origin == s.z0 - halo
        assert s.below == (r - 1) % world and s.above == (r + 1) % world
        loc = s.take(a)
        assert loc.shape[0] == s.nz_local
        for j in range(s.nz_local):
            assert np.array_equal(loc[j], a[(s.z_origin + j) % nz])
        own.append(s.own(loc))
        v = np.stack([a, a, a])  # a vector field: planes along axis 1
        assert np.array_equal(s.own(s.take(v, axis=1), axis=1)[2], s.own(loc))
    assert np.array_equal(np.concatenate(own), a)


def test_slab_errors():
    with pytest.raises(ValueError):
        slabs.make_slab(10, 3, 0, 1)      # not divisible
    with pytest.raises(ValueError):
        slabs.make_slab(8, 4, 0, 3)       # 2 planes per rank < halo 3
    with pytest.raises(ValueError):
        slabs.make_slab(8, 2, 2, 1)       # rank out of range


def test_message_plan_order():
    """Sends are posted [down..., up...], receives [from above..., from below...] (see message_plan)."""
    s = slabs.make_slab(12, 2, 0, 3)
    ch = [("sd0", -1, 0), ("sd1", -1, 0), ("su0", +1, 0), ("su1", +1, 0),
          ("rb0", -1, 1), ("rb1", -1, 1), ("ra0", +1, 1), ("ra1", +1, 1)]
    sends, recvs = slabs.message_plan(ch, s)
    assert [v for v, _ in sends] == ["sd0", "sd1", "su0", "su1"] and [p for _, p in sends] == [1, 1, 1, 1]
    assert [v for v, _ in recvs] == ["ra0", "ra1", "rb0", "rb1"]
    s3 = slabs.make_slab(12, 3, 0, 3)
    sends, recvs = slabs.message_plan(ch, s3)
    assert [p for _, p in sends] == [2, 2, 1, 1] and [p for _, p in recvs] == [1, 1, 2, 2]


# The fake state of one rank and the ranges of include/acclb.h (minimal set, two-phase): element value =
# rank * 10^6 + local plane * 100 + population index (phi: index 99).
WORKER = r"""
import sys
sys.path.insert(0, {root!r})
import torch
import torch.distributed as dist
from paper_2505_01126_b200 import slabs

world, rank, two_phase = {world}, int(sys.argv[1]), {two_phase}
dist.init_process_group("gloo", init_method="tcp://127.0.0.1:{port}", rank=rank, world_size=world)
h = 3 if two_phase else 1
K = 7                                  # elements per [ny][nx] plane
s = slabs.make_slab({nz}, world, rank, h)
nz = s.nz_local
f = torch.empty(nz, 27, K, dtype=torch.int64)
phi = torch.empty(nz, K, dtype=torch.int64)
def fill(r):
    z = torch.arange(nz).view(nz, 1, 1)
    i = torch.arange(27).view(1, 27, 1)
    return (r * 10**6 + z * 100 + i).expand(nz, 27, K).contiguous(), (r * 10**6 + torch.arange(nz).view(nz, 1) * 100 + 99).expand(nz, K).contiguous()
f0, p0 = fill(rank)
f.copy_(f0); phi.copy_(p0)
fb, pb = f.view(-1).view(torch.uint8), phi.view(-1).view(torch.uint8)
def pops(z, i0, i1, side, d):
    return (fb[(z * 27 + i0) * K * 8:(z * 27 + i1) * K * 8], side, d)
def phis(z0, side, d):
    return (pb[z0 * K * 8:(z0 + h) * K * 8], side, d)
lo, hi = (9, 18) if two_phase else (18, 9)
ch = [pops(h, 0, hi, -1, 0)] + ([pops(h + 1, 0, 9, -1, 0), phis(h, -1, 0)] if two_phase else [])
ch += [pops(nz - h - 1, lo, 27, +1, 0)] + ([pops(nz - h - 2, 18, 27, +1, 0), phis(nz - 2 * h, +1, 0)] if two_phase else [])
ch += [pops(h - 1, lo, 27, -1, 1)] + ([pops(h - 2, 18, 27, -1, 1), phis(0, -1, 1)] if two_phase else [])
ch += [pops(nz - h, 0, hi, +1, 1)] + ([pops(nz - h + 1, 0, 9, +1, 1), phis(nz - h, +1, 1)] if two_phase else [])
for _ in range(3):                     # repeated exchanges keep matching
    slabs.exchange(ch, s)
fb_, pb_ = fill(s.below)
fa_, pa_ = fill(s.above)
want_f, want_p = f0.clone(), p0.clone()
# from below: the lower neighbour's planes nz-h-1 (and nz-h-2, phi nz-2h ..) land in my planes h-1 (h-2, phi 0 ..)
want_f[h - 1, lo:] = fb_[nz - h - 1, lo:]
want_f[nz - h, :hi] = fa_[h, :hi]
if two_phase:
    want_f[h - 2, 18:] = fb_[nz - h - 2, 18:]
    want_f[nz - h + 1, :9] = fa_[h + 1, :9]
    want_p[0:h] = pb_[nz - 2 * h:nz - h]
    want_p[nz - h:] = pa_[h:2 * h]
assert torch.equal(f, want_f), (rank, (f != want_f).nonzero()[:5])
assert torch.equal(phi, want_p), rank
dist.barrier()
dist.destroy_process_group()
print("ok", rank)
"""


@pytest.mark.parametrize("world,two_phase", [(2, 1), (3, 1), (2, 0)])
def test_halo_exchange_gloo(world, two_phase):
    port = free_port()
    code = WORKER.format(root=str(ROOT), port=port, world=world, two_phase=two_phase, nz=12 * world)
    procs = [subprocess.Popen([sys.executable, "-c", code, str(r)], stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True)
             for r in range(world)]
    for p in procs:
        out, err = p.communicate(timeout=240)
        assert p.returncode == 0 and out.startswith("ok"), err[-3000:]


def test_exchange_single_rank_and_in_process():
    """world = 1 (the rank is its own neighbour) and the in-process exchange between several slabs, on CPU buffers."""
    import torch

    def state(r, nz):
        return torch.arange(nz * 4, dtype=torch.int64).view(nz, 4) + 1000 * r

    nz, h = 8, 1
    t = state(0, nz)
    b = t.view(-1).view(torch.uint8)
    row = lambda z: b[z * 32:(z + 1) * 32]
    ch = [(row(h), -1, 0), (row(nz - h - 1), +1, 0), (row(h - 1), -1, 1), (row(nz - h), +1, 1)]
    slabs.exchange(ch, slabs.make_slab(nz - 2 * h, 1, 0, h))
    assert torch.equal(t[0], t[nz - 2]) and torch.equal(t[nz - 1], t[1])
    parts, ts = [], []
    for r in range(3):
        t = state(r, nz)
        ts.append(t)
        b = t.view(-1).view(torch.uint8)
        row = lambda z, b=b: b[z * 32:(z + 1) * 32]
        parts.append(([(row(h), -1, 0), (row(nz - h - 1), +1, 0), (row(h - 1), -1, 1), (row(nz - h), +1, 1)],
                      slabs.make_slab(3 * (nz - 2 * h), 3, r, h)))
    slabs.exchange_in_process(parts)
    for r in range(3):
        assert torch.equal(ts[r][0], ts[(r - 1) % 3][nz - 2]) and torch.equal(ts[r][nz - 1], ts[(r + 1) % 3][1])
