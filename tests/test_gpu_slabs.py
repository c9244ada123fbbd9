"""z-slab decomposition through the C ABI on ONE GPU: the whole periodic domain cut into P slabs with halo
planes, advanced slab by slab with the halo ranges of accLB_halo_chunks copied between them after every step, must give
the fields of the undivided periodic box -- to rounding (the seam fluxes are added with atomics and the z chunks of a
padded box fall elsewhere), and the CPU oracle's fields within the usual 1e-11.  P = 1 uses the rank's own exchange()
(both neighbours are the rank itself), P = 2, 3 the in-process exchange between several contexts."""
import numpy as np
import pytest
import torch

from paper_2505_01126_b200 import slabs, workloads as wl
from test_gpu_parity import TOL, cpu_sim, gpu_sim, ragged_two_phase

pytestmark = pytest.mark.gpu

SAME = 1e-13  # slab run vs undivided run: the same arithmetic up to the order of the seam additions


class Domain:
    """All P slabs of one domain in this process, on cuda:0."""

    def __init__(self, acclb, cfg, shape, world, full_halo=False, **extra):
        nx, ny, nz = shape
        self.parts = [slabs.SlabAccLB(nx, ny, nz, rank=r, world=world, full_halo=full_halo, **cfg["params"], **extra)
                      for r in range(world)]
        dev = self.parts[0].device
        for p in self.parts:
            s = p.slab
            phi = cfg.get("phi")
            p.init(torch.from_numpy(s.take(cfg["rho"])).to(dev), torch.from_numpy(s.take(cfg["u"], axis=1)).to(dev),
                   torch.from_numpy(s.take(phi)).to(dev) if phi is not None else None)

    def step(self, n):
        for _ in range(n):
            for p in self.parts:
                p.sim.step(1)
            if len(self.parts) == 1:
                self.parts[0].exchange()
            else:
                slabs.exchange_in_process([(p.sim.halo_chunks(p.full_halo), p.slab) for p in self.parts])

    def moments(self):
        ms = [p.moments() for p in self.parts]
        rho = np.concatenate([m[0].cpu().numpy() for m in ms], axis=0)
        u = np.concatenate([m[1].cpu().numpy() for m in ms], axis=1)
        phi = np.concatenate([m[2].cpu().numpy() for m in ms], axis=0) if ms[0][2] is not None else None
        return rho, u, phi

    def diagnostics(self):
        ds = [p.sim.diagnostics() for p in self.parts]
        out = {k: sum(d[k] for d in ds) for k in ("sum_phi", "sum_pstar", "sum_mx", "sum_my", "sum_mz")}
        out["ke"] = sum(d["ke"] for d in ds) / len(ds)
        out["dissipation"] = sum(d["dissipation"] for d in ds) / len(ds)
        out["umax"] = max(d["umax"] for d in ds)
        return out


def diffs(a, b):
    return {k: float(np.abs(x - y).max()) for k, x, y in zip(("rho", "u", "phi"), a, b) if x is not None}


def two_phase_cfg(shape, ratio):
    rho, u, phi = ragged_two_phase(shape, ratio)
    return dict(n=None, rho=rho, u=u, phi=phi,
                params=dict(tau=0.7, two_phase=1, rho_l=ratio, rho_g=1.0, sigma=0.01, mobility=0.05, width=4.0,
                            force_type=1, force_amp=1e-5, force_k=1))


@pytest.mark.parametrize("world", [1, 2, 3])
@pytest.mark.parametrize("shape,ratio", [((64, 32, 48), 10.0), ((40, 26, 36), 1.0)])
def test_two_phase_slabs_equal_the_undivided_box_and_the_oracle(acclb, shape, ratio, world):
    """Density ratio 10 (F^p, F^nu: the velocity of the halo plane h-1 enters the phi flux through the slab face) and 1; ABC
    forcing (its z table is cut out of the whole domain's); tile-divisible (TMA pull) and ragged boxes; a droplet that
    straddles the periodic corner, so it also straddles the slab faces."""
    cfg = two_phase_cfg(shape, ratio)
    dom = Domain(acclb, cfg, shape, world)
    ref = gpu_sim(acclb, cfg, shape=shape)
    o = cpu_sim(cfg, shape=shape)
    for t in (1, 5, 6):
        dom.step(t)
        ref.step(t)
        o.step(t)
        got = dom.moments()
        d = diffs(got, [x.cpu().numpy() if x is not None else None for x in ref.moments()])
        assert all(v <= SAME for v in d.values()), (t, d)
        d = diffs(got, o.moments())
        assert all(v <= TOL for v in d.values()), (t, d)
    dg, dr = dom.diagnostics(), ref.diagnostics()
    for k in ("sum_phi", "ke", "dissipation", "umax"):
        assert abs(dg[k] - dr[k]) <= 1e-12 * abs(dr[k]), (k, dg[k], dr[k])
    n = shape[0] * shape[1] * shape[2]
    for k in ("sum_pstar", "sum_mx", "sum_my", "sum_mz"):
        assert abs(dg[k] - dr[k]) <= 1e-13 * n, (k, dg[k], dr[k])


@pytest.mark.parametrize("fp32,variant", [(1, 0), (0, 1), (1, 1)])
def test_two_phase_slabs_fp32_storage_and_unfused_variant(acclb, fp32, variant):
    """The same exchange serves fp32 population storage (ranges of 4-byte elements) and the unfused kernel pair (variant 1:
    u and r through HBM, k_advect reads u of the halo plane h-1): three slabs equal the undivided box run the same way."""
    shape = (64, 32, 48)
    cfg = two_phase_cfg(shape, 10.0)
    dom = Domain(acclb, cfg, shape, 3, store_fp32=fp32)
    ref = gpu_sim(acclb, cfg, shape=shape, store_fp32=fp32)
    for p in dom.parts:
        p.sim.set_variant(variant)
    ref.set_variant(variant)
    dom.step(12)
    ref.step(12)
    d = diffs(dom.moments(), [x.cpu().numpy() for x in ref.moments()])
    assert all(v <= (1e-9 if fp32 else SAME) for v in d.values()), d   # fp32: the seam-order noise is rounded to float steps
    if not fp32:
        o = cpu_sim(cfg, shape=shape)
        o.step(12)
        d = diffs(dom.moments(), o.moments())
        assert all(v <= TOL for v in d.values()), d


@pytest.mark.parametrize("fp32", [0, 1])
@pytest.mark.parametrize("world", [1, 2, 4])
def test_single_phase_slabs_equal_the_undivided_box(acclb, world, fp32):
    """Single component: one halo plane, nine populations per side and step; forced turbulence (sine forcing along z too).
    The one-node-per-thread kernel is deterministic: the slab run is bit-identical to the undivided one."""
    cfg = wl.make_config("hit", n=32)
    cfg["params"].update(force_type=1, force_amp=2e-5)
    shape = (32, 32, 32)
    dom = Domain(acclb, cfg, shape, world, store_fp32=fp32)
    ref = gpu_sim(acclb, cfg, store_fp32=fp32)
    dom.step(20)
    ref.step(20)
    got = dom.moments()
    want = [x.cpu().numpy() if x is not None else None for x in ref.moments()]
    assert np.array_equal(got[0], want[0]) and np.array_equal(got[1], want[1])
    if not fp32:
        o = cpu_sim(cfg)
        o.step(20)
        d = diffs(got, o.moments())
        assert all(v <= TOL for v in d.values()), d
    assert dom.parts[0].halo_bytes_per_step() == 2 * 9 * 32 * 32 * (4 if fp32 else 8)


def test_minimal_and_full_halo_agree_and_sum_phi_is_conserved_over_a_long_run(acclb):
    """The minimal exchange leaves parts of the halo planes as scratch; after 400 steps of bubble-laden forced turbulence on
    four slabs the own planes still equal those of a run that refreshes every population of every halo plane, and the
    whole domain's sum of phi (the fluxes through the slab faces are evaluated on both sides) is conserved to rounding."""
    cfg = wl.make_config("bubbly", n=64, void_fraction=0.03)
    shape = (64, 64, 64)
    a = Domain(acclb, cfg, shape, 4)
    b = Domain(acclb, cfg, shape, 4, full_halo=True)
    s0 = a.diagnostics()
    a.step(400)
    b.step(400)
    d = diffs(a.moments(), b.moments())
    assert all(v <= 1e-11 for v in d.values()), d
    s1 = a.diagnostics()
    assert abs(s1["sum_phi"] - s0["sum_phi"]) <= 1e-12 * s0["sum_phi"]
    assert abs(s1["sum_pstar"] - s0["sum_pstar"]) <= 1e-12 * s0["sum_pstar"]
    plane = 64 * 64 * 8
    assert a.parts[0].halo_bytes_per_step() == 2 * (27 + 3) * plane and b.parts[0].halo_bytes_per_step() == 2 * (81 + 3) * plane
    for p in a.parts:
        r, u, ph = p.sim.moments()  # halo planes included: the scratch parts stay finite
        assert bool(torch.isfinite(r).all()) and bool(torch.isfinite(u).all()) and bool(torch.isfinite(ph).all())


def test_halo_chunks_layout_and_errors(acclb):
    """Ranges: inside the workspace, send / receive lists of equal lengths, byte counts as include/acclb.h states; a
    periodic context has none; invalid slab parameters are refused."""
    nx, ny, nzg = 32, 16, 24
    s = slabs.SlabAccLB(nx, ny, nzg, tau=0.8, two_phase=1, rho_l=1.0, rho_g=1.0, sigma=0.01, mobility=0.05, width=4.0)
    plane = nx * ny * 8
    ch = s.sim.halo_chunks()
    for side in (-1, 1):
        for d in (0, 1):
            sizes = [v.numel() for v, sd, dd in ch if sd == side and dd == d]
            assert sizes == [18 * plane, 9 * plane, 3 * plane], (side, d, sizes)
    full = s.sim.halo_chunks(full=True)
    assert sorted(v.numel() for v, _, _ in full) == sorted([81 * plane, 3 * plane] * 4)
    # no two receive ranges overlap, and no receive range overlaps a send range
    spans = sorted((v.data_ptr(), v.data_ptr() + v.numel(), d) for v, _, d in ch)
    for (a0, a1, da), (b0, b1, db) in zip(spans, spans[1:]):
        assert a1 <= b0 or (da == 0 and db == 0)
    periodic = acclb.AccLB(nx, ny, nzg, tau=0.8)
    with pytest.raises(acclb.AccLBError):
        periodic.halo_chunks()
    for bad in (dict(halo_z=2, two_phase=1, rho_l=1.0, rho_g=1.0, width=4.0, nz_global=64),   # two-phase needs 3
                dict(halo_z=1, nz_global=8),                                                  # nz_global < own planes
                dict(halo_z=1, nz_global=64, moment_storage=1),
                dict(halo_z=3, two_phase=1, rho_l=1.0, rho_g=1.0, width=4.0, nz_global=64, phi_rk3=1),
                dict(halo_z=-1)):
        with pytest.raises(acclb.AccLBError):
            acclb.AccLB(nx, ny, nzg, tau=0.8, **bad)
