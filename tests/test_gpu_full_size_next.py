"""The SURVEY 8(f) rows at BASELINE's full size, 512^3, in the launch configurations bench.py times (its two_phase_rk3,
single_phase_moment_storage and z_slab legs): every node of the interiors of ten 64^3 sample boxes against the oracle run on
that periodic sub-box (exact beyond a rim of 3 k + 2 nodes; 9 k + 2 with the three-stage integrator of phi:
tests/test_oracle_physics.py::test_subbox_evaluation_matches_full_box_interior), fp64 max|d| <= 1e-11, plus the conserved
sums.  Same sample boxes as tests/test_gpu_parity.py::test_full_size_512_sampled_against_oracle (they straddle every z-chunk
seam, the periodic wraps and bubble interfaces)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2505_01126_b200 import slabs, workloads as wl
from test_gpu_parity import TOL, full_size_config, gpu_sim, sample_origins

pytestmark = pytest.mark.gpu


def run_case(acclb, mode, cfg, k):
    """(rho, u, phi) of the whole 512^3 domain after k steps as numpy arrays, and the diagnostics before / after."""
    n = 512
    dev = torch.device("cuda", 0)
    if mode == "slab":   # ONE z-slab of 512 own planes + halos that is its own neighbour: the halo exchange after every step
        part = slabs.SlabAccLB(n, n, n, **cfg["params"])
        sl = part.slab
        part.init(torch.from_numpy(sl.take(cfg["rho"])).to(dev), torch.from_numpy(sl.take(cfg["u"], axis=1)).to(dev),
                  torch.from_numpy(sl.take(cfg["phi"])).to(dev))
        d0 = part.diagnostics()
        part.step(k)
        out = [t.cpu().numpy() for t in part.moments()]
        d1 = part.diagnostics()
        assert part.sim.launch_count >= 2 * k and sl.nz_local == n + 6
        part.close()
        return out, d0, d1
    sim = gpu_sim(acclb, cfg, moment_storage=1) if mode == "moment" else gpu_sim(acclb, cfg)
    d0 = sim.diagnostics()
    sim.step(k)
    out = [t.cpu().numpy() if t is not None else None for t in sim.moments()]
    d1 = sim.diagnostics()
    sim.close()
    return out, d0, d1


@pytest.mark.parametrize("mode", ["rk3", "moment", "slab"])
def test_next_rows_full_size_512_sampled_against_oracle(acclb, mode):
    free, _ = torch.cuda.mem_get_info()
    if free < 90e9:
        pytest.skip("needs about 80 GB of free device memory")
    n, s = 512, 64
    base = full_size_config("hit" if mode == "moment" else "bubbly")
    cfg = dict(base, params=dict(base["params"]))
    if mode == "rk3":
        cfg["params"]["phi_rk3"] = 1
    k = 2 if mode == "rk3" else 5
    rim = (9 if mode == "rk3" else 3) * k + 2
    two_phase = cfg["phi"] is not None
    (rho, u, phi), d0, d1 = run_case(acclb, mode, cfg, k)
    assert d1["step"] == k
    assert abs(d1["sum_pstar"] - d0["sum_pstar"]) <= 1e-12 * n ** 3
    if two_phase:
        assert abs(d1["sum_phi"] - d0["sum_phi"]) <= 1e-12 * d0["sum_phi"]
    inner = (slice(rim, s - rim),) * 3
    seen_interface = False
    for org in sample_origins(n, s, wl.bubble_centres(n, 60), seed=20250501):
        o = oracle.Oracle(s, s, s, **cfg["params"], force_period=(n, n, n), force_origin=org)
        o.init(wl.subbox(cfg["rho"], org, s), wl.subbox(cfg["u"], org, s), wl.subbox(cfg["phi"], org, s) if two_phase else None)
        o.step(k)
        ro, uo, po = o.moments()
        o.close()
        for fld, a, b in (("rho", rho, ro), ("u", u, uo), ("phi", phi, po)):
            if a is None:
                continue
            ga, gb = wl.subbox(a, org, s)[..., inner[0], inner[1], inner[2]], b[..., inner[0], inner[1], inner[2]]
            assert np.abs(ga - gb).max() <= TOL, (mode, org, fld, np.abs(ga - gb).max())
        if two_phase:
            pin = po[inner]
            seen_interface |= bool(((pin > 0.1) & (pin < 0.9)).any())
    assert seen_interface or not two_phase, "no sampled box cut through an interface"
