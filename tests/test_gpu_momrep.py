"""GPU-vs-oracle parity of the moment-representation storage: the state is the ten
macroscopic fields (p*, u, a) per node, the step is a closed map on them.  The oracle IS this two-pass form, so the results
agree to rounding: fp64 max|d| <= 1e-11, conserved sums 1e-12, and the same as the population-storage path."""
import numpy as np
import pytest
import torch

from paper_2505_01126_b200 import workloads as wl
from test_gpu_parity import TOL, assert_parity, cpu_sim, crop, gpu_sim

pytestmark = pytest.mark.gpu


def test_momrep_tgv_100_steps(acclb):
    cfg = wl.make_config("tgv")
    sim, o = gpu_sim(acclb, cfg, moment_storage=1), cpu_sim(cfg)
    assert_parity(sim, o, what="t=0")
    sim.step(100)
    o.step(100)
    assert_parity(sim, o, what="t=100")
    dg, do = sim.diagnostics(), o.diagnostics()
    for k in ("ke", "dissipation"):
        assert abs(dg[k] - do[k]) <= 1e-11 * do[k], (k, dg[k], do[k])
    assert abs(dg["sum_pstar"] - do["sum_pstar"]) <= 1e-12 * 32 ** 3 and abs(dg["umax"] - do["umax"]) <= 1e-13


def test_momrep_forced_hit_first_10_steps_and_sums(acclb):
    """BASELINE config 2 at its stated size: parity after each of the first 10 steps, conserved sums over 1000 steps, and
    agreement with the population-storage path of this library."""
    n = 128
    cfg = wl.make_config("hit", n=n)
    sim, ref, o = gpu_sim(acclb, cfg, moment_storage=1), gpu_sim(acclb, cfg), cpu_sim(cfg)
    d0 = sim.diagnostics()
    for t in range(10):
        sim.step(1)
        o.step(1)
        assert_parity(sim, o, what=f"t={t + 1}")
    ref.step(10)
    for a, b in zip(sim.moments()[:2], ref.moments()[:2]):
        assert (a - b).abs().max().item() <= 1e-12
    sim.step(990)
    d1 = sim.diagnostics()
    assert d1["step"] == 1000 and abs(d1["sum_pstar"] - d0["sum_pstar"]) <= 1e-12 * n ** 3
    for k in ("sum_mx", "sum_my", "sum_mz"):
        assert abs(d1[k] - d0[k]) <= 1e-12 * n ** 3 * 0.03


@pytest.mark.parametrize("shape", [(44, 30, 18), (4, 4, 4), (34, 6, 70)])
def test_momrep_ragged_boxes_abc_forcing_and_gravity(acclb, shape):
    """Ragged, non-cubic and minimum-size boxes (tails in every direction, tiles that wrap onto themselves), ABC forcing
     and the uniform buoyancy acceleration (R31)."""
    nx, ny, nz = shape
    cfg = crop(wl.make_config("hit", n=max(48, 2 * ((max(shape) + 1) // 2))), shape)
    cfg["params"].update(force_type=1, force_amp=2e-5, force_k=2, tau=0.6, gravity=(1e-6, -2e-6, 3e-6), rho_ref=0.25)
    sim, o = gpu_sim(acclb, cfg, shape=shape, moment_storage=1), cpu_sim(cfg, shape=shape)
    sim.step(12)
    o.step(12)
    assert_parity(sim, o)
    dg, do = sim.diagnostics(), o.diagnostics()
    for k in ("sum_mx", "sum_my", "sum_mz", "sum_pstar"):
        assert abs(dg[k] - do[k]) <= 1e-11 * nx * ny * nz


def test_momrep_rejects_what_it_does_not_cover(acclb):
    with pytest.raises(acclb.AccLBError):
        acclb.AccLB(32, 32, 32, tau=0.8, two_phase=1, moment_storage=1)
    with pytest.raises(acclb.AccLBError):
        acclb.AccLB(32, 32, 32, tau=0.8, store_fp32=1, moment_storage=1)
