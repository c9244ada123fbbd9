"""GPU-vs-oracle parity for SURVEY 8(f) #1 through the C ABI: buoyancy (R31), density contrast 100 at tau = 0.515
 and the SSP-RK3 integrator of phi (R32).  Same seeded inputs on both sides, fp64 max|d| <= 1e-11."""
import numpy as np
import pytest
import torch

import oracle
from paper_2505_01126_b200 import workloads as wl
from test_gpu_parity import TOL, assert_parity, cpu_sim, gpu_sim, ragged_two_phase

pytestmark = pytest.mark.gpu


def both(acclb, cfg, shape=None, **extra):
    """(GPU context, oracle) for the same config; the binding spells the integrator flag like the oracle does."""
    return gpu_sim(acclb, cfg, shape=shape, **extra), cpu_sim(cfg, shape=shape)


@pytest.mark.parametrize("rk3,variant", [(0, 0), (1, 0), (1, 1)])
@pytest.mark.parametrize("shape", [(64, 32, 24), (40, 26, 22)])
def test_buoyant_two_phase_density_ratio_100(acclb, shape, rk3, variant):
    """Density contrast 100, nu = 0.005 (tau = 0.515), zero gauge pressure, gravity along -z with the mean density as
    reference, ABC forcing, a droplet straddling the periodic corner: tile-divisible (TMA path) and ragged boxes, forward
    Euler and SSP-RK3 (variant 0: the stages run in the tiled kernel, the first one fused with the LB step; variant 1:
    u and r through HBM, k_geom_r + k_advect per stage).  F^p, F^nu, F^g and A = F / rho all carry weight here."""
    rho, u, phi = ragged_two_phase(shape, 100.0)
    dens = 1.0 + 99.0 * phi
    cfg = dict(n=None, rho=rho, u=0.2 * u, phi=phi,
               params=dict(tau=0.515, two_phase=1, rho_l=100.0, rho_g=1.0, sigma=0.01, mobility=0.05, width=4.0,
                           force_type=1, force_amp=1e-6, force_k=1, gravity=(0.0, 1e-7, -2e-6), rho_ref=float(dens.mean()),
                           phi_rk3=rk3))
    sim, o = both(acclb, cfg, shape=shape)
    sim.set_variant(variant)
    assert_parity(sim, o, what="t=0")
    for t in (1, 9, 10):
        sim.step(t)
        o.step(t)
        assert_parity(sim, o, what=f"after {t} more steps")
    dg, do = sim.diagnostics(), o.diagnostics()
    assert abs(dg["sum_phi"] - do["sum_phi"]) <= 1e-12 * do["sum_phi"]
    for k in ("sum_mx", "sum_my", "sum_mz"):
        assert abs(dg[k] - do[k]) <= 1e-11 * shape[0] * shape[1] * shape[2]


def test_buoyancy_single_phase(acclb):
    """rho == 1: the uniform acceleration (1 - rho_ref) g on top of a turbulent field with sine forcing."""
    cfg = wl.make_config("hit", n=32)
    cfg["params"].update(gravity=(1e-6, -2e-6, 3e-6), rho_ref=0.25)
    sim, o = both(acclb, cfg)
    sim.step(10)
    o.step(10)
    assert_parity(sim, o)


@pytest.mark.parametrize("fp32", [0, 1])
def test_rk3_bubbly_first_10_steps(acclb, fp32):
    """BASELINE config 4 scaled to 64^3 with the SSP-RK3 integrator: field parity after each of the first 10 steps (fp64),
    relative L2 <= 1e-5 with fp32 population storage; sum phi conserved over 200 steps."""
    cfg = wl.make_config("bubbly", n=64, void_fraction=0.03)
    cfg["params"].update(phi_rk3=1)
    sim, o = both(acclb, cfg, store_fp32=fp32)
    for t in range(10):
        sim.step(1)
        o.step(1)
        if not fp32:
            assert_parity(sim, o, what=f"t={t + 1}")
    if fp32:
        for a, b in zip(sim.moments(), o.moments()):
            a = a.cpu().numpy()
            assert np.linalg.norm(a - b) / np.linalg.norm(b) <= 1e-5
    d0 = sim.diagnostics()
    sim.step(190)
    d1 = sim.diagnostics()
    assert abs(d1["sum_phi"] - d0["sum_phi"]) <= 1e-12 * d0["sum_phi"]


def test_rk3_minimum_size_box(acclb):
    """The smallest box (4 x 4 x 4): every tile of the stage kernels wraps onto itself."""
    shape = (4, 4, 4)
    nx, ny, nz = shape
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    md = lambda i, c, n: np.minimum(np.abs(i - c), n - np.abs(i - c))
    r = np.sqrt(md(x, 1.0, nx) ** 2 + md(y, 1.5, ny) ** 2 + md(z, 0.5, nz) ** 2)
    phi = 0.5 * (1.0 + np.tanh(2.0 * (1.6 - r) / 4.0))
    X, Y, Z = 2 * np.pi * x / nx, 2 * np.pi * y / ny, 2 * np.pi * z / nz
    u = np.stack([0.02 * np.sin(Y) * np.cos(Z), 0.015 * np.sin(Z + X), -0.01 * np.cos(X) * np.sin(Y)])
    cfg = dict(n=None, rho=np.ones((nz, ny, nx)), u=np.ascontiguousarray(u), phi=np.ascontiguousarray(phi),
               params=dict(tau=0.7, two_phase=1, rho_l=3.0, rho_g=1.0, sigma=0.005, mobility=0.05, width=4.0, force_type=2,
                           force_amp=1e-5, force_k=1, phi_rk3=1))
    sim, o = both(acclb, cfg, shape=shape)
    sim.step(8)
    o.step(8)
    assert_parity(sim, o)
