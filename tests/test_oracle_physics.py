"""Physics pins for the CPU oracle: closed forms and exact invariants of whole steps (P4, P6-P9, P11-P14).

Each test states the mathematical fact it leans on; tolerances are the ones DESIGN.md section 4 derives.  CPU only.
"""
import numpy as np
import pytest

import oracle
from paper_2505_01126_b200 import workloads as wl

import naive_numpy as nv

CS2 = 1.0 / 3.0


def run(cfg, steps, shape=None):
    n = cfg["n"]
    nx, ny, nz = shape or (n, n, n)
    o = oracle.Oracle(nx, ny, nz, **cfg["params"])
    o.init(cfg["rho"], cfg["u"], cfg["phi"])
    o.step(steps)
    return o


# ------------------------------------------------------------------ P7: special cases of one step
def test_p7_uniform_state_is_fixed_point():
    n = 6
    o = oracle.Oracle(n, n, n, tau=0.7)
    rho = np.full((n, n, n), 1.3)
    u = np.zeros((3, n, n, n))
    u[0], u[1], u[2] = 0.03, -0.02, 0.05
    o.init(rho, u)
    f0 = o.populations()
    o.step(5)
    assert np.abs(o.populations() - f0).max() < 1e-15
    r, uu, _ = o.moments()
    assert np.abs(r - 1.3).max() < 1e-15 and np.abs(uu - u).max() < 1e-15


def test_p7_tau_one_gives_equilibrium_plus_half_force():
    """omega = 1: Eq. 6 reduces to f_i(x + c_i, t+1) = f_i^eq + S_i/2, whatever the incoming non-equilibrium."""
    rng = np.random.default_rng(7)
    nx, ny, nz = 5, 6, 7
    p = dict(tau=1.0, force_type=1, force_amp=1e-3, force_k=1)
    o = oracle.Oracle(nx, ny, nz, **p)
    _, w = oracle.lattice()
    f = w[:, None, None, None] * (1 + 0.05 * rng.standard_normal((27, nz, ny, nx)))
    o.set_populations(f)
    pst, u, _ = o.moments()
    A = o.accel()
    o.step(1)
    f1 = o.populations()
    c, _ = oracle.lattice()
    for i in (0, 5, 13, 14, 22, 26):
        for (x, y, z) in [(0, 0, 0), (4, 5, 6), (2, 3, 1)]:
            xs, ys, zs = (x - c[i][0]) % nx, (y - c[i][1]) % ny, (z - c[i][2]) % nz
            ref = oracle.feq(pst[zs, ys, xs], u[:, zs, ys, xs])[i] + 0.5 * oracle.guo(u[:, zs, ys, xs], A[:, zs, ys, xs])[i]
            assert abs(f1[i, z, y, x] - ref) < 1e-16


# ------------------------------------------------------------------ P13: brute-force second evaluation
@pytest.mark.parametrize("two_phase,ratio", [(0, 1.0), (1, 1.0), (1, 10.0)])
def test_p13_oracle_equals_naive_collide_push(two_phase, ratio):
    """Pull/two-pass oracle (Eq. 6) == collide-at-node BGK on Hermite-projected populations + push (Eq. 4),
    on an anisotropic box (8 x 10 x 12) so that any axis or sign mix-up shows."""
    rng = np.random.default_rng(13)
    nx, ny, nz = 8, 10, 12
    p = dict(tau=0.6, two_phase=two_phase, rho_l=ratio, rho_g=1.0, sigma=0.01, mobility=0.05, width=4.0,
             force_type=1, force_amp=1e-4, force_k=1)
    Z, Y, X = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    rho = 1.0 + 0.01 * rng.standard_normal((nz, ny, nx))
    u = 0.02 * rng.standard_normal((3, nz, ny, nx))
    r = np.sqrt((X - 3.3) ** 2 + (Y - 4.1) ** 2 + (Z - 5.7) ** 2)
    phi = 0.5 * (1 + np.tanh(2 * (3.0 - r) / 4.0)) if two_phase else None
    o = oracle.Oracle(nx, ny, nz, **p)
    o.init(rho, u, phi)
    f = nv.init(rho, u, phi, p)
    assert np.abs(o.populations() - f).max() < 1e-15
    ph = phi
    for _ in range(3):
        f, ph = nv.step(f, ph, p)
    o.step(3)
    assert np.abs(o.populations() - f).max() < 1e-14
    r_o, u_o, phi_o = o.moments()
    r_n, u_n, *_ = nv.moments(f, ph, p)
    assert np.abs(r_o - r_n).max() < 1e-14 and np.abs(u_o - u_n).max() < 1e-14
    if two_phase:
        assert np.abs(phi_o - ph).max() < 1e-14


# ------------------------------------------------------------------ forcing closed forms (Eq. 5, R3, R4)
def test_uniform_acceleration_is_exact():
    """ABC forcing with k_f = 0 is the uniform force A(1,1,1): a uniform fluid accelerates as u(t) = u0 + A t with
    no error term (pins sum_i S_i c_i = A and the half-force in u, R4)."""
    n = 4
    o = oracle.Oracle(n, n, n, tau=0.9, force_type=1, force_amp=1e-4, force_k=0)
    u0 = np.zeros((3, n, n, n))
    u0[0] = 0.01
    o.init(np.ones((n, n, n)), u0)
    for t in (0, 1, 7):
        _, u, _ = o.moments()
        assert np.abs(u[0] - (0.01 + 1e-4 * t)).max() < 1e-15
        assert np.abs(u[1] - 1e-4 * t).max() < 1e-15
        o.step(1 if t == 0 else 6)


def test_kolmogorov_flow_steady_state():
    """F_x = F0 sin(k y): steady Stokes solution u_x = F0 sin(k y) / (nu k^2), nu = cs2 (tau - 1/2).
    Sine forcing (type 2) drives three such decoupled shear flows; amplitude is kept tiny so u.grad u ~ 1e-14."""
    n, tau, F0 = 16, 1.0, 1e-9
    nu = CS2 * (tau - 0.5)
    k = 2 * np.pi / n
    o = oracle.Oracle(n, n, n, tau=tau, force_type=2, force_amp=F0, force_k=1)
    o.init(np.ones((n, n, n)), np.zeros((3, n, n, n)))
    o.step(int(12 / (nu * k * k)))          # e^-12 of the transient left
    _, u, _ = o.moments()
    y = np.arange(n)
    expect = F0 * np.sin(k * y) / (nu * k * k)
    got = u[0][0, :, 0]
    assert np.abs(got - expect).max() / np.abs(expect).max() < 0.015   # O(k^2) lattice correction, k^2/12 = 1.3 %
    assert np.abs(u[0] - got[None, :, None]).max() < 1e-5 * np.abs(expect).max()   # u_x depends on y only (u.grad u ~ 1e-14)


# ------------------------------------------------------------------ P6 / P14: Taylor-Green vortex (config 1)
@pytest.fixture(scope="module")
def tgv_history():
    cfg = wl.make_config("tgv")
    o = oracle.Oracle(32, 32, 32, **cfg["params"])
    o.init(cfg["rho"], cfg["u"])
    hist = [o.diagnostics()]
    for _ in range(10):
        o.step(10)
        hist.append(o.diagnostics())
    return o, hist


def test_p6_tgv_energy_decay_rate(tgv_history):
    """E(t) = E(0) exp(-2 nu k^2 t), k^2 = 3 (2 pi / 32)^2, nu = (0.8 - 0.5)/3 = 0.1 (Stokes limit, Re ~ 1)."""
    _, hist = tgv_history
    nu, k2 = 0.1, 3 * (2 * np.pi / 32) ** 2
    t = np.array([h["step"] for h in hist])
    E = np.array([h["ke"] for h in hist])
    assert abs(E[0] - 0.02 ** 2 / 8) < 1e-18          # <|u|^2>/2 of the TGV field = U0^2 / 8
    sel = t >= 20                                      # skip the equilibrium-initialisation transient (R15)
    rate = -np.polyfit(t[sel], np.log(E[sel]), 1)[0]
    assert abs(rate / (2 * nu * k2) - 1) < 0.01
    assert abs(E[-1] / E[0] / np.exp(-2 * nu * k2 * 100) - 1) < 0.03


def test_p6_dissipation_diagnostic_is_minus_dEdt(tgv_history):
    """R21: eps = nu a:a / (2 cs4 tau^2) equals 2 nu k^2 E on the decaying vortex (uses a = -cs2 tau (du+du^T), L94)."""
    _, hist = tgv_history
    nu, k2 = 0.1, 3 * (2 * np.pi / 32) ** 2
    for h in hist[3:]:
        assert abs(h["dissipation"] / (2 * nu * k2 * h["ke"]) - 1) < 0.02


def test_p14_hermite_coefficient_is_strain(tgv_history):
    """a_ab = -cs2 tau (d_a u_b + d_b u_a) + O(Ma^3), gradient by the lattice stencil."""
    o, _ = tgv_history
    _, u, _ = o.moments()
    a = o.hermite()
    du = np.stack([oracle.gradient(u[b]) for b in range(3)], axis=1)   # du[a, b] = d_a u_b
    idx = [(0, 0), (1, 1), (2, 2), (0, 1), (0, 2), (1, 2)]
    scale = CS2 * 0.8 * np.abs(du).max()
    for j, (al, be) in enumerate(idx):
        expect = -CS2 * 0.8 * (du[al, be] + du[be, al])
        assert np.abs(a[j] - expect).max() < 0.05 * scale


def test_p4_tgv_mass_and_momentum(tgv_history):
    _, hist = tgv_history
    assert abs(hist[-1]["sum_pstar"] / hist[0]["sum_pstar"] - 1) < 1e-12
    for k in ("sum_mx", "sum_my", "sum_mz"):
        assert abs(hist[-1][k] - hist[0][k]) < 1e-12


# ------------------------------------------------------------------ P4: conservation under forcing, turbulent-like field
def test_p4_forced_hit_conserves_mass_and_momentum():
    cfg = wl.make_config("hit", n=16)
    o = run(cfg, 0)
    d0 = o.diagnostics()
    o.step(60)
    d1 = o.diagnostics()
    assert abs(d1["sum_pstar"] / d0["sum_pstar"] - 1) < 1e-12
    for k in ("sum_mx", "sum_my", "sum_mz"):          # sum_x F^b = 0 (R20) -> total momentum unchanged
        assert abs(d1[k] - d0[k]) < 1e-12
    assert np.isfinite(d1["ke"]) and d1["ke"] > 0


def test_p4_momentum_balance_two_phase():
    """sum_x m(t+1) - sum_x m(t) = sum_x F/rho(t): Guo forcing injects exactly A per node per step."""
    cfg = wl.make_config("droplet", n=16, density_ratio=10.0)
    cfg["params"].update(force_type=1, force_amp=1e-5)
    o = run(cfg, 3)
    d0 = o.diagnostics()
    A = o.accel()
    o.step(1)
    d1 = o.diagnostics()
    for al, k in enumerate(("sum_mx", "sum_my", "sum_mz")):
        assert abs((d1[k] - d0[k]) - A[al].sum()) < 1e-13
    assert abs(d1["sum_pstar"] - d0["sum_pstar"]) < 1e-12 * 16 ** 3   # zero-gauge run: absolute (R26)


# ------------------------------------------------------------------ P8 / P9: Allen-Cahn
def test_p8_total_phi_conserved_under_advection():
    cfg = wl.make_config("bubbly", n=24)
    cfg["phi"] = wl.droplet_phi(24, 6.0)
    o = run(cfg, 0)
    s0 = o.diagnostics()["sum_phi"]
    o.step(40)
    d = o.diagnostics()
    assert abs(d["sum_phi"] / s0 - 1) < 1e-12
    _, _, phi = o.moments()
    assert phi.min() > -0.02 and phi.max() < 1.05            # boundedness sanity (R = 6 is barely resolved)


def test_p9_flat_interface_relaxes_to_tanh_profile():
    """Steady 1-D solution of Eq. 3 with kappa = 4D/delta: D phi' = kappa phi (1 - phi)  ->
    phi = (1 + tanh(2 xi / delta)) / 2 (R10).  Start from a too-sharp slab and let it relax."""
    nx, ny, nz, W = 64, 4, 4, 4.0
    x = np.arange(nx) - (nx - 1) / 2
    prof = lambda w: 0.5 * (np.tanh(2 * (x + 16) / w) - np.tanh(2 * (x - 16) / w))
    phi = np.broadcast_to(prof(2.0), (nz, ny, nx)).copy()
    p = dict(tau=0.8, two_phase=1, rho_l=1.0, rho_g=1.0, sigma=0.0, mobility=0.05, width=W)
    o = oracle.Oracle(nx, ny, nz, **p)
    o.init(np.ones((nz, ny, nx)), np.zeros((3, nz, ny, nx)), phi)
    s0 = o.diagnostics()["sum_phi"]
    o.step(4000)
    _, u, ph = o.moments()
    assert abs(o.diagnostics()["sum_phi"] / s0 - 1) < 1e-12
    # conserved sum fixes the slab half-width; compare against the closed form with that half-width
    half = ph[0, 0].sum() / 2
    expect = 0.5 * (np.tanh(2 * (x + half) / W) - np.tanh(2 * (x - half) / W))
    assert np.abs(ph[0, 0] - expect).max() < 1e-2
    assert np.abs(ph - ph[0:1, 0:1]).max() < 1e-14      # stays one-dimensional
    assert np.abs(u).max() < 1e-12                        # sigma = 0, equal densities: no flow


# ------------------------------------------------------------------ P11: Laplace law
def laplace_ratio(o, n2d_or_3d, R_eff, sigma, rho_l, rho_g, centre, far):
    r, _, phi = o.moments()
    rho = rho_g + (rho_l - rho_g) * phi
    p = CS2 * rho * r                                   # p = p* rho cs2
    dp = p[centre] - p[far]
    return dp / (n2d_or_3d * sigma / R_eff)


def test_p11_laplace_cylinder():
    """z-invariant droplet (nz = 1): Delta p = sigma / R.  Pins the 3 delta / 2 normalisation and the sign of F^s (R8)."""
    n, R, sigma = 64, 16.0, 0.01
    ax = np.arange(n) - (n - 1) / 2
    Y, X = np.meshgrid(ax, ax, indexing="ij")
    phi = (0.5 * (1 + np.tanh(2 * (R - np.sqrt(X * X + Y * Y)) / 4.0)))[None]
    p = dict(tau=0.8, two_phase=1, rho_l=1.0, rho_g=1.0, sigma=sigma, mobility=0.05, width=4.0)
    o = oracle.Oracle(n, n, 1, **p)
    o.init(np.ones((1, n, n)), np.zeros((3, 1, n, n)), phi)
    ratios = []
    for _ in range(10):
        o.step(300)
        R_eff = np.sqrt(o.diagnostics()["sum_phi"] / np.pi)
        ratios.append(laplace_ratio(o, 1.0, R_eff, sigma, 1.0, 1.0, (0, n // 2, n // 2), (0, 0, 0)))
    assert abs(np.mean(ratios[4:]) - 1) < 0.05, ratios
    assert o.diagnostics()["umax"] < 1e-4               # spurious currents


@pytest.mark.parametrize("ratio,gauge", [(1.0, 1.0), (10.0, 0.0)])
def test_p11_laplace_sphere(ratio, gauge):
    """3-D droplet: Delta p = 2 sigma / R_eff, R_eff = (3 sum phi / 4 pi)^(1/3); density ratio 10 uses zero gauge
    pressure (R26) and exercises A = F/rho (R3), F^p and F^nu (R9)."""
    n, R, sigma = 32, 9.0, 0.01
    cfg = wl.make_config("droplet", n=n, density_ratio=ratio)
    cfg["phi"] = wl.droplet_phi(n, R)
    o = run(cfg, 0)
    ratios = []
    for _ in range(8):
        o.step(100)
        R_eff = (3 * o.diagnostics()["sum_phi"] / (4 * np.pi)) ** (1 / 3)
        ratios.append(laplace_ratio(o, 2.0, R_eff, sigma, ratio, 1.0, (n // 2,) * 3, (0, 0, 0)))
    assert abs(np.mean(ratios[3:]) - 1) < 0.10, ratios
    assert o.diagnostics()["umax"] < 2e-4


# ------------------------------------------------------------------ P12: lattice symmetries
def _two_phase_case(n=12, seed=12):
    rng = np.random.default_rng(seed)
    ax = np.arange(n)
    Z, Y, X = np.meshgrid(ax, ax, ax, indexing="ij")
    r = np.sqrt((X - 4.0) ** 2 + (Y - 6.5) ** 2 + (Z - 5.0) ** 2)
    phi = 0.5 * (1 + np.tanh(2 * (3.5 - r) / 4.0))
    u = 0.02 * rng.standard_normal((3, n, n, n))
    rho = 1 + 0.01 * rng.standard_normal((n, n, n))
    p = dict(tau=0.55, two_phase=1, rho_l=3.0, rho_g=1.0, sigma=0.01, mobility=0.05, width=4.0)
    return p, rho, u, phi


def _advance(p, rho, u, phi, steps=4):
    n = rho.shape[0]
    o = oracle.Oracle(n, n, n, **p)
    o.init(rho, u, phi)
    o.step(steps)
    return o.moments()


def test_p12_periodic_shift_is_bitwise():
    p, rho, u, phi = _two_phase_case()
    base = _advance(p, rho, u, phi)
    sh = dict(shift=(5, -3, 7), axis=(-3, -2, -1))
    moved = _advance(p, np.roll(rho, **sh), np.roll(u, **sh), np.roll(phi, **sh))
    for b, m in zip(base, moved):
        assert np.array_equal(np.roll(b, **sh), m)


def test_p12_axis_permutation_and_reflection():
    """x->y->z->x relabelling and the mirror x -> -x map solutions to solutions (no body force)."""
    p, rho, u, phi = _two_phase_case()
    r0, u0, f0 = _advance(p, rho, u, phi)
    # cyclic permutation: new field g(z,y,x) = old(y,x,z)  <=> transpose axes; vector components permute alike
    perm = (1, 2, 0)                                  # new axes (z',y',x') take old axes (y,x,z)
    tp = lambda s: np.transpose(s, perm)
    # old comps (ux,uy,uz) live on axes (2,1,0); after the transpose old axis y -> z', x -> y', z -> x'
    u_new = np.stack([tp(u[2]), tp(u[0]), tp(u[1])])  # (ux', uy', uz') = (uz, ux, uy)
    r1, u1, f1 = _advance(p, tp(rho), u_new, tp(phi))
    assert np.abs(tp(r0) - r1).max() < 1e-13 and np.abs(tp(f0) - f1).max() < 1e-13
    assert np.abs(np.stack([tp(u0[2]), tp(u0[0]), tp(u0[1])]) - u1).max() < 1e-13
    # reflection in x
    fl = lambda s: s[..., ::-1]
    u_ref = np.stack([-fl(u[0]), fl(u[1]), fl(u[2])])
    r2, u2, f2 = _advance(p, fl(rho), u_ref, fl(phi))
    assert np.abs(fl(r0) - r2).max() < 1e-13 and np.abs(fl(f0) - f2).max() < 1e-13
    assert np.abs(np.stack([-fl(u0[0]), fl(u0[1]), fl(u0[2])]) - u2).max() < 1e-13


# ------------------------------------------------------------------ sub-box evaluation used by the full-size GPU parity test
@pytest.mark.parametrize("rk3,n,s,k", [(0, 24, 18, 2), (1, 32, 28, 1)])
def test_subbox_evaluation_matches_full_box_interior(rk3, n, s, k):
    """k steps only depend on inputs within radius 3k (two-phase, forward Euler) of a node, 9k with the three-stage
    Runge-Kutta integrator of phi (each stage reaches 3 further, R32): running the oracle on a periodic sub-box reproduces
    the full-box values away from the sub-box rim."""
    cfg = wl.make_config("bubbly", n=n)
    cfg["params"]["phi_rk3"] = rk3
    cfg["phi"] = wl.bubbles_phi(n, np.array([[9.0, 10.0, 11.0]]), radius=5.0)
    full = run(cfg, k).moments()
    org = (n - 4, 3, n - 9)                             # wraps across the periodic boundary in x
    sub = oracle.Oracle(s, s, s, **cfg["params"], force_period=(n, n, n), force_origin=org)
    sub.init(wl.subbox(cfg["rho"], org, s), wl.subbox(cfg["u"], org, s), wl.subbox(cfg["phi"], org, s))
    sub.step(k)
    got = sub.moments()
    rim = (9 if rk3 else 3) * k + 2
    inner = (slice(rim, s - rim),) * 3
    for a, b in zip(full, got):
        assert np.abs(wl.subbox(a, org, s)[..., inner[0], inner[1], inner[2]] - b[..., inner[0], inner[1], inner[2]]).max() < 1e-15


# ------------------------------------------------------------------ advection of phi: direction, upwinding, order (Eq. 3, R12)
def _circular_com(phi):
    """Centre of mass of a periodic blob per axis (x, y, z) through the first Fourier mode (exact for a symmetric blob)."""
    out = []
    for ax in (2, 1, 0):
        n = phi.shape[ax]
        prof = phi.sum(axis=tuple(a for a in range(3) if a != ax))
        th = 2 * np.pi * np.arange(n) / n
        out.append(np.arctan2((prof * np.sin(th)).sum(), (prof * np.cos(th)).sum()) * n / (2 * np.pi))
    return np.array(out)


def test_phi_blob_translates_with_plus_u():
    """PAPER.md:L61 (Eq. 3): d_t phi + u.grad phi = ... moves phi WITH +u.  A tanh blob (R = 7, W = 4) in a uniform flow
    u = (0.05, -0.02, 0.03) with sigma = 0 and equal densities (uniform flow is then an exact fixed point of the LB part)
    must have its centre of mass displaced by u t after t = 100 steps (within 1 % of the smallest component) and stay
    bounded; also catches a face flux differenced along the wrong axis."""
    n, R, t = 32, 7.0, 100
    uvec = np.array([0.05, -0.02, 0.03])
    p = dict(tau=0.8, two_phase=1, rho_l=1.0, rho_g=1.0, sigma=0.0, mobility=0.05, width=4.0)
    phi0 = wl.droplet_phi(n, R)
    u0 = np.empty((3, n, n, n))
    for al in range(3):
        u0[al] = uvec[al]
    o = oracle.Oracle(n, n, n, **p)
    o.init(np.ones((n, n, n)), u0, phi0)
    c0 = _circular_com(phi0)
    o.step(t)
    _, u, phi = o.moments()
    assert np.abs(u - u0).max() < 1e-13                        # the carrier flow stays uniform
    shift = (_circular_com(phi) - c0 + n / 2) % n - n / 2
    assert np.abs(shift - uvec * t).max() < 0.01 * np.abs(uvec * t).min(), (shift, uvec * t)
    assert phi.min() > -1e-3 and phi.max() < 1 + 1e-3
    assert abs(o.diagnostics()["sum_phi"] / phi0.sum() - 1) < 1e-12


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("sign", [+1.0, -1.0])
def test_phi_advection_one_step_is_minus_u_dphi_at_fifth_order(axis, sign):
    """With D = 0 (mobility = 0 is legal: kappa = 4D/delta = 0) one forward-Euler step of Eq. 3 in a uniform flow is
    phi(t+1) - phi(t) = -u d_a phi, the flux difference of the finite-difference WENO5 reconstruction (PAPER.md:L67,
    R12), which approximates the derivative of a smooth profile to fifth order: error / k ~ k^5.  Pins the SIGN of the
    advective term, the axis each face flux belongs to, and the order (wrong candidate / weight constants give 3), for
    both upwind stencils.  (A multi-step refinement study cannot show more than first order: the integrator is
    forward Euler, R13.)"""
    errs = []
    uval = sign * 0.04
    for n in (16, 32, 64):
        shape = [4, 4, 4]
        shape[2 - axis] = n                                   # arrays are [z][y][x]; axis 0 = x
        nz, ny, nx = shape
        k = 2 * np.pi / n
        coord = np.arange(n, dtype=float)
        prof = 0.5 + 0.3 * np.sin(k * coord + 0.4)
        bshape = [1, 1, 1]
        bshape[2 - axis] = n
        phi0 = np.ascontiguousarray(np.broadcast_to(prof.reshape(bshape), shape))
        u0 = np.zeros((3, nz, ny, nx))
        u0[axis] = uval
        p = dict(tau=0.8, two_phase=1, rho_l=1.0, rho_g=1.0, sigma=0.0, mobility=0.0, width=4.0)
        o = oracle.Oracle(nx, ny, nz, **p)
        o.init(np.ones(shape), u0, phi0)
        o.step(1)
        _, _, phi1 = o.moments()
        dphi = ((phi1 - phi0) / (-uval)).reshape(-1, n) if axis == 0 else np.moveaxis((phi1 - phi0) / (-uval), 2 - axis, -1).reshape(-1, n)
        exact = 0.3 * k * np.cos(k * coord + 0.4)
        errs.append(np.abs(dphi - exact[None, :]).mean() / k)  # L1: WENO-JS drops to third order AT critical points only
    o1, o2 = np.log2(errs[0] / errs[1]), np.log2(errs[1] / errs[2])
    assert errs[0] < 2e-3 and o1 > 4.0 and o2 > 4.0, (errs, o1, o2)


def test_phi_advection_is_upwind_biased():
    """R12: the face value is reconstructed from the UPWIND side (`uf >= 0` takes cells x-2..x+2 for the face x+1/2).
    On a marginally resolved wave (4 points per wavelength, D = 0) the upwind-biased fifth-order stencil is dissipative,
    the downwind-biased one (the flipped test) amplifies: after 40 steps at |u| = 0.05 the L2 norm of the fluctuation
    has decreased, for both signs of u."""
    n = 32
    x = np.arange(n, dtype=float)
    prof = 0.5 + 0.05 * np.sin(2 * np.pi * x / 4)
    shape = (4, 4, n)
    phi0 = np.ascontiguousarray(np.broadcast_to(prof, shape))
    p = dict(tau=0.8, two_phase=1, rho_l=1.0, rho_g=1.0, sigma=0.0, mobility=0.0, width=4.0)
    for uval in (0.05, -0.05):
        u0 = np.zeros((3,) + shape)
        u0[0] = uval
        o = oracle.Oracle(n, 4, 4, **p)
        o.init(np.ones(shape), u0, phi0)
        o.step(40)
        _, _, phi = o.moments()
        amp0, amp1 = np.linalg.norm(phi0 - 0.5), np.linalg.norm(phi - 0.5)
        assert 0.5 * amp0 < amp1 < 0.995 * amp0, (uval, amp0, amp1)


# ------------------------------------------------------------------ F^nu on a prescribed shear (PAPER.md:L104 read as R9, L94)
@pytest.mark.parametrize("pstar", [0.0, 1.0])
def test_viscous_correction_force_on_prescribed_shear(pstar):
    """Populations are prescribed in second-order Hermite space, f_i = f_i^eq(p*, m) + w_i H_i:a / (2 cs4) with
    a = -cs2 tau (d_a u_b + d_b u_a) of a known smooth velocity m, rho(phi) a smooth wave, sigma = 0,
    no body force.  By the moment identities of P2/P3, sum_i f_i c c = p* cs2 I + m m + a, so R9's force is
      F^nu_a = -((tau-1/2)/tau) [a_ab + m_a m_b - ut_a ut_b] d_b rho,  ut = m + F^p/(2 rho),  F^p = -p* cs2 grad rho,
    and for p* = 0 (no F^p) it reduces to  nu (d_a u_b + d_b u_a) d_b rho  exactly -- the reduction SURVEY R9 quotes.
    The oracle's stored acceleration A = (F^p + F^nu)/rho is compared with this closed form; grad rho uses the lattice
    stencil's plane-wave symbol (P5).  A wrong contraction index, prefactor, sign, or a dropped p* cs2 delta term fails."""
    n, tau, rl, rg = 12, 0.9, 10.0, 1.0
    nu = CS2 * (tau - 0.5)
    c, w = oracle.lattice()
    k = 2 * np.pi / n
    ax = np.arange(n, dtype=float)
    Z, Y, X = np.meshgrid(ax, ax, ax, indexing="ij")
    amp = np.array([[0.0, 0.011, -0.007], [0.013, 0.0, 0.005], [-0.009, 0.006, 0.0]])   # amp[b][a]: u_b += amp sin(k x_a + ..)
    diag = np.array([0.004, -0.008, 0.003])
    pos = (X, Y, Z)
    m = np.zeros((3, n, n, n))
    du = np.zeros((3, 3, n, n, n))                    # du[a][b] = d_a u_b
    for b in range(3):
        for a in range(3):
            coef = diag[b] if a == b else amp[b][a]
            ph = k * pos[a] + 0.3 * (a + 1) + 0.5 * b
            m[b] += coef * np.sin(ph)
            du[a][b] += coef * k * np.cos(ph)
    a_t = -CS2 * tau * (du + np.transpose(du, (1, 0, 2, 3, 4)))
    kv = k * np.array([1, 2, -1])
    phase = kv[0] * X + kv[1] * Y + kv[2] * Z + 0.7
    phi = 0.5 + 0.25 * np.sin(phase)
    s3 = (2 + np.cos(kv)) / 3
    gphi = np.stack([np.sin(kv[al]) * np.prod(np.delete(s3, al)) * 0.25 * np.cos(phase) for al in range(3)])
    rho = rg + (rl - rg) * phi
    drho = (rl - rg) * gphi
    # populations in Hermite space (numpy, from the lattice table only)
    f = np.empty((27, n, n, n))
    for i in range(27):
        cu = sum(c[i][al] * m[al] for al in range(3))
        H = np.outer(c[i], c[i]) - CS2 * np.eye(3)
        huu = sum(H[al, be] * m[al] * m[be] for al in range(3) for be in range(3))
        ha = sum(H[al, be] * a_t[al][be] for al in range(3) for be in range(3))
        f[i] = w[i] * (pstar + cu / CS2 + huu / (2 * CS2 ** 2)) + w[i] * ha / (2 * CS2 ** 2)
    p = dict(tau=tau, two_phase=1, rho_l=rl, rho_g=rg, sigma=0.0, mobility=0.05, width=4.0)
    o = oracle.Oracle(n, n, n, **p)
    o.init(np.full((n, n, n), pstar), np.zeros((3, n, n, n)), phi)
    o.set_populations(f)
    o.moments()
    A = o.accel()
    Fp = -pstar * CS2 * drho
    ut = m + Fp / (2 * rho)
    expect = np.zeros((3, n, n, n))
    for al in range(3):
        for be in range(3):
            expect[al] += -((tau - 0.5) / tau) * (a_t[al][be] + m[al] * m[be] - ut[al] * ut[be]) * drho[be]
    expect = (expect + Fp) / rho
    assert np.abs(A - expect).max() < 1e-15 + 1e-13 * np.abs(expect).max(), np.abs(A - expect).max()
    if pstar == 0.0:                                   # the continuum form of SURVEY R9 / PAPER.md:L94
        visc = np.zeros((3, n, n, n))
        for al in range(3):
            for be in range(3):
                visc[al] += nu * (du[al][be] + du[be][al]) * drho[be]
        assert np.abs(A - visc / rho).max() < 1e-15 + 1e-13 * np.abs(visc / rho).max()
        assert np.abs(visc / rho).max() > 1e-4         # the force is really there
