"""Seeded synthetic inputs shaped like the paper's workloads (numpy only).

This module holds NONE of the method's arithmetic: it only builds initial fields (p*, u, phi) and the
parameter dictionaries of the five BASELINE.json configs.  The same arrays are handed, bit-identical, to the
CPU oracle (by the tests / bench) and to the CUDA library.  Recipes are stated in DESIGN.md section 5; the paper's
own initial states and forcing constants are unpublished, so these inputs
stand in for them.

Layout: scalars [nz][ny][nx] (x fastest), vectors [3][nz][ny][nx] with component 0 = x.
"""
from __future__ import annotations

import numpy as np

try:  # threaded pocketfft; same transform as numpy.fft
    from scipy import fft as _fft
    _FFT_KW = {"workers": -1}
except Exception:  # pragma: no cover
    from numpy import fft as _fft
    _FFT_KW = {}

SEED_VELOCITY = 1126
SEED_BUBBLES = 2505


def tgv_fields(n=32, u0=0.02):
    """Config 1: Taylor-Green vortex, u = U0 (sin X cos Y cos Z, -cos X sin Y cos Z, 0), X = 2 pi i / n, and the
    matching pressure p* = 1 + (3 U0^2 / 16)(cos 2X + cos 2Y)(cos 2Z + 2)."""
    ax = 2.0 * np.pi * np.arange(n) / n
    Z, Y, X = np.meshgrid(ax, ax, ax, indexing="ij")
    u = np.zeros((3, n, n, n))
    u[0] = u0 * np.sin(X) * np.cos(Y) * np.cos(Z)
    u[1] = -u0 * np.cos(X) * np.sin(Y) * np.cos(Z)
    rho = 1.0 + (3.0 * u0 * u0 / 16.0) * (np.cos(2 * X) + np.cos(2 * Y)) * (np.cos(2 * Z) + 2.0)
    return rho, u


_VELOCITY_CACHE = {}


def hit_velocity(n, urms=0.03, seed=SEED_VELOCITY, k_peak=4.0):
    """Configs 2/4/5: seeded random solenoidal field with shell spectrum E(k) ~ k^4 exp(-2 (k/k_peak)^2),
    normalised to sqrt(<u.u>/3) = urms (R28).  The last field is kept (callers must not modify it): configs 2 and 4 of one size share it."""
    key = (n, urms, seed, k_peak)
    if key in _VELOCITY_CACHE:
        return _VELOCITY_CACHE[key]
    _VELOCITY_CACHE.clear()
    u = _hit_velocity(n, urms, seed, k_peak)
    _VELOCITY_CACHE[key] = u
    return u


def _hit_velocity(n, urms, seed, k_peak):
    rng = np.random.Generator(np.random.PCG64(seed))
    a = rng.standard_normal((3, n, n, n))
    ah = _fft.rfftn(a, axes=(1, 2, 3), **_FFT_KW)
    del a
    kz = (np.fft.fftfreq(n) * n).reshape(n, 1, 1)
    ky = (np.fft.fftfreq(n) * n).reshape(1, n, 1)
    kx = (np.fft.rfftfreq(n) * n).reshape(1, 1, n // 2 + 1)
    k2 = kx * kx + ky * ky + kz * kz
    kdota = kx * ah[0] + ky * ah[1] + kz * ah[2]
    inv = np.zeros_like(k2)
    np.divide(1.0, k2, out=inv, where=k2 > 0)
    kmag = np.sqrt(k2)
    amp = kmag * np.exp(-(kmag / k_peak) ** 2)
    nyq = (np.abs(kx) == n // 2) | (np.abs(ky) == n // 2) | (np.abs(kz) == n // 2)
    amp = np.where(nyq, 0.0, amp)
    for al, kal in enumerate((kx, ky, kz)):
        ah[al] = (ah[al] - kal * kdota * inv) * amp
    ah[:, 0, 0, 0] = 0.0
    u = _fft.irfftn(ah, s=(n, n, n), axes=(1, 2, 3), **_FFT_KW)
    del ah
    u *= urms / np.sqrt(np.mean(u * u))  # mean over 3 n^3 entries == <u.u>/3
    return np.ascontiguousarray(u)


def droplet_phi(n, radius, width=4.0, centre=None):
    """Config 3: phi = 0.5 (1 + tanh(2 (R - r) / W)), sphere centred at (n-1)/2 so it is lattice-symmetric."""
    c = (n - 1) / 2.0 if centre is None else centre
    ax = np.arange(n, dtype=np.float64)
    Z, Y, X = np.meshgrid(ax, ax, ax, indexing="ij")
    r = np.sqrt((X - c) ** 2 + (Y - c) ** 2 + (Z - c) ** 2)
    return 0.5 * (1.0 + np.tanh(2.0 * (radius - r) / width))


def bubble_centres(n, n_bubbles, radius=16.0, width=4.0, seed=SEED_BUBBLES, max_draws=10_000_000):
    """Uniform centres with rejection at minimum-image separation < 2R + 2W."""
    rng = np.random.Generator(np.random.PCG64(seed))
    dmin = 2.0 * radius + 2.0 * width
    centres = []
    draws = 0
    while len(centres) < n_bubbles:
        draws += 1
        if draws > max_draws:
            raise RuntimeError("bubble rejection sampling did not converge")
        c = rng.uniform(0.0, n, 3)
        ok = True
        for o in centres:
            d = np.abs(c - o)
            d = np.minimum(d, n - d)
            if np.sqrt(np.sum(d * d)) < dmin:
                ok = False
                break
        if ok:
            centres.append(c)
    return np.array(centres)


def bubbles_phi(n, centres, radius=16.0, width=4.0):
    """R27: phi = sum_b 0.5 (1 + tanh(2 (R - r_b) / W)), r_b the periodic minimum-image distance.  Each term is
    evaluated on the cube of half-width R + 10 W around its centre; outside it the term is exactly 0 in fp64
    (1 + tanh(-x) rounds to 0 for x > 18.72), so this equals the full-domain sum bit for bit."""
    phi = np.zeros((n, n, n))
    half = int(np.ceil(radius + 10.0 * width)) + 1
    for c in np.atleast_2d(centres):
        cx, cy, cz = c
        if 2 * half + 1 >= n:
            ix = iy = iz = np.arange(n)
        else:
            ix = np.arange(int(np.floor(cx)) - half, int(np.floor(cx)) + half + 2)
            iy = np.arange(int(np.floor(cy)) - half, int(np.floor(cy)) + half + 2)
            iz = np.arange(int(np.floor(cz)) - half, int(np.floor(cz)) + half + 2)

        def mind(i, c0):
            d = np.abs((i % n).astype(np.float64) - c0)
            return np.minimum(d, n - d)

        dz = mind(iz, cz).reshape(-1, 1, 1)
        dy = mind(iy, cy).reshape(1, -1, 1)
        dx = mind(ix, cx).reshape(1, 1, -1)
        r = np.sqrt(dx * dx + dy * dy + dz * dz)
        term = 0.5 * (1.0 + np.tanh(2.0 * (radius - r) / width))
        phi[np.ix_(iz % n, iy % n, ix % n)] += term
    return phi


def n_bubbles_for_void_fraction(n, frac=0.03, radius=16.0):
    """Config 5: 'scaled to 3 % void fraction' -> 1, 4, 29, 99, 235 bubbles for n = 64..512."""
    return max(1, int(round(frac * n ** 3 / (4.0 / 3.0 * np.pi * radius ** 3))))


def subbox(field, origin, size):
    """Periodic sub-box [oz:oz+s, oy:oy+s, ox:ox+s] (origin given as (x, y, z)) of a scalar or vector field."""
    ox, oy, oz = origin
    sx, sy, sz = (size, size, size) if np.isscalar(size) else size
    nz, ny, nx = field.shape[-3:]
    out = np.take(field, np.arange(oz, oz + sz) % nz, axis=-3)
    out = np.take(out, np.arange(oy, oy + sy) % ny, axis=-2)
    out = np.take(out, np.arange(ox, ox + sx) % nx, axis=-1)
    return np.ascontiguousarray(out)


_BASE = dict(tau=0.8, two_phase=0, rho_l=1.0, rho_g=1.0, sigma=0.0, mobility=0.0, width=4.0,
             force_type=0, force_amp=0.0, force_k=1)


def make_config(name, n=None, density_ratio=1.0, void_fraction=None):
    """Return dict(name, n, steps, params, rho, u, phi) for a BASELINE.json config.

    name: 'tgv' (1), 'hit' (2), 'droplet' (3), 'bubbly' (4), 'sweep1' / 'sweep2' (5, single- / two-phase).
    n overrides the grid size (the tests run scaled-down copies of the same recipes)."""
    p = dict(_BASE)
    phi = None
    if name == "tgv":
        n = n or 32
        rho, u = tgv_fields(n)
        p.update(tau=0.8)
        steps = 100
    elif name in ("hit", "sweep1"):
        n = n or 128
        u = hit_velocity(n)
        rho = np.ones((n, n, n))
        p.update(tau=0.51, force_type=2, force_amp=1e-5, force_k=1)
        steps = 1000 if name == "hit" else 200
    elif name == "droplet":
        n = n or 256
        radius = 40.0 * n / 256.0
        phi = droplet_phi(n, radius)
        u = np.zeros((3, n, n, n))
        # R26: zero gauge pressure when the densities differ
        rho = np.ones((n, n, n)) if density_ratio == 1.0 else np.zeros((n, n, n))
        p.update(tau=0.8, two_phase=1, rho_l=float(density_ratio), rho_g=1.0, sigma=0.01, mobility=0.05, width=4.0)
        steps = 5000
    elif name in ("bubbly", "sweep2"):
        n = n or 512
        u = hit_velocity(n)
        rho = np.ones((n, n, n))
        if name == "bubbly" and void_fraction is None:
            nb = max(1, int(round(60 * (n / 512.0) ** 3)))
        else:
            nb = n_bubbles_for_void_fraction(n, 0.03 if void_fraction is None else void_fraction)
        phi = bubbles_phi(n, bubble_centres(n, nb))
        p.update(tau=0.505, two_phase=1, sigma=0.02, mobility=0.05, width=4.0,
                 force_type=2, force_amp=1e-5, force_k=1)
        steps = 2000 if name == "bubbly" else 200
    else:
        raise ValueError(f"unknown config {name!r}")
    return dict(name=name, n=n, steps=steps, params=p, rho=rho, u=u, phi=phi)
