"""turbulence statistics.  CPU: the numpy oracle (oracle/stats_oracle.py) against closed forms; GPU: the
CUDA kernels (accLB_stats_*) against the oracle on the seeded turbulent field of config 2."""
import numpy as np
import pytest

from oracle import stats_oracle as so
from paper_2505_01126_b200 import workloads as wl


def sine_field(n, a, m):
    x = np.arange(n)
    u = np.zeros((3, n, n, n))
    u[0] = a * np.sin(2 * np.pi * m * x / n)[None, None, :]
    return u


def test_oracle_structure_functions_of_a_sine():
    """u = (a sin kx, 0, 0): d_x = a (sin k(x + r) - sin kx), so S_2 = a^2 (1 - cos kr) / 3, S_3 = 0,
    S_4 = a^4 (3/2)(1 - cos kr)^2 / 3 (the 1/3: two of the three axes contribute nothing)."""
    n, a, m = 32, 0.7, 3
    k = 2 * np.pi * m / n
    rs = [1, 2, 5, 16]
    S = so.structure_functions(sine_field(n, a, m), rs)
    for (s2, s3, s4), r in zip(S, rs):
        c = 1.0 - np.cos(k * r)
        assert abs(s2 - a * a * c / 3) < 1e-15 and abs(s3) < 1e-16 and abs(s4 - a ** 4 * 1.5 * c * c / 3) < 1e-15


def test_oracle_gradient_moments_are_the_r2_increments():
    """The central difference is the r = 2 increment shifted by one cell and halved: same moments on a periodic box.
    For the sine: <g^2> = a^2 sin^2(k) / 6, skewness 0, flatness 4.5 (1.5 per contributing axis)."""
    n, a, m = 32, 0.7, 3
    u = sine_field(n, a, m)
    m2, S, F = so.gradient_moments(u)
    k = 2 * np.pi * m / n
    assert abs(m2 - a * a * np.sin(k) ** 2 / 6) < 1e-15 and abs(S) < 1e-12 and abs(F - 4.5) < 1e-12
    rng = np.random.default_rng(5)
    v = rng.standard_normal((3, 12, 10, 14))
    (s2, s3, s4), = so.structure_functions(v, [2])
    g2, gs, gf = so.gradient_moments(v)
    assert abs(g2 - s2 / 4) < 1e-14 and abs(gs - s3 / s2 ** 1.5) < 1e-13 and abs(gf - s4 / s2 ** 2) < 1e-13
    assert abs(gf - 3.0) < 0.3 and abs(gs) < 0.15            # Gaussian: flatness 3, no skewness


def test_oracle_spectrum_parseval_and_single_mode():
    n, a, m = 16, 0.7, 3
    E = so.spectrum(sine_field(n, a, m), n)
    assert abs(E[m] - a * a / 4) < 1e-15 and abs(E.sum() - E[m]) < 1e-15      # <u.u>/2 = a^2 / 4, all of it in shell m
    rng = np.random.default_rng(6)
    v = rng.standard_normal((3, 8, 10, 12))
    assert abs(so.spectrum(v, 12).sum() - 0.5 * np.mean((v ** 2).sum(axis=0))) < 1e-13


def test_oracle_pdf_counts():
    rng = np.random.default_rng(7)
    v = rng.standard_normal((3, 6, 8, 10))
    c = so.pdf_counts(v, 1, 1.3, -4.0, 4.0, 64)
    assert c.sum() == 3 * 6 * 8 * 10
    d = np.stack(so.increments(v, 1)) / 1.3
    assert c[40] == np.count_nonzero((d >= 1.0) & (d < 1.125))


@pytest.mark.gpu
def test_gpu_statistics_match_the_oracle(acclb):
    import torch

    n = 64
    u = np.ascontiguousarray(wl.hit_velocity(n))
    ud = torch.from_numpy(u).cuda()
    rs = [1, 2, 3, 4, 8, 16, 32]
    S = np.array(acclb.stats_increments(ud, rs))
    So = np.array(so.structure_functions(u, rs))
    scale = So[:, :1] ** (np.array([2, 3, 4]) / 2.0)                          # S_3(N/2) is zero by periodicity: absolute bound
    assert (np.abs(S - So) / scale).max() < 1e-11, (S, So)
    rms2 = np.sqrt(So[1][0])
    c = np.array(acclb.stats_pdf(ud, 2, rms2, -8.0, 8.0, 128), dtype=np.int64)
    co = so.pdf_counts(u, 2, rms2, -8.0, 8.0, 128)
    assert c.sum() == 3 * n ** 3 and np.abs(c - co).sum() <= 4               # a value within rounding of a bin edge may move
    uh = torch.fft.rfftn(ud, dim=(1, 2, 3))                                   # the caller's library FFT
    E = np.array(acclb.stats_spectrum(uh.contiguous(), n, n))
    Eo = so.spectrum(u, n)
    assert np.abs(E - Eo).max() < 1e-13 * Eo.max()
    assert abs(E.sum() - 0.5 * (u ** 2).sum(axis=0).mean()) < 1e-12 * E.sum()
    # non-cubic box, odd nx, single component (a pressure-like field)
    rng = np.random.default_rng(8)
    v = rng.standard_normal((3, 10, 12, 15))
    vd = torch.from_numpy(v).cuda()
    assert np.abs(np.array(acclb.stats_increments(vd, [1, 7])) - np.array(so.structure_functions(v, [1, 7]))).max() < 1e-12
    ph = torch.fft.rfftn(vd[:1], dim=(1, 2, 3)).contiguous()
    assert np.abs(np.array(acclb.stats_spectrum(ph, 15, 12)) - so.spectrum(v[:1], 12)).max() < 1e-13
