"""Turbulence statistics of a velocity field, plain numpy fp64 -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/__init__.py).

The definitions of PAPER.md:L171-189 and L205-213 written out:
  structure functions   S_p(r) = < (u_a(x + r e_a) - u_a(x))^p >, longitudinal, averaged over nodes and the three axes (L189)
  gradient moments      the central difference (u_a(x + e_a) - u_a(x - e_a)) / 2: skewness and flatness of L183
  PDFs                  histograms of increments / scale on equal bins (Fig. 3a, Fig. 6)
  spectra               E(k) = sum over modes with round(|k|) = k of |u^(k)|^2 / (2 N^2) (Fig. 2, Fig. 5), numpy.fft as the
                        library primitive
It shares nothing with paper_2505_01126_b200/csrc/stats.cuh.
"""
import numpy as np


def increments(u, r):
    """The three longitudinal increment fields d_a = u_a(x + r e_a) - u_a(x) of u [3][nz][ny][nx] (axis a=0 is x)."""
    return [np.roll(u[a], -r, axis=2 - a) - u[a] for a in range(3)]


def structure_functions(u, separations):
    out = []
    for r in separations:
        d = np.stack(increments(u, r))
        out.append([float(np.mean(d ** p)) for p in (2, 3, 4)])
    return out


def gradient_moments(u):
    """<g^2>, skewness <g^3>/<g^2>^{3/2}, flatness <g^4>/<g^2>^2 of g = central difference of u_a along a (L183)."""
    g = np.stack([(np.roll(u[a], -1, axis=2 - a) - np.roll(u[a], 1, axis=2 - a)) / 2.0 for a in range(3)])
    m2, m3, m4 = (float(np.mean(g ** p)) for p in (2, 3, 4))
    return m2, m3 / m2 ** 1.5, m4 / m2 ** 2


def pdf_counts(u, r, scale, lo, hi, nbins):
    d = np.stack(increments(u, r)) * (1.0 / scale)
    b = np.floor((d - lo) * (nbins / (hi - lo)))
    b = np.clip(b, 0, nbins - 1).astype(np.int64)
    return np.bincount(b.ravel(), minlength=nbins)


def spectrum(fields, nshell):
    """fields [ncomp][nz][ny][nx] real; E[k], k = 0..nshell-1, with sum_k E[k] = <f.f>/2 when all modes are covered."""
    ncomp, nz, ny, nx = fields.shape
    fh = np.fft.fftn(fields, axes=(1, 2, 3))                  # the full transform: no conjugate-half bookkeeping
    e = 0.5 * (np.abs(fh) ** 2).sum(axis=0) / float(nx * ny * nz) ** 2
    kz = np.fft.fftfreq(nz) * nz
    ky = np.fft.fftfreq(ny) * ny
    kx = np.fft.fftfreq(nx) * nx
    kk = np.sqrt(kz[:, None, None] ** 2 + ky[None, :, None] ** 2 + kx[None, None, :] ** 2)
    ks = np.floor(kk + 0.5).astype(np.int64)
    E = np.bincount(ks.ravel(), weights=e.ravel(), minlength=nshell)
    return E[:nshell]
