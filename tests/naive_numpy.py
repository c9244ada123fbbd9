"""P13: a second, deliberately different evaluation of the accLB step, used only to cross-check the oracle's
bookkeeping (index wraps, axis order, sign of c_i, neighbour look-ups) on tiny boxes.

Structure differs from oracle/acclb_oracle.c on purpose: whole-array numpy with np.roll, collide AT the node
(Eq. 4 in BGK form applied to Hermite-projected populations) followed by a PUSH stream, where the oracle
rebuilds populations at the neighbour from stored moments and pulls (Eq. 6).  The two are equal in exact
arithmetic.  Not imported by the product, the oracle, or bench.py.
"""
import itertools

import numpy as np

CS2 = 1.0 / 3.0


def lattice():
    c = np.array([(cx, cy, cz) for cz, cy, cx in itertools.product((-1, 0, 1), repeat=3)])
    nnz = np.abs(c).sum(1)
    w = np.choose(nnz, [8 / 27, 2 / 27, 1 / 54, 1 / 216])
    return c, w


C, W = lattice()
H = np.einsum("ia,ib->iab", C, C) - CS2 * np.eye(3)


def shift(field, c):
    """field(x + c) on the periodic box; field is [..., z, y, x], c = (cx, cy, cz)."""
    return np.roll(field, shift=(-c[2], -c[1], -c[0]), axis=(-3, -2, -1))


def grad(psi):
    return 3.0 * sum(W[i] * C[i][:, None, None, None] * shift(psi, C[i])[None] for i in range(27))


def div(vec):
    return 3.0 * sum(W[i] * sum(C[i][al] * shift(vec[al], C[i]) for al in range(3)) for i in range(27))


def lap(psi):
    return 6.0 * sum(W[i] * (shift(psi, C[i]) - psi) for i in range(27))


def weno5(a, b, c, d, e):
    q0 = (2 * a - 7 * b + 11 * c) / 6
    q1 = (-b + 5 * c + 2 * d) / 6
    q2 = (2 * c + 5 * d - e) / 6
    b0 = 13 / 12 * (a - 2 * b + c) ** 2 + 0.25 * (a - 4 * b + 3 * c) ** 2
    b1 = 13 / 12 * (b - 2 * c + d) ** 2 + 0.25 * (b - d) ** 2
    b2 = 13 / 12 * (c - 2 * d + e) ** 2 + 0.25 * (3 * c - 4 * d + e) ** 2
    a0, a1, a2 = 0.1 / (1e-6 + b0) ** 2, 0.6 / (1e-6 + b1) ** 2, 0.3 / (1e-6 + b2) ** 2
    return (a0 * q0 + a1 * q1 + a2 * q2) / (a0 + a1 + a2)


def body_force(p, shape):
    nz, ny, nx = shape
    Z, Y, X = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    k = p.get("force_k", 1)
    kx, ky, kz = 2 * np.pi * k / nx, 2 * np.pi * k / ny, 2 * np.pi * k / nz
    A = p.get("force_amp", 0.0)
    F = np.zeros((3,) + tuple(shape))
    if p.get("force_type", 0) == 1:
        F[0] = A * (np.sin(kz * Z) + np.cos(ky * Y))
        F[1] = A * (np.sin(kx * X) + np.cos(kz * Z))
        F[2] = A * (np.sin(ky * Y) + np.cos(kx * X))
    elif p.get("force_type", 0) == 2:
        F[0] = A * np.sin(ky * Y)
        F[1] = A * np.sin(kz * Z)
        F[2] = A * np.sin(kx * X)
    return F


def feq(pstar, u):
    cu = np.einsum("ia,a...->i...", C, u)
    huu = np.einsum("iab,a...,b...->i...", H, u, u)
    return W[:, None, None, None] * (pstar[None] + 3 * cu + 4.5 * huu)


def guo(u, A):
    cu = np.einsum("ia,a...->i...", C, u)
    cA = np.einsum("ia,a...->i...", C, A)
    uA = np.einsum("a...,a...->...", u, A)
    return W[:, None, None, None] * (3 * (cA - uA[None]) + 9 * cu * cA)


def forces(pstar, m, Pi, phi, p, with_visc=True):
    """rho, total force F, and the phi geometry (g, n) from the node moments p*, m, Pi."""
    shape = pstar.shape
    Fb = body_force(p, shape)
    if not p.get("two_phase", 0):
        return np.ones(shape), Fb, None, None
    g = grad(phi)
    gn = np.sqrt((g * g).sum(0))
    n = g / (gn + 1e-12)
    kc = div(n)
    rho = p["rho_g"] + (p["rho_l"] - p["rho_g"]) * phi
    drho = (p["rho_l"] - p["rho_g"]) * g
    Fs = -p["sigma"] * 1.5 * p["width"] * kc * gn * g
    Fp = -pstar * CS2 * drho
    Fv = np.zeros_like(Fs)
    if with_visc and p["rho_l"] != p["rho_g"]:
        ut = m + (Fs + Fp + Fb) / (2 * rho)
        T = Pi - pstar * CS2 * np.eye(3)[:, :, None, None, None] - np.einsum("a...,b...->ab...", ut, ut)
        Fv = -((p["tau"] - 0.5) / p["tau"]) * np.einsum("ab...,b...->a...", T, drho)
    return rho, Fs + Fp + Fv + Fb, g, n


def init(pstar, u0, phi, p):
    rho, F, _, _ = forces(pstar, None, None, phi, p, with_visc=False)
    A = F / rho
    return feq(pstar, u0) - 0.5 * guo(u0, A)


def moments(f, phi, p):
    m = np.einsum("i...,ia->a...", f, C)
    Pi = np.einsum("i...,ia,ib->ab...", f, C, C)
    rho, F, g, n = forces(f.sum(0), m, Pi, phi, p)
    A = F / rho
    u = np.einsum("i...,ia->a...", f, C) + 0.5 * A
    return f.sum(0), u, A, rho, n


def step(f, phi, p):
    """One step, collide-then-push.  Returns (f_new, phi_new)."""
    omega = 1.0 / p["tau"]
    pstar, u, A, rho, n = moments(f, phi, p)
    fe, S = feq(pstar, u), guo(u, A)
    fneq = f - fe + 0.5 * S
    a = np.einsum("i...,iab->ab...", fneq, H)
    fproj = fe - 0.5 * S + W[:, None, None, None] * 4.5 * np.einsum("iab,ab...->i...", H, a)  # Hermite-space f
    fpost = fproj + omega * (fe - fproj) + (1 - omega / 2) * S                              # Eq. 4
    fnew = np.stack([shift(fpost[i], -C[i]) for i in range(27)])                             # push: f_i(x+c_i) = post(x)
    phin = None
    if p.get("two_phase", 0):
        adv = np.zeros_like(phi)
        for ax, e in enumerate(((1, 0, 0), (0, 1, 0), (0, 0, 1))):
            e = np.array(e)
            uf = 0.5 * (u[ax] + shift(u[ax], e))
            P = lambda k: shift(phi, k * e)
            left = weno5(P(-2), P(-1), P(0), P(1), P(2))
            right = weno5(P(3), P(2), P(1), P(0), P(-1))
            flux = uf * np.where(uf >= 0, left, right)
            adv += flux - shift(flux, -e)
        q = phi * (1 - phi) * n
        D = p["mobility"]
        phin = phi + (-adv + D * lap(phi) - (4 * D / p["width"]) * div(q))
    return fnew, phin
