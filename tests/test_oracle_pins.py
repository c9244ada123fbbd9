"""Pins for the CPU oracle's building blocks: closed forms, invariants and textbook special cases.

Numbering P1..P14 follows DESIGN.md section 4 (= SURVEY.md section 8(c) "Pins").  Nothing here touches the CUDA path.
"""
import itertools

import numpy as np
import pytest

import oracle

CS2 = 1.0 / 3.0


# ---------------------------------------------------------------- P1: lattice identities (R1)
def test_p1_lattice_identities():
    c, w = oracle.lattice()
    assert c.shape == (27, 3) and set(np.unique(c)) == {-1, 0, 1}
    assert len({tuple(v) for v in c}) == 27
    # index convention i = (cx+1) + 3(cy+1) + 9(cz+1), rest = 13, opposite = 26 - i
    for i, (cx, cy, cz) in enumerate(c):
        assert i == (cx + 1) + 3 * (cy + 1) + 9 * (cz + 1)
        assert tuple(c[26 - i]) == (-cx, -cy, -cz)
    assert abs(w.sum() - 1) < 1e-15
    assert np.abs((w[:, None] * c).sum(0)).max() < 1e-15
    m2 = np.einsum("i,ia,ib->ab", w, c, c)
    assert np.abs(m2 - CS2 * np.eye(3)).max() < 1e-15
    m3 = np.einsum("i,ia,ib,ic->abc", w, c, c, c)
    assert np.abs(m3).max() < 1e-15
    d = np.eye(3)
    iso4 = CS2 ** 2 * (np.einsum("ab,cd->abcd", d, d) + np.einsum("ac,bd->abcd", d, d) + np.einsum("ad,bc->abcd", d, d))
    m4 = np.einsum("i,ia,ib,ic,id->abcd", w, c, c, c, c)
    assert np.abs(m4 - iso4).max() < 1e-15


# ---------------------------------------------------------------- P2: moments of f^eq and S_i
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_p2_equilibrium_and_forcing_moments(seed):
    rng = np.random.default_rng(seed)
    c, w = oracle.lattice()
    p = 1.0 + 0.1 * rng.standard_normal()
    u = 0.1 * rng.standard_normal(3)
    A = 0.01 * rng.standard_normal(3)
    fe = oracle.feq(p, u)
    assert abs(fe.sum() - p) < 2e-15
    assert np.abs(fe @ c - u).max() < 2e-15
    assert np.abs(np.einsum("i,ia,ib->ab", fe, c, c) - (p * CS2 * np.eye(3) + np.outer(u, u))).max() < 2e-15
    S = oracle.guo(u, A)
    H = np.einsum("ia,ib->iab", c, c) - CS2 * np.eye(3)
    assert abs(S.sum()) < 1e-16
    assert np.abs(S @ c - A).max() < 1e-16
    assert np.abs(np.einsum("i,iab->ab", S, H) - (np.outer(u, A) + np.outer(A, u))).max() < 1e-16


def test_p2_equilibrium_explicit_values():
    """Rest and one face direction written out by hand from PAPER.md:L88 for u = (ux,0,0)."""
    p, ux = 1.25, 0.05
    fe = oracle.feq(p, [ux, 0, 0])
    # rest i=13: w0 (p - ux^2/(2 cs2)) ; face +x i=14: w1 (p + ux/cs2 + (1-cs2) ux^2 / (2 cs4))
    assert abs(fe[13] - 8 / 27 * (p - 1.5 * ux * ux)) < 1e-16
    assert abs(fe[14] - 2 / 27 * (p + 3 * ux + 4.5 * (2 / 3) * ux * ux)) < 1e-16
    assert abs(fe[12] - 2 / 27 * (p - 3 * ux + 4.5 * (2 / 3) * ux * ux)) < 1e-16
    # corner (+,+,+) i=26: w3 (p + 3ux + 4.5 (1 - 1/3) ux^2)
    assert abs(fe[26] - 1 / 216 * (p + 3 * ux + 3.0 * ux * ux)) < 1e-16


# ---------------------------------------------------------------- P3: Hermite projection (R5)
def test_p3_projection_idempotent_and_conservative():
    rng = np.random.default_rng(3)
    c, w = oracle.lattice()
    H = np.einsum("ia,ib->iab", c, c) - CS2 * np.eye(3)
    a6 = 1e-3 * rng.standard_normal(6)
    fn = oracle.fneq(a6)
    assert abs(fn.sum()) < 1e-18          # mass: the form printed in PAPER.md:L88 (no w_i, no -cs2 delta) fails this
    assert np.abs(fn @ c).max() < 1e-18   # momentum
    a_back = np.einsum("i,iab->ab", fn, H)
    full = np.array([[a6[0], a6[3], a6[4]], [a6[3], a6[1], a6[5]], [a6[4], a6[5], a6[2]]])
    assert np.abs(a_back - full).max() < 1e-17


# ---------------------------------------------------------------- P5: lattice stencils (R7)
def test_p5_gradient_and_laplacian_polynomials():
    n = 12
    ax = np.arange(n, dtype=float)
    Z, Y, X = np.meshgrid(ax, ax, ax, indexing="ij")
    lin = 0.3 * X - 0.7 * Y + 1.1 * Z + 2.0
    g = oracle.gradient(lin)
    inner = (slice(1, -1),) * 3
    for al, val in enumerate((0.3, -0.7, 1.1)):
        assert np.abs(g[al][inner] - val).max() < 1e-13
    quad = 0.5 * X * X - 0.25 * Y * Y + 0.125 * Z * Z + 0.3 * X * Y - 0.2 * Y * Z + X
    lap = oracle.laplacian(quad)
    assert np.abs(lap[inner] - (1.0 - 0.5 + 0.25)).max() < 1e-12
    assert np.abs(oracle.laplacian(np.full((6, 6, 6), 3.7))).max() < 1e-14   # printed form gives 11/9 * 3.7
    gq = oracle.gradient(quad)  # central stencil is exact on quadratics too
    assert np.abs(gq[0][inner] - (X + 0.3 * Y + 1.0)[inner]).max() < 1e-12


@pytest.mark.parametrize("kvec", [(1, 0, 0), (0, 2, 0), (1, 2, 3), (3, 1, 2)])
def test_p5_stencil_plane_wave_symbols(kvec):
    """On exp(i k.x) the stencils act as multiplication by closed-form symbols that follow from the tensor-product
    structure of the D3Q27 weights: grad_a -> i sin(k_a) prod_{b!=a} (2+cos k_b)/3, lap -> 6(prod_a (2+cos k_a)/3 - 1)."""
    n = 16
    k = 2 * np.pi * np.array(kvec) / n
    ax = np.arange(n, dtype=float)
    Z, Y, X = np.meshgrid(ax, ax, ax, indexing="ij")
    ph = k[0] * X + k[1] * Y + k[2] * Z + 0.37
    s3 = (2 + np.cos(k)) / 3
    g = oracle.gradient(np.sin(ph))
    for al in range(3):
        sym = np.sin(k[al]) * np.prod(np.delete(s3, al))
        assert np.abs(g[al] - sym * np.cos(ph)).max() < 1e-13
    lap = oracle.laplacian(np.sin(ph))
    assert np.abs(lap - 6 * (np.prod(s3) - 1) * np.sin(ph)).max() < 1e-13


# ---------------------------------------------------------------- P10: WENO5 (R12, Jiang & Shu)
def test_p10_weno5_exact_on_quadratics_any_weights():
    """Every 3-cell candidate reproduces the face value of a quadratic from its cell AVERAGES, hence so does any
    convex combination: independent of the nonlinear weights."""
    rng = np.random.default_rng(10)
    for _ in range(20):
        c0, c1, c2 = rng.standard_normal(3)
        P = lambda x: c0 * x + c1 * x ** 2 / 2 + c2 * x ** 3 / 3        # antiderivative
        avg = [P(j + 0.5) - P(j - 0.5) for j in range(-2, 3)]
        face = c0 + c1 * 0.5 + c2 * 0.25
        assert abs(oracle.weno5(*avg) - face) < 1e-13


def test_p10_weno5_constant_and_eno_property():
    assert oracle.weno5(0.3, 0.3, 0.3, 0.3, 0.3) == pytest.approx(0.3, abs=1e-16)
    # discontinuity between c and d: only the left candidate (q0, beta0 = 0) is smooth -> value of the left state
    assert abs(oracle.weno5(0, 0, 0, 1, 1)) < 1e-11
    assert abs(oracle.weno5(1, 1, 1, 0, 0) - 1) < 1e-11
    # discontinuity between a and b: candidate q2 (cells c,d,e) is smooth
    assert abs(oracle.weno5(5, 1, 1, 1, 1) - 1) < 1e-11


def test_p10_weno5_fifth_order_on_smooth_data():
    """Weights -> (0.1,0.6,0.3) on smooth data, which makes the face value 5th-order accurate; wrong linear weights,
    candidate coefficients or smoothness indicators drop the order to 3."""
    def err(h):
        x0 = 0.4
        F = lambda x: -np.cos(x)                       # antiderivative of sin
        avg = [(F(x0 + (j + 0.5) * h) - F(x0 + (j - 0.5) * h)) / h for j in range(-2, 3)]
        return abs(oracle.weno5(*avg) - np.sin(x0 + 0.5 * h))
    e1, e2 = err(0.2), err(0.1)
    order = np.log2(e1 / e2)
    assert order > 4.5, (e1, e2, order)


def test_p10_weno5_linear_weight_limit_value():
    """With all smoothness indicators equal (data linear in j) the nonlinear weights equal d exactly and the face
    value is the classical 5th-order upwind formula (2a - 13b + 47c + 27d - 3e)/60."""
    a, b, c, d, e = [0.1 + 0.05 * j for j in range(5)]
    assert abs(oracle.weno5(a, b, c, d, e) - (2 * a - 13 * b + 47 * c + 27 * d - 3 * e) / 60) < 1e-15


# ---------------------------------------------------------------- R20: body force tables
def test_body_force_forms():
    P = oracle.OracleParams
    import ctypes as C
    p = P(16, 8, 4, 0.8, 0, 1, 1, 0, 0, 4, 1, 2.0, 1, (C.c_int * 3)(0, 0, 0), (C.c_int * 3)(0, 0, 0))
    x, y, z = 3, 5, 1
    kx, ky, kz = 2 * np.pi / 16, 2 * np.pi / 8, 2 * np.pi / 4
    F = oracle.body_force(p, x, y, z)   # ABC
    assert np.allclose(F, 2.0 * np.array([np.sin(kz * z) + np.cos(ky * y), np.sin(kx * x) + np.cos(kz * z),
                                          np.sin(ky * y) + np.cos(kx * x)]), atol=1e-15)
    p.force_type = 2
    F = oracle.body_force(p, x, y, z)
    assert np.allclose(F, 2.0 * np.array([np.sin(ky * y), np.sin(kz * z), np.sin(kx * x)]), atol=1e-15)
    # sub-box evaluation: origin shift + global period reproduce the global value
    q = P(4, 4, 4, 0.8, 0, 1, 1, 0, 0, 4, 2, 2.0, 1, (C.c_int * 3)(16, 8, 4), (C.c_int * 3)(2, 3, 1))
    assert np.allclose(oracle.body_force(q, 1, 2, 0), F, atol=1e-15)
    # both forms integrate to zero over the box (momentum pin P4 relies on it)
    tot = sum(oracle.body_force(p, i, j, k) for i, j, k in itertools.product(range(16), range(8), range(4)))
    assert np.abs(tot).max() < 1e-13
