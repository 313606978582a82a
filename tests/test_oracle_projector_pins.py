"""Pins of the oracle's fused projector consumer (oracle/sh_oracle.c: sh_oracle_projectors / sh_oracle_project;
SURVEY.md section 8(f2)) against what the definition and the mathematics fix -- none of them
calls the functions under test to produce the expected value:

  * a table of a LINEAR function is reproduced exactly by piecewise-linear interpolation, so
    beta = (a + b r) R_l^m with R from the separately pinned oracle.real (tests/test_oracle_pins.py);
  * at table nodes the tabulated value, at midpoints the mean of the neighbours (random tables);
  * beyond the table 0; at r = 0 only l = 0 survives;
  * column order for an unsorted channel list;
  * the projection against a quadrature rule that integrates products of two harmonics exactly gives the identity
    (orthonormality, Gauss-Legendre x uniform phi), scaled by the radial value;
  * the projection is linear in w and equals the brute-force dot product of independently built columns.
"""
import numpy as np
import pytest

import oracle

SQ4PI = np.sqrt(4.0 * np.pi)


def directions(n, seed):
    g = np.random.default_rng(seed).standard_normal((n, 3))
    return g / np.linalg.norm(g, axis=1)[:, None]


def columns(proj_l):
    """(p, l, m) of every output column, channel-major, m ascending (the stated convention)."""
    return [(p, l, m) for p, l in enumerate(proj_l) for m in range(-l, l + 1)]


def test_count_and_column_order():
    proj_l = [2, 0, 1, 1, 3, 0]
    assert oracle.projector_count(proj_l) == 5 + 1 + 3 + 3 + 7 + 1
    assert oracle.projector_count([]) == 0
    assert oracle.projector_count([-1]) == -1
    # distinct constant tables identify the channel of every column
    nr, dr = 41, 0.05
    tab = np.array([[float(p + 1)] * nr for p in range(len(proj_l))])
    pts = directions(50, 1) * np.random.default_rng(2).uniform(0.1, 1.5, 50)[:, None]
    got = oracle.projectors(pts, proj_l, tab, dr)
    R = oracle.real(pts, 3)
    for c, (p, l, m) in enumerate(columns(proj_l)):
        np.testing.assert_allclose(got[:, c], (p + 1) * R[:, l * (l + 1) + m], rtol=0, atol=2e-16 * (p + 1))


def test_linear_table_is_exact():
    proj_l = [0, 1, 2, 3, 5, 9]
    nr, dr = 301, 0.01
    r_nodes = np.arange(nr) * dr
    a = np.array([0.3, -1.2, 2.0, 0.7, -0.4, 1.1])
    b = np.array([1.5, 0.8, -0.6, 0.25, 2.2, -0.9])
    tab = a[:, None] + b[:, None] * r_nodes[None, :]
    rng = np.random.default_rng(3)
    rad = rng.uniform(0.0, 2.999, 4000)
    pts = directions(4000, 4) * rad[:, None]
    r = np.linalg.norm(pts, axis=1).astype(np.longdouble)   # the radius the definition uses, not `rad`
    pts64 = pts.astype(np.longdouble)
    r = np.sqrt(pts64[:, 0] ** 2 + pts64[:, 1] ** 2 + pts64[:, 2] ** 2)
    got = oracle.projectors(pts, proj_l, tab, dr)
    R = oracle.real(pts, 9)
    for c, (p, l, m) in enumerate(columns(proj_l)):
        want = (np.longdouble(a[p]) + np.longdouble(b[p]) * r) * R[:, l * (l + 1) + m].astype(np.longdouble)
        # R is the oracle's value rounded to double: half an ulp of R times |f| <= 8
        assert np.abs(got[:, c] - want.astype(np.float64)).max() <= 2e-15, (p, l, m)


def test_nodes_midpoints_cutoff_and_origin():
    rng = np.random.default_rng(5)
    proj_l = [0, 1, 2, 0]
    nr, dr = 33, 0.125   # dr a power of two: j*dr and (j+1/2)*dr are exact in fp64
    tab = rng.standard_normal((len(proj_l), nr))
    R1 = 1.0 / SQ4PI
    for axis, (l_axis, k_axis) in enumerate([(1, 3), (1, 1), (1, 2)]):   # R_1^{+1} ~ x, R_1^{-1} ~ y, R_1^0 ~ z  (k = l(l+1)+m)
        for j in range(0, nr + 4):
            for half in (0.0, 0.5):
                rr = (j + half) * dr
                p3 = np.zeros((1, 3))
                p3[0, axis] = rr
                got = oracle.projectors(p3, proj_l, tab, dr)[0]
                if rr >= (nr - 1) * dr:
                    assert np.all(got == 0.0), (axis, j, half)
                    continue
                f = tab[:, j] if half == 0.0 else 0.5 * (tab[:, j] + tab[:, j + 1])
                if rr == 0.0:
                    # only l = 0 survives
                    want = np.array([f[0] * R1, 0, 0, 0, 0, 0, 0, 0, 0, f[3] * R1])
                    np.testing.assert_allclose(got, want, rtol=0, atol=1e-16 * np.abs(f).max())
                    continue
                assert abs(got[0] - f[0] * R1) <= 3e-16 * abs(f[0]) + 1e-18
                assert abs(got[9] - f[3] * R1) <= 3e-16 * abs(f[3]) + 1e-18
                # l = 1 along a coordinate axis: R_1 = sqrt(3/4pi) on that axis' own function, 0 on the two others
                want_p = np.zeros(3)
                want_p[k_axis - 1] = np.sqrt(3.0 / (4.0 * np.pi)) * f[1]
                np.testing.assert_allclose(got[1:4], want_p, rtol=0, atol=3e-16 * abs(f[1]) + 1e-18)


def gauss_legendre_sphere(nt=12, nphi=24):
    """Nodes and weights integrating every product of two harmonics with l <= 9 exactly (degree 18 polynomials)."""
    ct, wt = np.polynomial.legendre.leggauss(nt)
    phi = 2.0 * np.pi * np.arange(nphi) / nphi
    st = np.sqrt(1.0 - ct * ct)
    pts = np.stack([np.outer(st, np.cos(phi)).ravel(), np.outer(st, np.sin(phi)).ravel(), np.repeat(ct, nphi)], axis=1)
    w = np.repeat(wt, nphi) * (2.0 * np.pi / nphi)
    return pts, w


def test_projection_against_exact_quadrature_is_the_identity():
    pts, qw = gauss_legendre_sphere()
    r0 = 1.7
    proj_l = list(range(10))                         # one channel per l: columns are exactly k = l(l+1)+m
    nr, dr = 64, 0.05
    r_nodes = np.arange(nr) * dr
    slope = 0.3 + 0.1 * np.arange(10)
    tab = 1.0 + slope[:, None] * r_nodes[None, :]    # linear tables: f_l(r0) = 1 + slope_l r0 exactly
    R = oracle.real(pts, 9)                          # separately pinned; used only to build the weights
    ks = [0, 2, 5, 17, 42, 63, 80, 99]
    w = np.stack([qw * R[:, k] for k in ks])
    coeff, abs_sum = oracle.project(pts * r0, proj_l, tab, dr, w)
    want = np.zeros((len(ks), 100))
    for v, k in enumerate(ks):
        l = int(np.floor(np.sqrt(k)))
        want[v, k] = 1.0 + slope[l] * r0
    # fp64 quadrature weights, fp64-rounded R in w and the rounding of r0 * unit vector each contribute ~1e-16 relative per term
    assert np.abs(coeff - want).max() <= 3e-14
    assert np.all(abs_sum >= np.abs(coeff) - 1e-15)


def test_projection_is_the_dot_product_and_linear_in_w():
    rng = np.random.default_rng(11)
    pts = directions(3000, 12) * rng.uniform(0, 3.2, 3000)[:, None]
    proj_l = [1, 0, 2, 2, 3]
    nr, dr = 31, 0.1
    r_nodes = np.arange(nr) * dr
    a, b = rng.standard_normal(5), rng.standard_normal(5)
    tab = a[:, None] + b[:, None] * r_nodes[None, :]     # linear up to the table's end at r = 3.0
    w = rng.standard_normal((3, 3000))
    coeff, abs_sum = oracle.project(pts, proj_l, tab, dr, w)
    # columns built independently from the pinned R and the closed-form radial function
    p64 = pts.astype(np.longdouble)
    r = np.sqrt(p64[:, 0] ** 2 + p64[:, 1] ** 2 + p64[:, 2] ** 2)
    inside = np.floor(r / np.longdouble(dr)) < nr - 1
    R = oracle.real(pts, 3).astype(np.longdouble)
    for c, (p, l, m) in enumerate(columns(proj_l)):
        beta = np.where(inside, np.longdouble(a[p]) + np.longdouble(b[p]) * r, 0) * R[:, l * (l + 1) + m]
        for v in range(3):
            terms = w[v].astype(np.longdouble) * beta
            assert abs(coeff[v, c] - float(terms.sum())) <= 1e-15 * float(np.abs(terms).sum()) + 1e-18
            assert abs(abs_sum[v, c] - float(np.abs(terms).sum())) <= 1e-14 * float(np.abs(terms).sum())
    both, _ = oracle.project(pts, proj_l, tab, dr, (2.0 * w[0] - 3.0 * w[1])[None, :])
    np.testing.assert_allclose(both[0], 2.0 * coeff[0] - 3.0 * coeff[1], rtol=0, atol=1e-12)


def test_bad_arguments_are_refused():
    pts = np.zeros((2, 3))
    with pytest.raises(ValueError):
        oracle.projectors(pts, [0], np.ones((1, 1)), 0.1)    # nr < 2
    with pytest.raises(ValueError):
        oracle.projectors(pts, [0], np.ones((1, 4)), 0.0)    # dr <= 0
    with pytest.raises(ValueError):
        oracle.projectors(pts, [0, 1], np.ones((1, 4)), 0.1)  # table rows != channels
