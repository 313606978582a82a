"""Pins for the CPU oracle beyond the paper's explicit range, 10 <= l <= 32 (the "extension by recurrence" the paper
proposes in its conclusion; sh_real_ext / sh_complex_ext on the CUDA side).

The oracle's arithmetic is the same Eq. 5 / Eq. 6 code as for l <= 9 (oracle/sh_oracle.c); the paper prints no values
beyond l = 9, so everything here pins it to closed forms, exact identities, quadrature and independent library
routines (mpmath.spherharm at 40 digits, scipy.special.sph_harm_y, numpy's Legendre series).  No GPU, no CUDA path.
"""
import math

import numpy as np

LEXT = 32


def k_of(l, m):
    return l * (l + 1) + m


def unit_vectors(n, seed):
    rng = np.random.default_rng(seed)
    g = rng.standard_normal((n, 3))
    return g / np.linalg.norm(g, axis=1)[:, None]


def angles(pts):
    r = np.linalg.norm(pts, axis=1)
    return np.arccos(np.clip(pts[:, 2] / r, -1, 1)), np.arctan2(pts[:, 1], pts[:, 0])


def test_prefix_property(oracle_mod):
    """The first (l'+1)^2 columns do not depend on lmax (bitwise): the l <= 9 pins carry over to the larger call."""
    pts = unit_vectors(300, 60) * 1.7
    big = oracle_mod.real(pts, LEXT)
    assert big.shape == (300, (LEXT + 1) ** 2)
    for lmax in (0, 4, 9, 15):
        assert np.array_equal(big[:, : (lmax + 1) ** 2], oracle_mod.real(pts, lmax))
    cbig = oracle_mod.complex_(pts, LEXT)
    assert np.array_equal(cbig[:, :100], oracle_mod.complex_(pts, 9))


def test_against_mpmath_spherharm(oracle_mod):
    """mpmath.spherharm at 40 digits, all m of selected l, at random points and at points close to the poles."""
    import mpmath

    mpmath.mp.dps = 40
    pts = list(unit_vectors(3, 61) * 0.3)
    for s in (1e-2, 1e-5):
        pts.append(np.array([s * np.cos(0.7), s * np.sin(0.7), 1.0]))
        pts.append(np.array([-s * np.cos(0.2), s * np.sin(0.2), -1.0]))
    pts = np.array(pts)
    Y = oracle_mod.complex_(pts, LEXT)
    R = oracle_mod.real(pts, LEXT)
    worst = 0.0
    for i, (x, y, z) in enumerate(pts):
        X, Yc, Z = mpmath.mpf(float(x)), mpmath.mpf(float(y)), mpmath.mpf(float(z))
        rr = mpmath.sqrt(X * X + Yc * Yc + Z * Z)
        theta, phi = mpmath.acos(Z / rr), mpmath.atan2(Yc, X)
        for l in (10, 11, 16, 23, 32):
            for m in range(0, l + 1):
                ref = mpmath.spherharm(l, m, theta, phi)
                worst = max(worst, abs(complex(ref) - Y[i, k_of(l, m)]))
                refm = (-1) ** m * mpmath.conj(ref)  # Eq. 10
                worst = max(worst, abs(complex(refm) - Y[i, k_of(l, -m)]))
                if m > 0:
                    worst = max(worst, abs(float(mpmath.sqrt(2) * (-1) ** m * ref.real) - R[i, k_of(l, m)]))
                    worst = max(worst, abs(float(mpmath.sqrt(2) * (-1) ** m * ref.imag) - R[i, k_of(l, -m)]))
                else:
                    worst = max(worst, abs(float(ref.real) - R[i, k_of(l, 0)]))
    assert worst <= 5e-15, worst


def test_against_scipy_all_lm(oracle_mod):
    """Every (l, m), 10 <= l <= 32, against the fp64 library routine (its own error grows with l and near the poles)."""
    from scipy.special import sph_harm_y

    pts = unit_vectors(400, 62) * 2.0
    th, ph = angles(pts)
    keep = np.sin(th) > 0.1
    Y = oracle_mod.complex_(pts, LEXT)
    for l in range(10, LEXT + 1):
        for m in range(-l, l + 1):
            assert np.abs(Y[keep, k_of(l, m)] - sph_harm_y(l, m, th[keep], ph[keep])).max() <= 1e-12, (l, m)


def test_zonal_and_sectoral_closed_forms(oracle_mod):
    """m = 0: Y_l^0 = sqrt((2l+1)/4pi) P_l(cos theta), P_l from numpy's Legendre series (library routine).
    m = l:  Y_l^l = (-1)^l/(2^l l!) sqrt((2l+1)!/(4 pi)) sin^l(theta) e^{i l phi}   (closed form, any l)."""
    from numpy.polynomial import legendre

    pts = unit_vectors(500, 63)
    th, ph = angles(pts)
    Y = oracle_mod.complex_(pts, LEXT)
    for l in range(10, LEXT + 1):
        c = np.zeros(l + 1)
        c[l] = 1.0
        zonal = math.sqrt((2 * l + 1) / (4 * math.pi)) * legendre.legval(np.cos(th), c)
        assert np.abs(Y[:, k_of(l, 0)].real - zonal).max() <= 2e-13 and np.abs(Y[:, k_of(l, 0)].imag).max() == 0.0
        # exact integer arithmetic for the constant
        amp = (-1) ** l * math.sqrt(math.factorial(2 * l + 1) / (4 * math.pi)) / (2**l * math.factorial(l))
        sect = amp * np.sin(th) ** l * np.exp(1j * l * ph)
        assert np.abs(Y[:, k_of(l, l)] - sect).max() <= 1e-13, l


def test_unsoeld_all_l(oracle_mod):
    """Addition theorem: sum_m |Y_l^m|^2 = sum_m (R_l^m)^2 = (2l+1)/(4 pi) at every point with r > 0."""
    pts = unit_vectors(1000, 64) * np.random.default_rng(65).uniform(1e-3, 1e2, (1000, 1))
    R = oracle_mod.real(pts, LEXT)
    Y = oracle_mod.complex_(pts, LEXT)
    for l in range(LEXT + 1):
        sl = slice(l * l, (l + 1) ** 2)
        want = (2 * l + 1) / (4 * math.pi)
        assert np.abs((R[:, sl] ** 2).sum(1) - want).max() <= 1e-14 * (2 * l + 1)
        assert np.abs((np.abs(Y[:, sl]) ** 2).sum(1) - want).max() <= 1e-14 * (2 * l + 1)


def test_orthonormality_by_quadrature(oracle_mod):
    """All 1089 real functions for l <= 32: Gauss-Legendre(33) in cos(theta) x 66 uniform phi integrates every product
    (degree <= 64 in cos(theta), |m + m'| <= 64 < 66) exactly: Gram matrix = identity."""
    n_t, n_p = LEXT + 1, 2 * LEXT + 2
    ct, wt = np.polynomial.legendre.leggauss(n_t)
    ph = 2 * np.pi * np.arange(n_p) / n_p
    T, P = np.meshgrid(np.arccos(ct), ph, indexing="ij")
    W = (wt[:, None] * np.full((1, n_p), 2 * np.pi / n_p)).ravel()
    tp = np.stack([T.ravel(), P.ravel()], axis=1)
    R = oracle_mod.real_angular(tp, LEXT)
    G = (R * W[:, None]).T @ R
    assert np.abs(G - np.eye(G.shape[0])).max() <= 2e-13
    Y = oracle_mod.complex_angular(tp, LEXT)
    Gc = (Y.conj() * W[:, None]).T @ Y
    assert np.abs(Gc - np.eye(Gc.shape[0])).max() <= 2e-13


def test_symmetries_high_l(oracle_mod):
    pts = unit_vectors(300, 66) * 0.8
    R = oracle_mod.real(pts, LEXT)
    Rm = oracle_mod.real(-pts, LEXT)
    Rz = oracle_mod.real(pts * np.array([1.0, 1.0, -1.0]), LEXT)
    Rs = oracle_mod.real(pts * 37.5, LEXT)
    Y = oracle_mod.complex_(pts, LEXT)
    for l in range(10, LEXT + 1):
        sl = slice(l * l, (l + 1) ** 2)
        assert np.abs(Rm[:, sl] - (-1) ** l * R[:, sl]).max() <= 1e-15  # parity
        assert np.abs(Rs[:, sl] - R[:, sl]).max() <= 5e-15  # norm independence
        for m in range(-l, l + 1):
            assert np.abs(Rz[:, k_of(l, m)] - (-1) ** (l + abs(m)) * R[:, k_of(l, m)]).max() <= 1e-15  # z mirror
            assert np.abs(Y[:, k_of(l, -m)] - (-1) ** m * Y[:, k_of(l, m)].conj()).max() <= 2.3e-16  # Eq. 10 (a property of the oracle, not an input: equal up to the final rounding to fp64)


def test_origin_and_poles_high_l(oracle_mod):
    pts = np.array([[0.0, 0.0, 0.0], [0.0, 0.0, 2.5], [0.0, 0.0, -0.1]])
    R = oracle_mod.real(pts, LEXT)
    assert R[0, 0] == 1 / math.sqrt(4 * math.pi) and np.all(R[0, 1:] == 0)
    for l in range(LEXT + 1):
        for m in range(-l, l + 1):
            want = math.sqrt((2 * l + 1) / (4 * math.pi)) if m == 0 else 0.0
            assert abs(R[1, k_of(l, m)] - want) <= 1e-15
            assert abs(R[2, k_of(l, m)] - (-1) ** l * want) <= 1e-15
