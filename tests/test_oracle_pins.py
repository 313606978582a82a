"""Pins for the CPU oracle (oracle/sh_oracle.c): everything here checks the oracle against
something OTHER than itself -- values the paper prints, the paper's Appendix C formulas, hand-derived
closed forms, exact identities, quadrature orthonormality, and independent library routines
(scipy.special.sph_harm_y, mpmath.spherharm).  No GPU, no CUDA path.

Citations: P:n = /root/reference/PAPER.md line n (arxiv 2510.05282).
"""
import os

import numpy as np
import pytest

from appendix_c import FORMULAS, p

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_tables_II_III.txt")

# Appendix D points (P:407, P:409 with reading #4 for phi of Table III)
TABLE_POINTS = {
    "II": (2.12160245947564796, -1.82732370250979703),
    "III": (1.69050041976591414, 0.758228122208986166),
}


def k_of(l, m):
    return l * (l + 1) + m


def unit_vectors(n, seed):
    rng = np.random.default_rng(seed)
    g = rng.standard_normal((n, 3))
    return g / np.linalg.norm(g, axis=1)[:, None]


def load_golden():
    rows = []
    for line in open(GOLDEN):
        if line.startswith("#") or not line.strip():
            continue
        t, l, m, v, ln = line.split()
        rows.append((t, int(l), int(m), float(v)))
    return rows


# ----------------------------------------------------------------------------- paper tables
def test_golden_file_complete():
    rows = load_golden()
    assert len(rows) == 122
    for t in ("II", "III"):
        plus = {(l, m) for tt, l, m, _ in rows if tt == t and m >= 0}
        assert plus == {(l, m) for l in range(10) for m in range(l + 1)}  # all 55 R_l^{+m}
        minus = {(l, m) for tt, l, m, _ in rows if tt == t and m < 0}
        assert minus == {(1, -1), (2, -1), (6, -6), (7, -7), (8, -8), (9, -9)}


def test_tables_II_III_angular_core(oracle_mod):
    """Appendix D, Tables II/III: the oracle's angular core at the printed (theta, phi)."""
    R = {t: oracle_mod.real_angular(np.array([tp]), 9)[0] for t, tp in TABLE_POINTS.items()}
    for t, l, m, v in load_golden():
        assert abs(R[t][k_of(l, m)] - v) <= 1e-15, (t, l, m)


def test_tables_II_III_cartesian_entry(oracle_mod):
    """Same values through Eq. 3-4: x = sin(theta)cos(phi), ...."""
    for t, (th, ph) in TABLE_POINTS.items():
        th_l, ph_l = np.longdouble(th), np.longdouble(ph)
        xyz = np.array(
            [[np.sin(th_l) * np.cos(ph_l), np.sin(th_l) * np.sin(ph_l), np.cos(th_l)]], dtype=np.float64
        )
        R = oracle_mod.real(2.5 * xyz, 9)[0]  # any radius: harmonics do not depend on the norm
        for tt, l, m, v in load_golden():
            if tt == t:
                assert abs(R[k_of(l, m)] - v) <= 1e-14, (t, l, m)


# ----------------------------------------------------------------------------- Appendix C
def test_appendix_c_printed_formulas(oracle_mod):
    """47 factorized formulas of Appendix C as printed, at random unit vectors: pins
    every m <= 0 real harmonic family (sign, normalisation, which of sin/cos type)."""
    u = unit_vectors(4000, 11)
    R = oracle_mod.real(u, 9)
    assert len(FORMULAS) == 47
    for (l, m), f in FORMULAS.items():
        assert np.abs(f(u[:, 0], u[:, 1], u[:, 2]) - R[:, k_of(l, m)]).max() <= 3e-14, (l, m)


def test_worked_example_eq15(oracle_mod):
    """R_7^{-3}: Eq. 15 equals Eq. 5+6; Eq. 11-14 equal it after reading #24
    (prefactors 1/128 and 3/64 instead of the garbled 128 and 768)."""
    u = unit_vectors(1000, 12)
    x, y, z = u.T
    ref = oracle_mod.real(u, 7)[:, k_of(7, -3)]
    s35 = np.sqrt(35 / np.pi)
    eq15 = 429 / 64 * s35 * y * p(np.sqrt(3) * x, y) * p(np.sqrt((33 - 2 * np.sqrt(165)) / 143), z) * p(
        np.sqrt((33 + 2 * np.sqrt(165)) / 143), z
    )
    eq11 = (1 / 128) * s35 * y * (
        2574 * x**6 + 4290 * x**4 * y**2 + 858 * x**2 * y**4 - 858 * y**6 - 3960 * x**4 - 2640 * x**2 * y**2
        + 1320 * y**4 + 1440 * x**2 - 480 * y**2
    )
    eq12 = (3 / 64) * s35 * y * (3 * x**2 - y**2) * (
        143 * x**4 + 286 * x**2 * y**2 + 143 * y**4 - 220 * x**2 - 220 * y**2 + 80
    )
    eq14 = (3 / 64) * s35 * y * (3 * x**2 - y**2) * (11 * (z**2 - 1) * (13 * z**2 + 7) + 80)
    assert np.abs(eq15 - ref).max() <= 2e-14
    for e in (eq11, eq12, eq14):  # canonical forms carry more round-off
        assert np.abs(e - ref).max() <= 5e-13


# ----------------------------------------------------------------------------- closed forms l <= 2
def test_closed_forms_real_l2(oracle_mod):
    u = unit_vectors(500, 13) * np.random.default_rng(1).uniform(0.1, 9.0, (500, 1))
    r = np.linalg.norm(u, axis=1)
    x, y, z = (u / r[:, None]).T
    R = oracle_mod.real(u, 2)
    c1 = np.sqrt(3 / (4 * np.pi))
    expect = {
        (0, 0): 0.5 / np.sqrt(np.pi) + 0 * x,
        (1, -1): c1 * y, (1, 0): c1 * z, (1, 1): c1 * x,
        (2, -2): 0.5 * np.sqrt(15 / np.pi) * x * y,
        (2, -1): 0.5 * np.sqrt(15 / np.pi) * y * z,
        (2, 0): 0.25 * np.sqrt(5 / np.pi) * (3 * z * z - 1),
        (2, 1): 0.5 * np.sqrt(15 / np.pi) * x * z,
        (2, 2): 0.25 * np.sqrt(15 / np.pi) * (x * x - y * y),
    }
    for (l, m), e in expect.items():
        assert np.abs(R[:, k_of(l, m)] - e).max() <= 2e-15, (l, m)


def test_closed_forms_complex_l2(oracle_mod):
    u = unit_vectors(500, 14)
    x, y, z = u.T
    Y = oracle_mod.complex_(u, 2)
    xp, xm = x + 1j * y, x - 1j * y
    expect = {
        (0, 0): 0.5 / np.sqrt(np.pi) + 0j * x,
        (1, -1): np.sqrt(3 / (8 * np.pi)) * xm,
        (1, 0): np.sqrt(3 / (4 * np.pi)) * z + 0j,
        (1, 1): -np.sqrt(3 / (8 * np.pi)) * xp,          # Condon-Shortley sign
        (2, -2): 0.25 * np.sqrt(15 / (2 * np.pi)) * xm**2,
        (2, -1): 0.5 * np.sqrt(15 / (2 * np.pi)) * xm * z,
        (2, 0): 0.25 * np.sqrt(5 / np.pi) * (3 * z * z - 1) + 0j,
        (2, 1): -0.5 * np.sqrt(15 / (2 * np.pi)) * xp * z,
        (2, 2): 0.25 * np.sqrt(15 / (2 * np.pi)) * xp**2,
    }
    for (l, m), e in expect.items():
        assert np.abs(Y[:, k_of(l, m)] - e).max() <= 2e-15, (l, m)


# ----------------------------------------------------------------------------- identities
def test_unsoeld_addition_theorem(oracle_mod):
    """sum_m |Y_l^m|^2 = sum_m (R_l^m)^2 = (2l+1)/(4 pi) at every r > 0 point."""
    pts = unit_vectors(2000, 15) * 10.0 ** np.random.default_rng(2).uniform(-3, 2, (2000, 1))
    R = oracle_mod.real(pts, 9)
    Y = oracle_mod.complex_(pts, 9)
    for l in range(10):
        sl = slice(l * l, (l + 1) ** 2)
        want = (2 * l + 1) / (4 * np.pi)
        assert np.abs((R[:, sl] ** 2).sum(1) - want).max() <= 2e-14
        assert np.abs((np.abs(Y[:, sl]) ** 2).sum(1) - want).max() <= 2e-14


def test_spinor_sum_rule(oracle_mod):
    """sum_{m_j} S^dagger S = (2j+1)/(4 pi) for every (l, j)."""
    pts = unit_vectors(500, 16) * 3.0
    S = oracle_mod.spinor(pts, 9)
    dens = (np.abs(S) ** 2).sum(-1)  # [n][200]
    for l in range(10):
        for twoj in (2 * l - 1, 2 * l + 1):
            if twoj < 1:
                continue
            idx = [oracle_mod.index_spinor(l, twoj, tm) for tm in range(-twoj, twoj + 1, 2)]
            assert np.abs(dens[:, idx].sum(1) - (twoj + 1) / (4 * np.pi)).max() <= 2e-14, (l, twoj)


def quadrature_grid():
    """Gauss-Legendre (10 nodes in cos theta) x 20 uniform phi: exact for all products with l <= 9."""
    xs, ws = np.polynomial.legendre.leggauss(10)
    phis = 2 * np.pi * np.arange(20) / 20
    th, ph = np.meshgrid(np.arccos(xs), phis, indexing="ij")
    w = np.repeat(ws, 20) * (2 * np.pi / 20)
    return np.stack([th.ravel(), ph.ravel()], axis=1), w


def test_orthonormality_real_and_complex(oracle_mod):
    tp, w = quadrature_grid()
    R = oracle_mod.real_angular(tp, 9)
    G = (R * w[:, None]).T @ R
    assert np.abs(G - np.eye(100)).max() <= 1e-13
    Y = oracle_mod.complex_angular(tp, 9)
    G = (Y.conj() * w[:, None]).T @ Y
    assert np.abs(G - np.eye(100)).max() <= 1e-13


def test_orthonormality_spinor(oracle_mod):
    tp, w = quadrature_grid()
    S = oracle_mod.spinor_angular(tp, 9)          # [n][200][2]
    A = S.reshape(S.shape[0], 200, 2)
    G = np.einsum("n,nsc,ntc->st", w, A.conj(), A)
    assert np.abs(G - np.eye(200)).max() <= 1e-13


def test_symmetries(oracle_mod):
    pts = unit_vectors(1000, 17) * np.random.default_rng(3).uniform(0.2, 4.0, (1000, 1))
    R = oracle_mod.real(pts, 9)
    Y = oracle_mod.complex_(pts, 9)
    Rneg = oracle_mod.real(-pts, 9)
    Rscaled = oracle_mod.real(7.25 * pts, 9)
    Rmirror = oracle_mod.real(pts * np.array([1.0, 1.0, -1.0]), 9)
    for l in range(10):
        for m in range(-l, l + 1):
            k = k_of(l, m)
            assert np.abs(Rneg[:, k] - (-1) ** l * R[:, k]).max() <= 1e-14          # parity
            assert np.abs(Rscaled[:, k] - R[:, k]).max() <= 1e-14                   # norm independence
            assert np.abs(Rmirror[:, k] - (-1) ** (l + abs(m)) * R[:, k]).max() <= 1e-14
            # Eq. 10: Y_l^{-m} = (-1)^m conj(Y_l^m)
            assert np.abs(Y[:, k_of(l, -m)] - (-1) ** m * Y[:, k].conj()).max() <= 1e-15
            # Eq. 9 with reading #2 (1/sqrt2), m > 0: Y_l^m = (-1)^m (R_l^m + i R_l^{-m}) / sqrt 2
            if m > 0:
                want = (-1) ** m * (R[:, k] + 1j * R[:, k_of(l, -m)]) / np.sqrt(2)
                assert np.abs(Y[:, k] - want).max() <= 1e-15
            if m == 0:
                assert np.abs(Y[:, k] - R[:, k]).max() == 0.0


def test_appendix_b_rotations(oracle_mod):
    """Eq. B2, B4, B5: R_l^{m} from R_l^{-m} at rotated (x, y)."""
    pts = unit_vectors(600, 18)
    x, y, z = pts.T
    R = oracle_mod.real(pts, 9)
    for l in range(1, 10):
        for m in range(1, l + 1):
            a = np.pi / (2 * m)                                                    # B2
            rot = np.stack([np.cos(a) * x - np.sin(a) * y, np.sin(a) * x + np.cos(a) * y, z], axis=1)
            assert np.abs(oracle_mod.real(rot, l)[:, k_of(l, -m)] - R[:, k_of(l, m)]).max() <= 2e-14
            if m % 2 == 1:                                                          # B4
                n = (m - 1) // 2
                rot = np.stack([-y, x, z], axis=1)
                assert np.abs((-1) ** n * oracle_mod.real(rot, l)[:, k_of(l, -m)] - R[:, k_of(l, m)]).max() <= 2e-14
            if m % 4 == 2:                                                          # B5
                n = (m // 2 - 1) // 2
                rot = np.stack([(x - y) / np.sqrt(2), (x + y) / np.sqrt(2), z], axis=1)
                assert np.abs((-1) ** n * oracle_mod.real(rot, l)[:, k_of(l, -m)] - R[:, k_of(l, m)]).max() <= 2e-14


# ----------------------------------------------------------------------------- library routines
def test_against_scipy_sph_harm_y(oracle_mod):
    from scipy.special import sph_harm_y

    pts = unit_vectors(2000, 19) * 2.0
    r = np.linalg.norm(pts, axis=1)
    th, ph = np.arccos(pts[:, 2] / r), np.arctan2(pts[:, 1], pts[:, 0])
    keep = np.sin(th) > 0.05  # the fp64 library loses accuracy near the poles; the oracle does not
    Y = oracle_mod.complex_(pts, 9)
    for l in range(10):
        for m in range(-l, l + 1):
            assert np.abs(Y[keep, k_of(l, m)] - sph_harm_y(l, m, th[keep], ph[keep])).max() <= 5e-14, (l, m)


def test_against_mpmath_including_near_poles(oracle_mod):
    """mpmath.spherharm at 40 digits: an independent arbitrary-precision routine; includes points
    with sin(theta) down to 1e-9, where an fp64 Eq. 5 evaluation would be off by > 1e-12."""
    import mpmath

    mpmath.mp.dps = 40
    rng = np.random.default_rng(20)
    pts = list(unit_vectors(6, 21))
    for s in (1e-2, 2.4e-4, 1e-5, 1e-7, 1e-9):
        phi = rng.uniform(-np.pi, np.pi)
        for sign in (1.0, -1.0):
            pts.append(np.array([s * np.cos(phi), s * np.sin(phi), sign * 1.0]))
    pts = np.array(pts)
    Y = oracle_mod.complex_(pts, 9)
    R = oracle_mod.real(pts, 9)
    worst = 0.0
    for i, (x, y, z) in enumerate(pts):
        X, Yc, Z = mpmath.mpf(float(x)), mpmath.mpf(float(y)), mpmath.mpf(float(z))
        rr = mpmath.sqrt(X * X + Yc * Yc + Z * Z)
        theta, phi = mpmath.acos(Z / rr), mpmath.atan2(Yc, X)
        for l in range(10):
            for m in range(0, l + 1):
                ref = mpmath.spherharm(l, m, theta, phi)
                got = Y[i, k_of(l, m)]
                worst = max(worst, abs(complex(ref) - got))
                if m > 0:  # Eq. 6 in terms of Y_l^{m}: R^{+m} = sqrt2 (-1)^m Re Y, R^{-m} = sqrt2 (-1)^m Im Y
                    worst = max(worst, abs(float(mpmath.sqrt(2) * (-1) ** m * ref.real) - R[i, k_of(l, m)]))
                    worst = max(worst, abs(float(mpmath.sqrt(2) * (-1) ** m * ref.imag) - R[i, k_of(l, -m)]))
    assert worst <= 2e-15, worst


def test_theta_modes_agree_away_from_poles(oracle_mod):
    pts = unit_vectors(500, 22)
    a = oracle_mod.real(pts, 9)
    oracle_mod.set_theta_mode(1)
    try:
        b = oracle_mod.real(pts, 9)
    finally:
        oracle_mod.set_theta_mode(0)
    assert np.abs(a - b).max() <= 1e-15


# ----------------------------------------------------------------------------- special points
def test_origin_convention(oracle_mod):
    """at r = 0 every harmonic is 0 except l = 0."""
    z3 = np.array([[0.0, 0.0, 0.0], [-0.0, 0.0, -0.0]])
    R = oracle_mod.real(z3, 9)
    Y = oracle_mod.complex_(z3, 9)
    S = oracle_mod.spinor(z3, 9)
    c = 1 / np.sqrt(4 * np.pi)
    assert np.all(R[:, 1:] == 0) and np.all(Y[:, 1:] == 0)
    assert np.allclose(R[:, 0], c, atol=1e-16) and np.allclose(Y[:, 0], c, atol=1e-16)
    # l = 0, j = 1/2: m_j = -1/2 -> (0, Y00), m_j = +1/2 -> (Y00, 0); everything else 0
    assert np.allclose(S[:, 0], [0, c], atol=1e-16) and np.allclose(S[:, 1], [c, 0], atol=1e-16)
    assert np.all(S[:, 2:] == 0)


def test_poles_and_axes(oracle_mod):
    pts = np.array([[0, 0, 2.0], [0, 0, -0.5], [3.0, 0, 0], [0, -1.0, 0]])
    R = oracle_mod.real(pts, 9)
    for l in range(10):
        K0 = np.sqrt((2 * l + 1) / (4 * np.pi))
        assert abs(R[0, k_of(l, 0)] - K0) <= 1e-15 and abs(R[1, k_of(l, 0)] - (-1) ** l * K0) <= 1e-15
        for m in range(1, l + 1):
            assert R[0, k_of(l, m)] == 0 and R[0, k_of(l, -m)] == 0
            # south pole: theta = pi is not exactly representable in long double, sin(theta) ~ 5e-20
            assert abs(R[1, k_of(l, m)]) <= 1e-18 and abs(R[1, k_of(l, -m)]) <= 1e-18
            assert abs(R[2, k_of(l, -m)]) <= 1e-18          # sin(m*0) = 0 on the +x axis


def test_spinor_hand_cases(oracle_mod):
    """Eq. 7 by hand for l = 0 and l = 1."""
    pts = unit_vectors(50, 23)
    Y = oracle_mod.complex_(pts, 1)
    S = oracle_mod.spinor(pts, 1)
    ix = oracle_mod.index_spinor
    y00, y1m, y10, y1p = Y[:, 0], Y[:, 1], Y[:, 2], Y[:, 3]
    s3 = np.sqrt(3.0)

    def chk(l, twoj, twomj, up, dn):
        s = S[:, ix(l, twoj, twomj)]
        assert np.abs(s[:, 0] - up).max() <= 1e-15 and np.abs(s[:, 1] - dn).max() <= 1e-15, (l, twoj, twomj)

    chk(0, 1, 1, y00, 0 * y00)
    chk(0, 1, -1, 0 * y00, y00)
    # l = 1, j = 1/2 (lower sign): (-sqrt(l - mj + 1/2) Y^{mj-1/2}, sqrt(l + mj + 1/2) Y^{mj+1/2}) / sqrt 3
    chk(1, 1, 1, -y10 / s3, np.sqrt(2) * y1p / s3)
    chk(1, 1, -1, -np.sqrt(2) * y1m / s3, y10 / s3)
    # l = 1, j = 3/2 (upper sign): (sqrt(l + mj + 1/2) Y^{mj-1/2}, sqrt(l - mj + 1/2) Y^{mj+1/2}) / sqrt 3
    chk(1, 3, 3, y1p, 0 * y1p)
    chk(1, 3, 1, np.sqrt(2) * y10 / s3, y1p / s3)
    chk(1, 3, -1, y1m / s3, np.sqrt(2) * y10 / s3)
    chk(1, 3, -3, 0 * y1m, y1m)


def test_spinor_index_is_a_bijection(oracle_mod):
    seen = []
    for l in range(10):
        for twoj in (2 * l - 1, 2 * l + 1):
            if twoj < 1:
                continue
            for twomj in range(-twoj, twoj + 1, 2):
                seen.append(oracle_mod.index_spinor(l, twoj, twomj))
    assert seen == list(range(200))


def test_imaginary_residue_of_eq6_vanishes(oracle_mod):
    oracle_mod.reset_imag_residue()
    oracle_mod.real(unit_vectors(2000, 24), 9)
    assert oracle_mod.max_imag_residue() <= 1e-18


def test_bad_arguments(oracle_mod):
    with pytest.raises(ValueError):
        oracle_mod.real(np.zeros((1, 3)), 33)  # the oracle's cap (32) covers the l > 9 extension
    with pytest.raises(ValueError):
        oracle_mod.real(np.zeros((1, 3)), -1)
    assert oracle_mod.real(np.zeros((0, 3)), 3).shape == (0, 16)


def test_spinor_weights_against_sympy_clebsch_gordan(oracle_mod):
    """Eq. 7 is the coupling of Y_l^{m_j -+ 1/2} with the spin-1/2 basis states: its weights must be the
    Clebsch-Gordan coefficients <l m_l 1/2 m_s | j m_j> (Condon-Shortley convention).  sympy's CG is an independent
    library routine; with the separately pinned Y_l^m this pins every spinor component, signs included."""
    from sympy import Rational
    from sympy.physics.quantum.cg import CG

    pts = unit_vectors(40, 25) * 1.7
    Y = oracle_mod.complex_(pts, 9)
    S = oracle_mod.spinor(pts, 9)
    half = Rational(1, 2)
    worst = 0.0
    for l in range(10):
        for twoj in (2 * l - 1, 2 * l + 1):
            if twoj < 1:
                continue
            j = Rational(twoj, 2)
            for twomj in range(-twoj, twoj + 1, 2):
                mj = Rational(twomj, 2)
                m_up, m_dn = int(mj - half), int(mj + half)
                cu = float(CG(l, m_up, half, half, j, mj).doit()) if abs(m_up) <= l else 0.0
                cd = float(CG(l, m_dn, half, -half, j, mj).doit()) if abs(m_dn) <= l else 0.0
                up = cu * Y[:, k_of(l, m_up)] if abs(m_up) <= l else 0 * Y[:, 0]
                dn = cd * Y[:, k_of(l, m_dn)] if abs(m_dn) <= l else 0 * Y[:, 0]
                s = S[:, oracle_mod.index_spinor(l, twoj, twomj)]
                worst = max(worst, np.abs(s[:, 0] - up).max(), np.abs(s[:, 1] - dn).max())
    assert worst <= 2e-16, worst
