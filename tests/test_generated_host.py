"""GPU-less check of the generator's output: paper_2510_05282_b200/csrc/sh_generated.cuh
compiled as plain host C++ (baseline/sh_cpu_method.cpp) and evaluated at random unit vectors, against
  (i)  the oracle (Eq. 5 + Eq. 6, long double), for every l <= 9, both polynomial forms (root-pair products, Eq. 16
       P:118-122; Horner in z^2), both layouts, Cartesian and normalized input, the r = 0 convention;
  (ii) the 47 formulas of Appendix C that are correct as printed (tests/appendix_c.py).
A generator regression (a wrong root, constant, sign or index) fails here without a B200.  The harness links nothing
from oracle/ and is not reachable from the product path (see the header of baseline/sh_cpu_method.cpp).
"""
import numpy as np
import pytest

from appendix_c import FORMULAS


@pytest.fixture(scope="module")
def host():
    import baseline

    baseline.build()
    return baseline


def unit_vectors(n, seed):
    g = np.random.default_rng(seed).standard_normal((n, 3))
    return g / np.linalg.norm(g, axis=1)[:, None]


@pytest.mark.parametrize("form,tol", [("factorized", 3e-14), ("horner", 1e-13)])
def test_generated_formulas_against_the_oracle(host, oracle_mod, form, tol):
    u = unit_vectors(4003, 21)   # 500 full vectors of 8 points and a ragged tail of 3
    for lmax in range(10):
        want = oracle_mod.real(u, lmax)
        for normalized in (True, False):
            pts = u if normalized else u * np.random.default_rng(22).uniform(1e-3, 1e2, (len(u), 1))
            got_aos = host.real(pts, lmax, "aos", normalized=normalized, form=form)
            got_soa = host.real(pts, lmax, "soa", normalized=normalized, form=form)
            assert got_aos.shape == want.shape and got_soa.shape == want.T.shape
            assert np.array_equal(got_aos, got_soa.T)
            assert np.abs(got_aos - want).max() <= tol, (lmax, normalized)


def test_generated_formulas_against_appendix_c_as_printed(host):
    u = unit_vectors(4000, 11)
    x, y, z = u.T
    got = host.real(u, 9, "aos", normalized=True)
    horner = host.real(u, 9, "aos", normalized=True, form="horner")
    assert len(FORMULAS) == 47
    for (l, m), f in FORMULAS.items():
        k = l * (l + 1) + m
        assert np.abs(got[:, k] - f(x, y, z)).max() <= 3e-14, (l, m)
        assert np.abs(horner[:, k] - f(x, y, z)).max() <= 1e-13, (l, m)


def test_generated_formulas_special_points(host, oracle_mod):
    """r = 0, poles and axes: the polynomials alone do not vanish at the origin, the
    convention must."""
    from paper_2510_05282_b200 import inputs

    pts = inputs.config1_cube(100, seed=3)   # 100 random points + the 8 specials
    got = host.real(pts, 9, "aos")
    assert np.abs(got - oracle_mod.real(pts, 9)).max() <= 3e-14
    for row in (100, 107):   # the origin, as +0 and as -0
        assert got[row, 0] == pytest.approx(1 / np.sqrt(4 * np.pi), abs=1e-16) and np.all(got[row, 1:] == 0)
    assert np.all(got[101:103, 1:4] == np.array([[0, 1, 0], [0, -1, 0]]) * np.sqrt(3 / (4 * np.pi)))   # poles: R_1^0 = +-sqrt(3/4pi), R_1^{+-1} = 0


def test_accumulate_matches_the_stored_values(host):
    u = unit_vectors(4096, 5) * 3.0
    assert host.accumulate_l9(u) == pytest.approx(host.real(u, 9).sum(), rel=1e-12)
