#!/usr/bin/env python3
"""Build-time generator: closed forms -> factorized CUDA polynomial code (csrc/sh_generated.cuh).

What the paper did by hand with a CAS script and Wolfram Alpha (canonical
polynomial -> factorize -> use x^2+y^2 = 1-z^2 -> roots), this script does from closed forms in
arbitrary precision (mpmath, 60 digits), for every (l, m), 0 <= m <= l <= 9:

  R_l^0    = K_l^0 P_l(z)                         K_l^m = sqrt((2l+1)/(4 pi) (l-m)!/(l+m)!)   (Eq. 5)
  R_l^{+m} = sqrt2 K_l^m Q_l^m(z) C_m(x, y)       Q_l^m = d^m P_l / dz^m                       (Eq. 6)
  R_l^{-m} = sqrt2 K_l^m Q_l^m(z) S_m(x, y)       C_m + i S_m = (x + i y)^m
  Y_l^{+m} = (-1)^m K_l^m Q_l^m (C_m + i S_m),    Y_l^{-m} = K_l^m Q_l^m (C_m - i S_m)         (Eq. 5, 10)

in the normalized coordinates x = x/r, y = y/r, z = z/r (Eq. 8).  Every polynomial is emitted in the
paper's fully factorized form with the root-pair function p(a, b) = (a - b)(a + b) of Eq. 16
(PAPER.md lines 118-122):

  Q_l^m(z) = lead_lm * z^((l-m) mod 2) * prod_i p(z, rho_i)        rho_i: positive roots, all in (0, 1)
  S_m      = y * prod_{k=1}^{(m-1)/2} p(tan(k pi/m) x, y)                          (m odd)
  C_m      = (-1)^((m-1)/2) * x * prod_k p(tan(k pi/m) y, x)                       (m odd;  Eq. B4)
  S_m      = m x y * prod_{k=1}^{m/2-1} p(tan(k pi/m) x, y)                        (m even)
  C_m      = prod_{k=0}^{m/2-1} p(tan((2k+1) pi/(2m)) x, y)                        (m even)

Nothing numeric is copied from PAPER.md (its printed roots contain typos): all
roots and constants are computed here and printed with 17 significant digits.  Before writing the
file the script re-evaluates every emitted product in mpmath against the closed form it came from
(Legendre derivatives via exact rational coefficients AND mpmath's own legendre(); (x+iy)^m) and
aborts on any mismatch > 1e-45.

The spinor table follows Eq. 7: for l = j -+ 1/2,
  up   = +-sqrt(l +- m_j + 1/2)/sqrt(2l+1) * Y_l^{m_j-1/2},   down = sqrt(l -+ m_j + 1/2)/sqrt(2l+1) * Y_l^{m_j+1/2}.

Beyond the explicit range (the paper's conclusion: "could be easily extended using recurrence
relationships for higher values of l"), for 10 <= l <= 32 the script emits the coefficient tables of the upward
recurrence in l at fixed m for the normalized polar factors q_lm = f_m K_l^m Q_l^m(z) (f_0 = 1, f_m = sqrt2):

  q_lm = A_lm (z q_{l-1,m} - B_lm q_{l-2,m}),   A_lm = sqrt((4l^2-1)/(l^2-m^2)),  B_lm = sqrt(((l-1)^2-m^2)/(4(l-1)^2-1))
  q_ll = sqrt((2l+1)/(2l)) q_{l-1,l-1}                                                        (l >= 2)

seeded by the explicit l = 8, 9 block, and checks them against the closed forms above before writing.

This file shares no code with oracle/ (which never evaluates a polynomial in x, y, z).
Usage: python generate.py [output.cuh]
"""
from __future__ import annotations

import os
import sys
from fractions import Fraction
from math import comb, factorial

import mpmath as mp

mp.mp.dps = 60
LMAX = 9
LMAX_EXT = 32   # reach of the recurrence extension


# ----------------------------------------------------------------------------- closed forms
def legendre_coeffs(l: int) -> list[Fraction]:
    """Exact coefficients c[k] of P_l(z) = sum_k c[k] z^k (explicit sum formula)."""
    c = [Fraction(0)] * (l + 1)
    for k in range(l // 2 + 1):
        c[l - 2 * k] = Fraction((-1) ** k * comb(l, k) * comb(2 * l - 2 * k, l), 2**l)
    return c


def derivative(c: list[Fraction], m: int) -> list[Fraction]:
    for _ in range(m):
        c = [k * c[k] for k in range(1, len(c))] or [Fraction(0)]
    return c


def q_poly(l: int, m: int) -> list[Fraction]:
    """Q_l^m(z) = d^m P_l / dz^m, exact coefficients."""
    return derivative(legendre_coeffs(l), m)


def q_factorization(l: int, m: int):
    """Q_l^m = lead * z^par * prod_i (z^2 - rho_i^2): returns (lead: Fraction, par, [rho_i] mp.mpf)."""
    c = q_poly(l, m)
    deg = l - m
    par = deg % 2
    lead = c[deg]
    assert lead == Fraction(factorial(2 * l), 2**l * factorial(l) * factorial(deg))
    # polynomial in w = z^2 after removing z^par, made monic
    w = [c[par + 2 * i] / lead for i in range(deg // 2 + 1)]
    roots = []
    if len(w) > 1:
        rts = mp.polyroots([mp.mpf(x.numerator) / mp.mpf(x.denominator) for x in reversed(w)], maxsteps=500, extraprec=400)
        for r in rts:
            assert abs(mp.im(r)) < mp.mpf(10) ** -50 and 0 < mp.re(r) < 1, (l, m, r)
            roots.append(mp.sqrt(mp.re(r)))
        roots.sort()
    return lead, par, roots


def q_monic_in_z2(l: int, m: int) -> list[Fraction]:
    """Qhat_l^m / z^par as a MONIC polynomial in w = z^2: exact coefficients, ascending powers (last one is 1)."""
    c = q_poly(l, m)
    deg = l - m
    par = deg % 2
    return [c[par + 2 * i] / c[deg] for i in range(deg // 2 + 1)]


def K(l: int, m: int):
    return mp.sqrt(mp.mpf(2 * l + 1) / (4 * mp.pi) * mp.mpf(factorial(l - m)) / mp.mpf(factorial(l + m)))


def azimuthal_roots(m: int):
    """(S roots t: p(t x, y) factors, C roots) per the docstring; for odd m the C roots are the S roots
    used with x and y swapped."""
    if m % 2 == 1:
        ts = [mp.tan(k * mp.pi / m) for k in range(1, (m - 1) // 2 + 1)]
        return ts, ts
    ts = [mp.tan(k * mp.pi / m) for k in range(1, m // 2)]
    tc = [mp.tan((2 * k + 1) * mp.pi / (2 * m)) for k in range(m // 2)]
    return ts, tc


# ----------------------------------------------------------------------------- self-check
def p(a, b):
    return (a - b) * (a + b)


def self_check():
    tol = mp.mpf(10) ** -45
    pts = [(mp.mpf("0.3141"), mp.mpf("-0.7713")), (mp.mpf("-0.91"), mp.mpf("0.05")), (mp.mpf("0.002"), mp.mpf("0.9"))]
    for m in range(1, LMAX + 1):
        ts, tc = azimuthal_roots(m)
        for x, y in pts:
            ref = (x + 1j * y) ** m
            if m % 2 == 1:
                s = y
                for t in ts:
                    s *= p(t * x, y)
                c = (-1) ** ((m - 1) // 2) * x
                for t in tc:
                    c *= p(t * y, x)
            else:
                s = m * x * y
                for t in ts:
                    s *= p(t * x, y)
                c = mp.mpf(1)
                for t in tc:
                    c *= p(t * x, y)
            assert abs(s - mp.im(ref)) < tol and abs(c - mp.re(ref)) < tol, ("azimuthal", m)
    for l in range(LMAX + 1):
        for m in range(l + 1):
            lead, par, roots = q_factorization(l, m)
            for z in (mp.mpf("0.123456789"), mp.mpf("-0.87"), mp.mpf("0.5")):
                val = mp.mpf(lead.numerator) / lead.denominator * z**par
                for r in roots:
                    val *= p(z, r)
                ref = mp.diff(lambda t: mp.legendre(l, t), z, m) if m else mp.legendre(l, z)
                assert abs(val - ref) < mp.mpf(10) ** -25 * max(1, abs(ref)), ("polar/mpmath", l, m)
                exact = sum((mp.mpf(c.numerator) / c.denominator) * z**k for k, c in enumerate(q_poly(l, m)))
                assert abs(val - exact) < tol * max(1, abs(exact)), ("polar/exact", l, m)
                # the Horner form in z^2 emitted for the FP64-bound consumer (PolarHorner)
                w = q_monic_in_z2(l, m)
                acc = mp.mpf(1)
                for cf in reversed(w[:-1]):
                    acc = acc * z * z + mp.mpf(cf.numerator) / cf.denominator
                hv = mp.mpf(lead.numerator) / lead.denominator * z**par * acc
                assert abs(hv - exact) < tol * max(1, abs(exact)), ("polar/horner", l, m)


# ----------------------------------------------------------------------------- recurrence extension, l > 9
def rec_a(l: int, m: int):
    return mp.sqrt(mp.mpf(4 * l * l - 1) / mp.mpf(l * l - m * m))


def rec_b(l: int, m: int):
    return mp.sqrt(mp.mpf((l - 1) ** 2 - m * m) / mp.mpf(4 * (l - 1) ** 2 - 1))


def rec_sect(l: int):
    return mp.sqrt(mp.mpf(2 * l + 1) / mp.mpf(2 * l))


def self_check_recurrence():
    """q_lm = f_m K_l^m Q_l^m(z) from the exact Legendre coefficients obeys the emitted recurrences for every l <= LMAX_EXT."""
    tol = mp.mpf(10) ** -40

    def q(l, m, z):
        if m > l:
            return mp.mpf(0)
        val = sum((mp.mpf(c.numerator) / c.denominator) * z**k for k, c in enumerate(q_poly(l, m)))
        return (mp.sqrt(2) if m else 1) * K(l, m) * val

    for z in (mp.mpf("0.31"), mp.mpf("-0.95")):
        for l in range(2, LMAX_EXT + 1):
            assert abs(q(l, l, z) - rec_sect(l) * q(l - 1, l - 1, z)) < tol * abs(q(l, l, z)), ("sectoral", l)
            for m in range(l):
                want = q(l, m, z)
                got = rec_a(l, m) * (z * q(l - 1, m, z) - rec_b(l, m) * q(l - 2, m, z))
                assert abs(got - want) < tol * max(1, abs(want)), ("recurrence", l, m)


# ----------------------------------------------------------------------------- emission
def scaled(t, var: str) -> str:
    """t * var, with the factor dropped when the root is exactly 1 (tan(pi/4))."""
    return var if abs(t - 1) < mp.mpf(10) ** -50 else f"{lit(t)} * {var}"


def lit(v) -> str:
    """17 significant digits: round-trips fp64 exactly; cast to T (9 digits are enough for fp32)."""
    return "T(" + mp.nstr(mp.mpf(v), 17, strip_zeros=False, min_fixed=-5, max_fixed=5) + ")"


def dlit(v) -> str:
    return mp.nstr(mp.mpf(v), 17, strip_zeros=False, min_fixed=-5, max_fixed=5)


def emit() -> str:
    o = []
    w = o.append
    w("// GENERATED FILE -- do not edit.  Written by paper_2510_05282_b200/gen/generate.py from closed forms")
    w("// (mpmath, 60 digits); see that script's docstring for the formulas and the paper citations.")
    w("// Factorized real/complex/spinor spherical-harmonic building blocks, l <= 9 (arxiv 2510.05282,")
    w("// Eq. 5-7, Eq. 16, Appendix B/C), in normalized Cartesian coordinates x, y, z (Eq. 8).")
    w("#pragma once")
    w("")
    w("#ifndef SHGEN_FN")
    w("#define SHGEN_FN __host__ __device__ __forceinline__")
    w("#endif")
    w("")
    w("namespace shgen {")
    w("")
    w(f"constexpr int LMAX_CAP = {LMAX};")
    w("")
    w("// Eq. 16 (PAPER.md line 120): factor of a +-root pair; NOT a*a - b*b (round-off when |a| ~ |b|).")
    w("template <typename T> SHGEN_FN T p(T a, T b) { return (a - b) * (a + b); }")
    w("")
    w("// ---- azimuthal factors: C_m + i S_m = (x + i y)^m as products over root pairs ----")
    w("template <int M, typename T> struct Azimuthal;")
    w("template <typename T> struct Azimuthal<0, T> { static SHGEN_FN void eval(T, T, T& c, T& s) { c = T(1); s = T(0); } };")
    for m in range(1, LMAX + 1):
        ts, tc = azimuthal_roots(m)
        w(f"template <typename T> struct Azimuthal<{m}, T> {{")
        w("    static SHGEN_FN void eval(T x, T y, T& c, T& s) {")
        if m % 2 == 1:
            sgn = "-" if ((m - 1) // 2) % 2 else ""
            s_expr = "y" + "".join(f" * p({scaled(t, 'x')}, y)" for t in ts)
            c_expr = f"{sgn}x" + "".join(f" * p({scaled(t, 'y')}, x)" for t in tc)
            w(f"        s = {s_expr};")
            w(f"        c = {c_expr};")
        else:
            s_expr = f"T({m}) * x * y" + "".join(f" * p({scaled(t, 'x')}, y)" for t in ts)
            c_expr = " * ".join(f"p({scaled(t, 'x')}, y)" for t in tc)
            w(f"        s = {s_expr};")
            w(f"        c = {c_expr};")
        w("    }")
        w("};")
    w("")
    w("// ---- polar factors: Qhat_l^m(z) = Q_l^m(z) / lead_lm = z^((l-m)%2) prod_i p(z, rho_i) ----")
    w("template <int L, int M, typename T> struct Polar;")
    for l in range(LMAX + 1):
        for m in range(l + 1):
            lead, par, roots = q_factorization(l, m)
            terms = (["z"] if par else []) + [f"p(z, {lit(r)})" for r in roots]
            body = " * ".join(terms) if terms else "T(1)"
            arg = "T z" if terms else "T"
            w(f"template <typename T> struct Polar<{l}, {m}, T> {{ static SHGEN_FN T eval({arg}) {{ return {body}; }} }};")
    w("")
    w("// ---- the same polar factors in Horner form in t = z^2 (the paper's fallback form, PAPER.md line 124), monic: ----")
    w("// Qhat_l^m(z) = z^((l-m)%2) (((t + c_{k-1}) t + c_{k-2}) t + ... + c_0).  One FMA per root pair instead of four")
    w("// instructions; not used by the sh_* calls (PAPER.md lines 93, 122: accuracy), offered to the FP64-bound projection.")
    w("template <int L, int M, typename T> struct PolarHorner;")
    for l in range(LMAX + 1):
        for m in range(l + 1):
            cs = q_monic_in_z2(l, m)
            par = (l - m) % 2
            body = None
            for cf in reversed(cs[:-1]):
                c_lit = "T(" + dlit(mp.mpf(cf.numerator) / cf.denominator) + ")"
                body = f"(t + {c_lit})" if body is None else f"({body} * t + {c_lit})"
            if body is None:
                body = "z" if par else "T(1)"
            elif par:
                body = f"z * {body}"
            w(f"template <typename T> struct PolarHorner<{l}, {m}, T> {{ static SHGEN_FN T eval(T z, T t) {{ (void)z; (void)t; return {body}; }} }};")
    w("")
    w("// ---- constants (fp64; cast at the point of use) ----")
    w("// A_REAL[l][m]: R_l^0 = A Qhat,  R_l^{+-m} = A Qhat {C_m, S_m}   (A = sqrt2 K_l^m lead_lm, m > 0)")
    w("// B_CPLX[l][m]: Y_l^{-m} = B Qhat (C_m - i S_m),  Y_l^{+m} = (-1)^m B Qhat (C_m + i S_m)   (B = K_l^m lead_lm)")
    for name, fac in (("A_REAL", lambda m: mp.sqrt(2) if m else mp.mpf(1)), ("B_CPLX", lambda m: mp.mpf(1))):
        w(f"constexpr double {name}[{LMAX + 1}][{LMAX + 1}] = {{")
        for l in range(LMAX + 1):
            row = []
            for m in range(LMAX + 1):
                if m <= l:
                    lead, _, _ = q_factorization(l, m)
                    row.append(dlit(fac(m) * K(l, m) * mp.mpf(lead.numerator) / lead.denominator))
                else:
                    row.append("0.0")
            w("    {" + ", ".join(row) + "},")
        w("};")
    w("")
    w("// Y_0^0 = R_0^0 = 1/sqrt(4 pi): the only non-zero harmonic at r = 0 (PAPER.md line 60)")
    w(f"constexpr double Y00 = {dlit(1 / mp.sqrt(4 * mp.pi))};")
    w("")
    w("// ---- spinor table, Eq. 7: entry s = 2 l^2 + (j = l-1/2 ? m_j + j : 2l + m_j + j) ----")
    w("// (up, down) = (CU * Y_l^{M_UP}, CD * Y_l^{M_DN}); a component whose m is out of range has C* = 0.")
    w("struct SpinorEntry { int l, twoj, twomj, m_up, m_dn; double cu, cd; };")
    ents = []
    for l in range(LMAX + 1):
        for sign in (-1, +1):
            twoj = 2 * l + sign
            if twoj < 1:
                continue
            for twomj in range(-twoj, twoj + 1, 2):
                mj = mp.mpf(twomj) / 2
                pref = 1 / mp.sqrt(2 * l + 1)
                cu = sign * mp.sqrt(l + sign * mj + mp.mpf(1) / 2) * pref
                cd = mp.sqrt(l - sign * mj + mp.mpf(1) / 2) * pref
                m_up, m_dn = (twomj - 1) // 2, (twomj + 1) // 2
                if abs(m_up) > l:
                    assert abs(cu) < mp.mpf(10) ** -50
                    cu = mp.mpf(0)
                if abs(m_dn) > l:
                    assert abs(cd) < mp.mpf(10) ** -50
                    cd = mp.mpf(0)
                ents.append((l, twoj, twomj, m_up, m_dn, cu, cd))
    assert len(ents) == 2 * (LMAX + 1) ** 2
    w(f"constexpr SpinorEntry SPINOR[{len(ents)}] = {{")
    for (l, twoj, twomj, m_up, m_dn, cu, cd) in ents:
        w(f"    {{{l}, {twoj}, {twomj}, {m_up}, {m_dn}, {dlit(cu)}, {dlit(cd)}}},")
    w("};")
    w("")
    w("// ---- recurrence extension, 10 <= l <= 32 (PAPER.md line 183): q_lm = REC_A (z q_{l-1,m} - REC_B q_{l-2,m}), m < l;")
    w("// q_ll = REC_SECT[l] q_{l-1,l-1}; q_lm = f_m K_l^m Q_l^m(z), seeded by the explicit l = 8, 9 block.  Index [l * 33 + m].")
    w(f"constexpr int LMAX_EXT = {LMAX_EXT};")
    w("#ifndef SHGEN_TABLE")
    w("#define SHGEN_TABLE static const")
    w("#endif")
    n1 = LMAX_EXT + 1
    for name, fn in (("REC_A", rec_a), ("REC_B", rec_b)):
        w(f"SHGEN_TABLE double {name}[{n1} * {n1}] = {{")
        for l in range(n1):
            row = [dlit(fn(l, m)) if (l >= 2 and m < l) else "0.0" for m in range(n1)]
            w("    " + ", ".join(row) + ",")
        w("};")
    w(f"SHGEN_TABLE double REC_SECT[{n1}] = {{" + ", ".join(dlit(rec_sect(l)) if l >= 2 else "0.0" for l in range(n1)) + "};")
    w("")
    w("}  // namespace shgen")
    w("")
    return "\n".join(o)


def main(argv):
    here = os.path.dirname(os.path.abspath(__file__))
    out = argv[1] if len(argv) > 1 else os.path.join(here, "..", "csrc", "sh_generated.cuh")
    self_check()
    self_check_recurrence()
    text = emit()
    out = os.path.abspath(out)
    if not os.path.exists(out) or open(out).read() != text:
        with open(out, "w") as f:
            f.write(text)
    return out


if __name__ == "__main__":
    print(main(sys.argv))
