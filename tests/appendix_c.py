"""Appendix C of the paper, restated: the printed factorized formulas
for R_l^m, m <= 0, in normalized Cartesian coordinates.  Used ONLY as an oracle pin
(tests/test_oracle_pins.py) -- the CUDA path's generator derives its own constants from closed
forms and copies nothing from here.

Only formulas that SURVEY.md section 8c #15 lists as correct exactly as printed are included (plus the
Horner form of R_8^{-1} and the canonical form of R_9^{-9}); the garbled ones (#6-#14) are
left out rather than repaired, so that every entry is the paper's own text.
Each entry: (l, m) -> function of numpy arrays x, y, z with x^2+y^2+z^2 = 1.
"""
import numpy as np

pi = np.pi
sqrt = np.sqrt


def p(a, b):
    """Eq. 16: p(a, b) = (a - b)(a + b)."""
    return (a - b) * (a + b)


T7 = (0.481574618807528644332162353056970575219,
      1.253960337662703837570910978336464443221,
      4.381286267534823072404689085032695444150)

FORMULAS = {
    # l = 0, 1, 2
    (0, 0): lambda x, y, z: 1 / sqrt(4 * pi) + 0 * x,
    (1, -1): lambda x, y, z: sqrt(3 / (4 * pi)) * y,
    (1, 0): lambda x, y, z: sqrt(3 / (4 * pi)) * z,
    (2, -2): lambda x, y, z: 0.5 * sqrt(15 / pi) * x * y,
    (2, -1): lambda x, y, z: 0.5 * sqrt(15 / pi) * y * z,
    (2, 0): lambda x, y, z: 0.25 * sqrt(5 / pi) * p(sqrt(3) * z, 1),
    # l = 3   (line 262)
    (3, -3): lambda x, y, z: 1 / 8 * sqrt(70 / pi) * y * p(sqrt(3) * x, y),
    (3, -2): lambda x, y, z: 0.5 * sqrt(105 / pi) * x * y * z,
    (3, -1): lambda x, y, z: 1 / 8 * sqrt(42 / pi) * y * p(sqrt(5) * z, 1),
    (3, 0): lambda x, y, z: 0.25 * sqrt(7 / pi) * p(sqrt(5) * z, sqrt(3)) * z,
    # l = 4   (line 266)
    (4, -4): lambda x, y, z: 0.75 * sqrt(35 / pi) * x * y * p(x, y),
    (4, -3): lambda x, y, z: 3 / 8 * sqrt(70 / pi) * y * p(sqrt(3) * x, y) * z,
    (4, -2): lambda x, y, z: 0.75 * sqrt(5 / pi) * x * y * p(sqrt(7) * z, 1),
    (4, -1): lambda x, y, z: 3 / 8 * sqrt(10 / pi) * y * z * p(sqrt(7) * z, sqrt(3)),
    (4, 0): lambda x, y, z: 105 / 16 * sqrt(1 / pi) * p(sqrt((3 + 2 * sqrt(6 / 5)) / 7), z)
    * p(sqrt((3 - 2 * sqrt(6 / 5)) / 7), z),
    # l = 5   (line 270; R_5^0 is garbled there, reading #6, and is left out)
    (5, -5): lambda x, y, z: 30 / 64 * sqrt(154 / pi) * y * p(sqrt(1 - 2 / sqrt(5)) * y, x)
    * p(sqrt(1 + 2 / sqrt(5)) * y, x),
    (5, -4): lambda x, y, z: 0.75 * sqrt(385 / pi) * p(x, y) * y * z * x,
    (5, -3): lambda x, y, z: 1 / 32 * sqrt(770 / pi) * y * p(y, sqrt(3) * x) * p(1, 3 * z),
    (5, -2): lambda x, y, z: 0.25 * sqrt(1155 / pi) * x * y * p(sqrt(3) * z, 1) * z,
    (5, -1): lambda x, y, z: 21 / 16 * sqrt(165 / pi) * y * p(sqrt((7 - 2 * sqrt(7)) / 21), z)
    * p(sqrt((7 + 2 * sqrt(7)) / 21), z),
    # l = 6   (line 274)
    (6, -6): lambda x, y, z: 1 / 32 * sqrt(6006 / pi) * x * y * p(x, sqrt(3) * y) * p(sqrt(3) * x, y),
    (6, -5): lambda x, y, z: 3 / 32 * sqrt(2002 / pi) * y * z * p(sqrt(5 - 2 * sqrt(5)) * x, y)
    * p(sqrt(5 + 2 * sqrt(5)) * x, y),
    (6, -4): lambda x, y, z: 3 / 8 * sqrt(91 / pi) * x * y * p(x, y) * p(sqrt(11) * z, 1),
    (6, -3): lambda x, y, z: 1 / 32 * sqrt(2730 / pi) * y * z * p(sqrt(3) * x, y) * p(sqrt(11) * z, sqrt(3)),
    (6, -2): lambda x, y, z: 33 / 32 * sqrt(2730 / pi) * x * y * p(sqrt((3 - 4 / sqrt(3)) / 11), z)
    * p(sqrt((3 + 4 / sqrt(3)) / 11), z),
    (6, -1): lambda x, y, z: 33 / 16 * sqrt(273 / pi) * y * z * p(sqrt((15 - 2 * sqrt(15)) / 33), z)
    * p(sqrt((15 + 2 * sqrt(15)) / 33), z),
    (6, 0): lambda x, y, z: 1 / 32 * sqrt(13 / pi) * (z**2 * ((231 * z**2 - 315) * z**2 + 105) - 5),
    # l = 7   (lines 278-286)
    (7, -7): lambda x, y, z: 3 / 64 * sqrt(715 / pi) * y * p(T7[0] * x, y) * p(T7[1] * x, y) * p(T7[2] * x, y),
    (7, -6): lambda x, y, z: 3 / 32 * sqrt(10010 / pi) * x * y * z * p(x, sqrt(3) * y) * p(sqrt(3) * x, y),
    (7, -5): lambda x, y, z: 3 / 64 * sqrt(385 / pi) * y * p(sqrt(13) * z, 1) * p(sqrt(5 - 2 * sqrt(5)) * x, y)
    * p(sqrt(5 + 2 * sqrt(5)) * x, y),
    (7, -4): lambda x, y, z: 3 / 8 * sqrt(385 / pi) * x * y * z * p(x, y) * p(sqrt(13) * z, sqrt(3)),
    (7, -3): lambda x, y, z: 429 / 64 * sqrt(35 / pi) * y * p(sqrt(3) * x, y)
    * p(sqrt((33 - 2 * sqrt(165)) / 143), z) * p(sqrt((33 + 2 * sqrt(165)) / 143), z),  # = Eq. 15
    (7, -2): lambda x, y, z: 429 / 32 * sqrt(70 / pi) * x * y * z * p(sqrt((55 - 4 * sqrt(55)) / 143), z)
    * p(sqrt((55 + 4 * sqrt(55)) / 143), z),
    (7, -1): lambda x, y, z: 1 / 64 * sqrt(105 / pi) * y * (z**2 * ((429 * z**2 - 495) * z**2 + 135) - 5),
    (7, 0): lambda x, y, z: 1 / 32 * sqrt(15 / pi) * z * (-35 + z**2 * (315 + z**2 * (-693 + 429 * z**2))),
    # l = 8   (lines 290-298; R_8^{-5} has a misplaced x-bar, reading #8, left out; R_8^{-1}: Horner form)
    (8, -8): lambda x, y, z: 12 / 128 * sqrt(12155 / pi) * x * y * p(x, y) * p((1 + sqrt(2)) * x, y)
    * p((1 - sqrt(2)) * x, y),
    (8, -7): lambda x, y, z: 3 / 64 * sqrt(12155 / pi) * y * z * p(T7[0] * x, y) * p(T7[1] * x, y) * p(T7[2] * x, y),
    (8, -6): lambda x, y, z: 1 / 64 * sqrt(14586 / pi) * x * y * p(x, sqrt(3) * y) * p(sqrt(3) * x, y)
    * p(sqrt(15) * z, 1),
    (8, -4): lambda x, y, z: 195 / 32 * sqrt(1309 / pi) * x * y * p(x, y) * p(sqrt((13 - 2 * sqrt(26)) / 65), z)
    * p(sqrt((13 + 2 * sqrt(26)) / 65), z),
    (8, -3): lambda x, y, z: 39 / 64 * sqrt(19635 / pi) * y * z * p(sqrt(3) * x, y)
    * p(sqrt((1 - 2 / sqrt(13)) / 3), z) * p(sqrt((1 + 2 / sqrt(13)) / 3), z),
    (8, -2): lambda x, y, z: 3 / 64 * sqrt(1190 / pi) * x * y * (z**2 * ((143 * z**2 - 143) * z**2 + 33) - 1),
    (8, -1): lambda x, y, z: 3 / 64 * sqrt(17 / pi) * y * z * (z**2 * ((715 * z**2 - 1001) * z**2 + 385) - 35),
    (8, 0): lambda x, y, z: 1 / 256 * sqrt(17 / pi)
    * ((z**2 * ((6435 * z**2 - 12012) * z**2 + 6930) - 1260) * z**2 + 35),
    # l = 9   (line 302: only the entries printed intact)
    (9, -9): lambda x, y, z: 1 / 512 * sqrt(461890 / pi) * y * p(sqrt(3) * x, y)
    * (3 * x**6 - 27 * x**4 * y**2 + 33 * x**2 * y**4 - y**6),
    (9, -6): lambda x, y, z: 1 / 64 * sqrt(81510 / pi) * x * y * z * p(x, sqrt(3) * y) * p(sqrt(3) * x, y)
    * p(sqrt(17) * z, sqrt(3)),
    (9, -4): lambda x, y, z: 51 / 32 * sqrt(95095 / pi) * x * y * z * p(x, y) * p(sqrt((5 - 2 * sqrt(2)) / 17), z)
    * p(sqrt((5 + 2 * sqrt(2)) / 17), z),
    (9, -3): lambda x, y, z: 1 / 256 * sqrt(43890 / pi) * y * p(sqrt(3) * x, y)
    * (z**2 * ((221 * z**2 - 195) * z**2 + 39) - 1),
}
