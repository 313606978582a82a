/*
 * sh_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU oracle for the real, complex and spin-1/2 spinor
 * spherical harmonics, written from the DEFINITIONS in the paper (arxiv 2510.05282,
 * "SHarmonic"), in `long double` (x87 80-bit on this host):
 *
 *   Eq. 3   theta = acos(z / r)
 *   Eq. 4   phi   = atan2(y, x)
 *   Eq. 5   Y_l^m = (-1)^m sqrt((2l+1)/(4 pi) (l-m)!/(l+m)!) P_l^m(cos theta) e^{i m phi}
 *   Eq. 6   real harmonics R_l^m from Y_l^{+-m}
 *   Eq. 7   spinor harmonics from Y_l^m with Clebsch-Gordan weights
 *   r = 0   all harmonics 0 except l = 0, which is the constant
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this.  It shares NO code, table, constant generator or helper with the CUDA path
 * (paper_2510_05282_b200/csrc, .../gen): that path evaluates generated factorized polynomials in
 * x/r, y/r, z/r; this file goes through the angles, the associated-Legendre recurrence and
 * cos/sin(m phi), exactly as Eq. 3-5 are written.  There is no blocking, fusion or reordering.
 *
 * Readings of the paper taken here:
 *   #1  Eq. 5 prints P_m^l: read as the associated Legendre function of degree l, order m,
 *       WITHOUT the Condon-Shortley phase (the (-1)^m is explicit in Eq. 5).
 *   Negative m in Eq. 5 uses the standard P_l^{-m} = (-1)^m (l-m)!/(l+m)! P_l^m (Arfken, the
 *       paper's ref. 19), so Eq. 10 is a PROPERTY that the tests check, not an input.
 *   #16 r = 0 is the exact test r == 0 (no epsilon).
 *   #18 the acos argument is clamped to [-1, 1].
 *   #19 Eq. 7: upper sign <=> l = j - 1/2, lower sign <=> l = j + 1/2; Y_l^{m'} with |m'| > l is 0.
 *   Near the poles (x^2 + y^2 < 1e-10 r^2) theta = acos(z/r) loses sin(theta) to cancellation
 *       (the paper's own remark on theta -> 0); there the mathematically
 *       identical theta = atan2(hypot(x, y), z) is used.  sh_oracle_set_theta_mode(1) forces the
 *       literal acos everywhere (reported cross-check).
 *
 * Output layouts (all AoS, one point after another):
 *   real    out[i][k]            k = l(l+1)+m                      K = (lmax+1)^2 doubles / point
 *   complex out[i][k][re,im]                                       2K doubles / point
 *   spinor  out[i][s][up.re, up.im, down.re, down.im]              8K doubles / point
 *           s = 2 l^2 + (j = l-1/2 ? m_j + j : 2l + m_j + j)       (l ascending; j = l-1/2 block
 *           of 2l entries, then j = l+1/2 block of 2l+2 entries; m_j ascending)
 *
 * Parity pins: see tests/test_oracle_pins.py (Tables II/III of the paper, Appendix C formulas,
 * l <= 2 closed forms, Unsoeld sums, quadrature orthonormality, symmetries, scipy's sph_harm_y,
 * mpmath's spherharm).  The paper prints no spinor values: the spinor weights and signs are pinned
 * against sympy's Clebsch-Gordan coefficients, plus orthonormality, the sum rule and hand cases.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef long double ld;

/* The paper's explicit formulas stop at l = 9; Eq. 5 itself and the recurrence below hold for
 * every l, and the paper's conclusion proposes going beyond 9 by recurrence.  The cap is 32 so that
 * this oracle can also check that extension (sh_real_ext / sh_complex_ext); nothing in the arithmetic depends on it. */
#define LMAX_CAP 32
#define KMAX ((LMAX_CAP + 1) * (LMAX_CAP + 1))

static const ld PI_L = 3.14159265358979323846264338327950288419716939937510L;

static int g_theta_mode = 0;      /* 0: acos + near-pole atan2 switch; 1: literal acos everywhere */
static int g_threads = 0;         /* 0: OpenMP default */
static double g_max_imag = 0.0;   /* largest |Im| residue seen in Eq. 6 (must be rounding-level) */

void sh_oracle_set_theta_mode(int mode) { g_theta_mode = mode; }
void sh_oracle_set_threads(int t) { g_threads = t; }
double sh_oracle_max_imag_residue(void) { return g_max_imag; }
void sh_oracle_reset_imag_residue(void) { g_max_imag = 0.0; }

int sh_oracle_threads_used(void) {
#ifdef _OPENMP
    return g_threads > 0 ? g_threads : omp_get_max_threads();
#else
    return 1;
#endif
}

static ld factorial(int n) {
    ld f = 1.0L;
    for (int i = 2; i <= n; ++i) f *= (ld)i;
    return f;
}

/* Associated Legendre functions P_l^m(c), 0 <= m <= l <= lmax, WITHOUT Condon-Shortley phase,
 * c = cos(theta), s = sin(theta) >= 0.  Standard upward recurrence in l at fixed m:
 *   P_m^m     = (2m-1)!! s^m
 *   P_{m+1}^m = (2m+1) c P_m^m
 *   (l-m) P_l^m = (2l-1) c P_{l-1}^m - (l+m-1) P_{l-2}^m                                   */
static void assoc_legendre(int lmax, ld c, ld s, ld P[LMAX_CAP + 1][LMAX_CAP + 1]) {
    for (int m = 0; m <= lmax; ++m) {
        ld pmm = 1.0L;
        for (int i = 1; i <= m; ++i) pmm *= (ld)(2 * i - 1) * s;
        P[m][m] = pmm;
        if (m + 1 <= lmax) P[m + 1][m] = (ld)(2 * m + 1) * c * pmm;
        for (int l = m + 2; l <= lmax; ++l)
            P[l][m] = ((ld)(2 * l - 1) * c * P[l - 1][m] - (ld)(l + m - 1) * P[l - 2][m]) / (ld)(l - m);
    }
}

/* Eq. 5 for every l <= lmax and every m = -l..l at the angles (theta, phi).
 * Y[l(l+1)+m] = (re, im). */
static void ylm_angular(int lmax, ld theta, ld phi, ld Yre[KMAX], ld Yim[KMAX]) {
    ld P[LMAX_CAP + 1][LMAX_CAP + 1];
    assoc_legendre(lmax, cosl(theta), sinl(theta), P);
    for (int l = 0; l <= lmax; ++l) {
        for (int m = -l; m <= l; ++m) {
            int am = m < 0 ? -m : m;
            /* P_l^m for the signed m: P_l^{-|m|} = (-1)^|m| (l-|m|)!/(l+|m|)! P_l^{|m|} */
            ld plm = P[l][am];
            if (m < 0) {
                plm *= factorial(l - am) / factorial(l + am);
                if (am & 1) plm = -plm;
            }
            ld norm = sqrtl((ld)(2 * l + 1) / (4.0L * PI_L) * factorial(l - m) / factorial(l + m));
            ld cs = (am & 1) ? -1.0L : 1.0L; /* Condon-Shortley (-1)^m */
            ld amp = cs * norm * plm;
            Yre[l * (l + 1) + m] = amp * cosl((ld)m * phi);
            Yim[l * (l + 1) + m] = amp * sinl((ld)m * phi);
        }
    }
}

/* r = 0 convention: only l = 0 survives, Y_0^0 = 1/sqrt(4 pi). */
static void ylm_origin(int lmax, ld Yre[KMAX], ld Yim[KMAX]) {
    int K = (lmax + 1) * (lmax + 1);
    for (int k = 0; k < K; ++k) { Yre[k] = 0.0L; Yim[k] = 0.0L; }
    Yre[0] = 1.0L / sqrtl(4.0L * PI_L);
}

/* Eq. 3-4 front end: Cartesian point -> Y_l^m. */
static void ylm_cartesian(int lmax, double xd, double yd, double zd, ld Yre[KMAX], ld Yim[KMAX]) {
    ld x = xd, y = yd, z = zd;
    ld r = sqrtl(x * x + y * y + z * z);
    if (r == 0.0L) { ylm_origin(lmax, Yre, Yim); return; }
    ld cz = z / r;
    if (cz > 1.0L) cz = 1.0L;
    if (cz < -1.0L) cz = -1.0L;
    ld theta = acosl(cz);                                                   /* Eq. 3 */
    if (g_theta_mode == 0 && (x * x + y * y) < 1e-10L * (r * r))
        theta = atan2l(hypotl(x, y), z);                                    /* same angle, no cancellation */
    ld phi = atan2l(y, x);                                                  /* Eq. 4 */
    ylm_angular(lmax, theta, phi, Yre, Yim);
}

/* Eq. 6, literally, from the complex values. */
static void real_from_complex(int lmax, const ld Yre[KMAX], const ld Yim[KMAX], ld R[KMAX], ld* max_imag) {
    const ld inv_sqrt2 = 1.0L / sqrtl(2.0L);
    for (int l = 0; l <= lmax; ++l) {
        for (int m = -l; m <= l; ++m) {
            int kp = l * (l + 1) + m, kn = l * (l + 1) - m;
            int am = m < 0 ? -m : m;
            ld sg = (am & 1) ? -1.0L : 1.0L; /* (-1)^m */
            ld re, im;
            if (m < 0) {
                /* (i/sqrt2) (Y_l^m - (-1)^m Y_l^{-m});  i (a + i b) = -b + i a */
                ld a = Yre[kp] - sg * Yre[kn], b = Yim[kp] - sg * Yim[kn];
                re = -b * inv_sqrt2; im = a * inv_sqrt2;
            } else if (m == 0) {
                re = Yre[kp]; im = Yim[kp];
            } else {
                /* (1/sqrt2) (Y_l^{-m} + (-1)^m Y_l^m) */
                re = (Yre[kn] + sg * Yre[kp]) * inv_sqrt2;
                im = (Yim[kn] + sg * Yim[kp]) * inv_sqrt2;
            }
            R[kp] = re;
            ld aim = fabsl(im);
            if (aim > *max_imag) *max_imag = aim;
        }
    }
}

/* Y_l^{m'} with |m'| > l is identically zero (reading #19). */
static void y_or_zero(int l, int m, const ld Yre[KMAX], const ld Yim[KMAX], ld* re, ld* im) {
    if (m < -l || m > l) { *re = 0.0L; *im = 0.0L; return; }
    *re = Yre[l * (l + 1) + m]; *im = Yim[l * (l + 1) + m];
}

int sh_oracle_index_spinor(int l, int twoj, int twomj) {
    /* (m_j + j) = (twomj + twoj)/2 */
    int off = (twomj + twoj) / 2;
    return 2 * l * l + (twoj == 2 * l - 1 ? off : 2 * l + off);
}

/* Eq. 7 for every l <= lmax, j = l -+ 1/2, m_j = -j..j.  out[s][4] = (up.re, up.im, down.re, down.im).
 * Half-integers are carried doubled: twoj = 2j, twomj = 2 m_j (both odd). */
static void spinor_from_complex(int lmax, const ld Yre[KMAX], const ld Yim[KMAX], double* out) {
    for (int l = 0; l <= lmax; ++l) {
        for (int sign = -1; sign <= 1; sign += 2) {
            /* sign = +1: upper sign of Eq. 7, l = j - 1/2;  sign = -1: lower sign, l = j + 1/2 */
            int twoj = 2 * l + sign;
            if (twoj < 1) continue;
            ld pref = 1.0L / sqrtl((ld)(2 * l + 1));          /* 1/sqrt(2 (j -+ 1/2) + 1) */
            for (int twomj = -twoj; twomj <= twoj; twomj += 2) {
                ld mj = 0.5L * (ld)twomj;
                /* upper: (+sqrt(l + m_j + 1/2) Y^{m_j-1/2}, sqrt(l - m_j + 1/2) Y^{m_j+1/2})
                 * lower: (-sqrt(l - m_j + 1/2) Y^{m_j-1/2}, sqrt(l + m_j + 1/2) Y^{m_j+1/2}) */
                ld cu = (ld)sign * sqrtl((ld)l + (ld)sign * mj + 0.5L);
                ld cd = sqrtl((ld)l - (ld)sign * mj + 0.5L);
                int m_up = (twomj - 1) / 2, m_dn = (twomj + 1) / 2;   /* exact: twomj is odd */
                ld ur, ui, dr, di;
                y_or_zero(l, m_up, Yre, Yim, &ur, &ui);
                y_or_zero(l, m_dn, Yre, Yim, &dr, &di);
                double* o = out + 4 * (size_t)sh_oracle_index_spinor(l, twoj, twomj);
                o[0] = (double)(pref * cu * ur); o[1] = (double)(pref * cu * ui);
                o[2] = (double)(pref * cd * dr); o[3] = (double)(pref * cd * di);
            }
        }
    }
}

static void note_imag(ld max_imag) {
    if ((double)max_imag > g_max_imag) {
#ifdef _OPENMP
#pragma omp critical(sh_oracle_imag)
#endif
        { if ((double)max_imag > g_max_imag) g_max_imag = (double)max_imag; }
    }
}

#ifdef _OPENMP
#define PAR_FOR _Pragma("omp parallel for schedule(static) num_threads(sh_oracle_threads_used())")
#else
#define PAR_FOR
#endif

/* kind: 0 real, 1 complex, 2 spinor.  angular != 0: `a` holds (theta, phi) pairs instead of xyz. */
static int run(int kind, int angular, const double* a, int64_t n, int lmax, double* out) {
    if (lmax < 0 || lmax > LMAX_CAP || n < 0 || (n > 0 && (!a || !out))) return -1;
    const int K = (lmax + 1) * (lmax + 1);
    PAR_FOR
    for (int64_t i = 0; i < n; ++i) {
        ld Yre[KMAX], Yim[KMAX];
        if (angular) ylm_angular(lmax, (ld)a[2 * i], (ld)a[2 * i + 1], Yre, Yim);
        else ylm_cartesian(lmax, a[3 * i], a[3 * i + 1], a[3 * i + 2], Yre, Yim);
        if (kind == 0) {
            ld R[KMAX], mi = 0.0L;
            real_from_complex(lmax, Yre, Yim, R, &mi);
            note_imag(mi);
            for (int k = 0; k < K; ++k) out[(size_t)i * K + k] = (double)R[k];
        } else if (kind == 1) {
            for (int k = 0; k < K; ++k) {
                out[((size_t)i * K + k) * 2 + 0] = (double)Yre[k];
                out[((size_t)i * K + k) * 2 + 1] = (double)Yim[k];
            }
        } else {
            spinor_from_complex(lmax, Yre, Yim, out + (size_t)i * 8 * K);
        }
    }
    return 0;
}

int sh_oracle_real(const double* xyz, int64_t n, int lmax, double* out) { return run(0, 0, xyz, n, lmax, out); }
int sh_oracle_complex(const double* xyz, int64_t n, int lmax, double* out) { return run(1, 0, xyz, n, lmax, out); }
int sh_oracle_spinor(const double* xyz, int64_t n, int lmax, double* out) { return run(2, 0, xyz, n, lmax, out); }
/* angular front end (theta, phi pairs): lets the paper's Tables II/III be fed directly. */
int sh_oracle_real_angular(const double* tp, int64_t n, int lmax, double* out) { return run(0, 1, tp, n, lmax, out); }
int sh_oracle_complex_angular(const double* tp, int64_t n, int lmax, double* out) { return run(1, 1, tp, n, lmax, out); }
int sh_oracle_spinor_angular(const double* tp, int64_t n, int lmax, double* out) { return run(2, 1, tp, n, lmax, out); }

/* ------------------------------------------------------------------------------------------------
 * Fused projector consumer (the use case of PAPER.md lines 14 and 20: "the atomic problem is
 * solved in a radial grid ... This produces a series of angular-momentum dependent projectors.  To represent these
 * projectors in a 3-dimensional grid we need to calculate the spherical harmonics for each point").
 *
 * Definition (the paper names the use case but fixes no formula beyond
 * "radial function times spherical harmonic", so the radial interpolation below is reading #25):
 *   channel p = 0..nproj-1 has angular momentum l_p and a radial function f_p tabulated on the uniform radial grid
 *   r_j = j dr, j = 0..nr-1:  radial[p*nr + j] = f_p(r_j).
 *   f_p(r) = radial[p][j] + (r/dr - j)(radial[p][j+1] - radial[p][j]),  j = floor(r/dr),   for r < (nr-1) dr   (piecewise linear)
 *   f_p(r) = 0                                                                             for r >= (nr-1) dr  (beyond the table)
 *   beta_{p,m}(r_vec) = f_p(|r_vec|) R_{l_p}^m(r_vec/|r_vec|),  m = -l_p..l_p                (Eq. 6; r = 0: PAPER.md line 60)
 *   column of (p, m) = sum_{p' < p} (2 l_{p'} + 1) + (m + l_p);   ncols = sum_p (2 l_p + 1)
 *   projection:  coeff[v][col] = sum_i w[v][i] beta_col(r_i)       (w = wave-function values times the volume element)
 * Everything in long double, rounded to double once at the end; the projection is the plain sum in point order.
 * Parity pins: tests/test_oracle_projector_pins.py (linear-table exactness against the separately pinned R_l^m, table
 * nodes and midpoints, cutoff, r = 0, column order, quadrature orthonormality of the projection). */
static ld radial_linear(const double* tab, int nr, ld dr, ld r) {
    ld t = r / dr;
    ld fj = floorl(t);
    if (fj >= (ld)(nr - 1)) return 0.0L;
    int j = (int)fj;
    return (ld)tab[j] + (t - fj) * ((ld)tab[j + 1] - (ld)tab[j]);
}

int sh_oracle_projector_count(int nproj, const int* proj_l) {
    if (nproj < 0 || (nproj > 0 && !proj_l)) return -1;
    int ncols = 0;
    for (int p = 0; p < nproj; ++p) {
        if (proj_l[p] < 0 || proj_l[p] > LMAX_CAP) return -1;
        ncols += 2 * proj_l[p] + 1;
    }
    return ncols;
}

/* beta_{p,m} of one point, long double, all columns */
static void projector_row(const double* p3, int nproj, const int* proj_l, int lmax, const double* radial, int nr, ld dr, ld* row) {
    ld Yre[KMAX], Yim[KMAX], R[KMAX], mi = 0.0L;
    ylm_cartesian(lmax, p3[0], p3[1], p3[2], Yre, Yim);
    real_from_complex(lmax, Yre, Yim, R, &mi);
    ld x = p3[0], y = p3[1], z = p3[2];
    ld r = sqrtl(x * x + y * y + z * z);
    int col = 0;
    for (int p = 0; p < nproj; ++p) {
        int l = proj_l[p];
        ld f = radial_linear(radial + (size_t)p * nr, nr, dr, r);
        for (int m = -l; m <= l; ++m) row[col++] = f * R[l * (l + 1) + m];
    }
}

/* out[i][col], AoS */
int sh_oracle_projectors(const double* xyz, int64_t n, int nproj, const int* proj_l, const double* radial, int nr, double dr, double* out) {
    const int ncols = sh_oracle_projector_count(nproj, proj_l);
    if (ncols < 0 || ncols > KMAX * 4 || n < 0 || nr < 2 || !(dr > 0.0) || (n > 0 && (!xyz || !out || !radial))) return -1;
    int lmax = 0;
    for (int p = 0; p < nproj; ++p) if (proj_l[p] > lmax) lmax = proj_l[p];
    PAR_FOR
    for (int64_t i = 0; i < n; ++i) {
        ld row[KMAX * 4];
        projector_row(xyz + 3 * i, nproj, proj_l, lmax, radial, nr, (ld)dr, row);
        for (int c = 0; c < ncols; ++c) out[(size_t)i * ncols + c] = (double)row[c];
    }
    return 0;
}

/* coeff[v][col] = sum_i w[v][i] beta_col(r_i): the plain sum, in point order, in long double (single thread).
 * abs_sum (optional, same shape) receives sum_i |w[v][i] beta_col(r_i)|, the scale of the tolerance. */
int sh_oracle_project(const double* xyz, int64_t n, int nproj, const int* proj_l, const double* radial, int nr, double dr,
                      const double* w, int nvec, double* coeff, double* abs_sum) {
    const int ncols = sh_oracle_projector_count(nproj, proj_l);
    if (ncols < 0 || ncols > KMAX * 4 || n < 0 || nvec < 0 || nvec > 64 || nr < 2 || !(dr > 0.0)) return -1;
    if ((n > 0 && (!xyz || !radial || (nvec > 0 && !w))) || (nvec > 0 && !coeff)) return -1;
    int lmax = 0;
    for (int p = 0; p < nproj; ++p) if (proj_l[p] > lmax) lmax = proj_l[p];
    ld* acc = (ld*)calloc((size_t)(nvec > 0 ? nvec : 1) * (ncols > 0 ? ncols : 1) * 2, sizeof(ld));
    if (!acc) return -2;
    ld* aabs = acc + (size_t)(nvec > 0 ? nvec : 1) * (ncols > 0 ? ncols : 1);
    for (int64_t i = 0; i < n; ++i) {
        ld row[KMAX * 4];
        projector_row(xyz + 3 * i, nproj, proj_l, lmax, radial, nr, (ld)dr, row);
        for (int v = 0; v < nvec; ++v) {
            ld wi = (ld)w[(size_t)v * n + i];
            for (int c = 0; c < ncols; ++c) {
                ld term = wi * row[c];
                acc[(size_t)v * ncols + c] += term;
                aabs[(size_t)v * ncols + c] += fabsl(term);
            }
        }
    }
    for (int v = 0; v < nvec; ++v)
        for (int c = 0; c < ncols; ++c) {
            coeff[(size_t)v * ncols + c] = (double)acc[(size_t)v * ncols + c];
            if (abs_sum) abs_sum[(size_t)v * ncols + c] = (double)aabs[(size_t)v * ncols + c];
        }
    free(acc);
    return 0;
}
