/* shb200_lm.cuh -- header-only, per-point, per-(l, m) interface to the generated formulas (C++17; host or device).
 *
 * This is the API shape of the paper's own library: one function per harmonic, "callable from host and device code", taking
 * the NORMALIZED Cartesian coordinates x = X/r, y = Y/r, z = Z/r (Eq. 8) and returning one value.  The batched
 * C ABI of shb200.h is what the kernels of this repository are built around (normalization and the azimuthal factors are paid
 * once per point there); this header is for a caller who needs ONE (l, m), or who writes their own kernel:
 *
 *     #include "shb200_lm.cuh"
 *     double v = shb200::sh_real_lm<7, -3>(x, y, z);            // R_7^{-3} (Eq. 6), the paper's worked example (Eq. 11-15)
 *     shb200::sh_complex_lm<2, 1>(x, y, z, re, im);             // Y_2^1 (Eq. 5, Condon-Shortley phase)
 *
 * l <= 9, |m| <= l, both compile-time (the formulas are straight-line code per (l, m): Eq. 16 root-pair products, every root and
 * constant computed by paper_2510_05282_b200/gen/generate.py).  The caller guarantees x^2 + y^2 + z^2 = 1; the r = 0 convention
 * is the caller's to apply, as in the paper.  T = double, or float (fp32 polynomials), or any type with * + - and
 * construction from double / int.  In CUDA code the functions are __host__ __device__; compiled as plain C++ define nothing. */
#ifndef SHB200_LM_CUH
#define SHB200_LM_CUH
#if !defined(SHGEN_FN) && !defined(__CUDACC__)
#define SHGEN_FN inline
#endif
#include "../paper_2510_05282_b200/csrc/sh_generated.cuh"

namespace shb200 {

/* R_l^m(x, y, z), Eq. 6: m > 0 cosine-type, m < 0 sine-type, k = l(l+1)+m in the batched calls. */
template <int L, int M, typename T = double>
SHGEN_FN T sh_real_lm(T x, T y, T z) {
    static_assert(L >= 0 && L <= shgen::LMAX_CAP && M >= -L && M <= L, "0 <= l <= 9, |m| <= l");
    constexpr int MA = M < 0 ? -M : M;
    const T q = T(shgen::A_REAL[L][MA]) * shgen::Polar<L, MA, T>::eval(z);
    if constexpr (M == 0) {
        return q;
    } else {
        T c, s;
        shgen::Azimuthal<MA, T>::eval(x, y, c, s);
        if constexpr (M < 0) return q * s;
        else return q * c;
    }
}

/* Y_l^m(x, y, z) = re + i im, Eq. 5 with the Condon-Shortley phase; Y_l^{-m} = (-1)^m conj(Y_l^m) (Eq. 10). */
template <int L, int M, typename T = double>
SHGEN_FN void sh_complex_lm(T x, T y, T z, T& re, T& im) {
    static_assert(L >= 0 && L <= shgen::LMAX_CAP && M >= -L && M <= L, "0 <= l <= 9, |m| <= l");
    constexpr int MA = M < 0 ? -M : M;
    const T u = T(shgen::B_CPLX[L][MA]) * shgen::Polar<L, MA, T>::eval(z);
    if constexpr (M == 0) {
        re = u; im = T(0);
    } else {
        T c, s;
        shgen::Azimuthal<MA, T>::eval(x, y, c, s);
        const T a = u * c, b = u * s;             /* a + i b = B Qhat (C + i S) */
        if constexpr (M < 0) { re = a; im = -b; }
        else if constexpr (MA % 2) { re = -a; im = -b; }
        else { re = a; im = b; }
    }
}

}  /* namespace shb200 */
#endif /* SHB200_LM_CUH */
