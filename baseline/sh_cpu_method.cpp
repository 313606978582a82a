// sh_cpu_method.cpp -- the paper's method on the HOST cores: the same generated factorized formulas the CUDA kernels
// include (paper_2510_05282_b200/csrc/sh_generated.cuh, compiled here as plain C++), evaluated in fp64 for every
// l <= lmax at a batch of points and stored as AoS [n][K] or SoA [K][n].
//
// What this is for, and what it is NOT:
//   * a GPU-less check of the generator's output (tests/test_generated_host.py compares it with the oracle and with the
//     formulas the paper prints in Appendix C) -- a generator regression is then caught without a B200;
//   * the timed CPU baseline of bench.py ("cpu_method"): the paper's own CPU scheme -- explicit factorized polynomials in
//     normalized Cartesian coordinates, fp64 (its Table I, reports 553 M harmonics/s on one core for
//     normalized input and 228 M/s for Cartesian input, accumulating instead of storing) -- next to the long-double
//     oracle, which is a deliberately slow checker and understates what a CPU can do by two orders of magnitude;
//   * NOT a fallback: paper_2510_05282_b200/binding.py never loads it, libshb200.so does not link it, and nothing on the
//     sh_* product path can reach it.  Only tests/ and bench.py's cpu_method leg load this library.
// It shares sh_generated.cuh with the CUDA path on purpose (that header is what is being checked / timed) and shares
// nothing with oracle/.
//
// Per point: a2 normalize (skipped for normalized input), a3 azimuthal factors, a4 polar factors,
// a5 combine; r = 0 -> R_0^0 = 1/sqrt(4 pi), everything else 0.  W points are evaluated together in one GCC vector
// (the formulas are templates over the value type), OpenMP over blocks of points.
#include <cmath>
#include <cstdint>
#include <cstring>
#include <type_traits>
#ifdef _OPENMP
#include <omp.h>
#endif

#define SHGEN_FN inline __attribute__((always_inline))
#include "../paper_2510_05282_b200/csrc/sh_generated.cuh"

namespace {

constexpr int W = 8;   // points per vector (one zmm, or two ymm)
typedef double vraw __attribute__((vector_size(8 * W)));

struct vd {
    vraw v;
    vd() = default;
    explicit vd(double s) { for (int i = 0; i < W; ++i) v[i] = s; }
    explicit vd(int s) : vd((double)s) {}
};
static inline __attribute__((always_inline)) vd operator*(vd a, vd b) { vd r; r.v = a.v * b.v; return r; }
static inline __attribute__((always_inline)) vd operator+(vd a, vd b) { vd r; r.v = a.v + b.v; return r; }
static inline __attribute__((always_inline)) vd operator-(vd a, vd b) { vd r; r.v = a.v - b.v; return r; }
static inline __attribute__((always_inline)) vd operator-(vd a) { vd r; r.v = -a.v; return r; }

template <int B, int E, class F>
static inline __attribute__((always_inline)) void static_for(F&& f) {
    if constexpr (B < E) {
        f(std::integral_constant<int, B>{});
        static_for<B + 1, E>(f);
    }
}

// all (lmax+1)^2 real harmonics of W unit vectors, k = l(l+1)+m (Eq. 6): vals[k]
template <int LMAX, bool HORNER>
static inline __attribute__((always_inline)) void eval_unit(vd x, vd y, vd z, vd* vals) {
    vd C[LMAX + 1], S[LMAX + 1];
    static_for<0, LMAX + 1>([&](auto mc) {
        constexpr int M = decltype(mc)::value;
        shgen::Azimuthal<M, vd>::eval(x, y, C[M], S[M]);
    });
    const vd z2 = z * z;
    static_for<0, LMAX + 1>([&](auto lc) {
        constexpr int L = decltype(lc)::value;
        static_for<0, L + 1>([&](auto mc) {
            constexpr int M = decltype(mc)::value;
            vd q;
            if constexpr (HORNER) q = vd(shgen::A_REAL[L][M]) * shgen::PolarHorner<L, M, vd>::eval(z, z2);
            else q = vd(shgen::A_REAL[L][M]) * shgen::Polar<L, M, vd>::eval(z);
            if constexpr (M == 0) vals[L * (L + 1)] = q;
            else {
                vals[L * (L + 1) - M] = q * S[M];
                vals[L * (L + 1) + M] = q * C[M];
            }
        });
    });
}

template <int LMAX, bool HORNER>
__attribute__((target_clones("default", "avx2,fma", "avx512f")))
void run(const double* xyz, int64_t n, double* out, int soa, int normalized) {
    constexpr int K = (LMAX + 1) * (LMAX + 1);
    const int64_t nblocks = (n + W - 1) / W;
#pragma omp parallel for schedule(static)
    for (int64_t b = 0; b < nblocks; ++b) {
        const int64_t i0 = b * W;
        const int cnt = (n - i0) < W ? (int)(n - i0) : W;
        vd x(0.0), y(0.0), z(1.0);
        bool origin[W] = {};
        bool any_origin = false;
        for (int j = 0; j < cnt; ++j) {
            double px = xyz[3 * (i0 + j)], py = xyz[3 * (i0 + j) + 1], pz = xyz[3 * (i0 + j) + 2];
            const double r2 = px * px + py * py + pz * pz;
            origin[j] = (r2 == 0.0);
            any_origin |= origin[j];
            if (!normalized) {
                const double inv = origin[j] ? 0.0 : 1.0 / std::sqrt(r2);   // a2; the configs keep r^2 inside the fp64 range
                px *= inv; py *= inv; pz *= inv;
            }
            x.v[j] = px; y.v[j] = py; z.v[j] = pz;
        }
        vd vals[K];
        eval_unit<LMAX, HORNER>(x, y, z, vals);
        if (any_origin)
            for (int j = 0; j < cnt; ++j)
                if (origin[j])
                    for (int k = 1; k < K; ++k) vals[k].v[j] = 0.0;   // only l = 0 survives at r = 0
        if (soa) {
            if (cnt == W) {
                for (int k = 0; k < K; ++k) std::memcpy(out + (int64_t)k * n + i0, &vals[k].v, sizeof(vraw));
            } else {
                for (int k = 0; k < K; ++k)
                    for (int j = 0; j < cnt; ++j) out[(int64_t)k * n + i0 + j] = vals[k].v[j];
            }
        } else {
            for (int j = 0; j < cnt; ++j) {
                double* row = out + (i0 + j) * K;
                for (int k = 0; k < K; ++k) row[k] = vals[k].v[j];
            }
        }
    }
}

// compute-only variant in the manner of the paper's timing loop (results are accumulated, never stored):
// returns the sum of every harmonic over the batch
template <int LMAX, bool HORNER>
__attribute__((target_clones("default", "avx2,fma", "avx512f")))
double run_accumulate(const double* xyz, int64_t n, int normalized) {
    constexpr int K = (LMAX + 1) * (LMAX + 1);
    const int64_t nblocks = n / W;   // whole blocks only: a timing loop
    double total = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : total)
    for (int64_t b = 0; b < nblocks; ++b) {
        const int64_t i0 = b * W;
        vd x, y, z;
        for (int j = 0; j < W; ++j) {
            double px = xyz[3 * (i0 + j)], py = xyz[3 * (i0 + j) + 1], pz = xyz[3 * (i0 + j) + 2];
            if (!normalized) {
                const double r2 = px * px + py * py + pz * pz;
                const double inv = r2 == 0.0 ? 0.0 : 1.0 / std::sqrt(r2);
                px *= inv; py *= inv; pz *= inv;
            }
            x.v[j] = px; y.v[j] = py; z.v[j] = pz;
        }
        vd vals[K];
        eval_unit<LMAX, HORNER>(x, y, z, vals);
        vd acc(0.0);
        for (int k = 0; k < K; ++k) acc = acc + vals[k];
        for (int j = 0; j < W; ++j) total += acc.v[j];
    }
    return total;
}

}  // namespace

extern "C" {

// R_l^m for all l <= lmax at Cartesian (normalized = 0) or unit (normalized = 1) points xyz [n][3];
// out: AoS [n][K] (soa = 0) or SoA [K][n] (soa = 1); form: 0 = factorized root-pair products (Eq. 16), 1 = Horner in z^2.
// Returns 0, or -1 on bad arguments.
int shcpu_real(const double* xyz, int64_t n, int lmax, double* out, int soa, int normalized, int form) {
    if (n < 0 || lmax < 0 || lmax > shgen::LMAX_CAP || (n > 0 && (!xyz || !out))) return -1;
    switch (lmax) {
#define SH_CASE(L) case L: if (form) run<L, true>(xyz, n, out, soa, normalized); else run<L, false>(xyz, n, out, soa, normalized); return 0;
        SH_CASE(0) SH_CASE(1) SH_CASE(2) SH_CASE(3) SH_CASE(4) SH_CASE(5) SH_CASE(6) SH_CASE(7) SH_CASE(8) SH_CASE(9)
#undef SH_CASE
    }
    return -1;
}

// sum over the batch of all harmonics with l <= 9 (nothing stored), for a compute-only rate comparable with the paper's Table I
double shcpu_real_accumulate_l9(const double* xyz, int64_t n, int normalized, int form) {
    if (n <= 0 || !xyz) return 0.0;
    return form ? run_accumulate<9, true>(xyz, n, normalized) : run_accumulate<9, false>(xyz, n, normalized);
}

void shcpu_set_threads(int t) {
#ifdef _OPENMP
    omp_set_num_threads(t > 0 ? t : omp_get_num_procs());
#else
    (void)t;
#endif
}

int shcpu_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
