// lm_harness.cpp -- compiled by tests/test_lm_header.py with g++ (no CUDA): every sh_real_lm<L, M> / sh_complex_lm<L, M> of
// include/shb200_lm.cuh at n unit vectors -> real[n][100], cplx[n][100][2], k = l(l+1)+m.
#include <type_traits>

#include "../include/shb200_lm.cuh"

template <int B, int E, class F>
static inline void static_for(F&& f) {
    if constexpr (B < E) {
        f(std::integral_constant<int, B>{});
        static_for<B + 1, E>(f);
    }
}

extern "C" void lm_eval(const double* xyz, int n, double* real, double* cplx) {
    for (int i = 0; i < n; ++i) {
        const double x = xyz[3 * i], y = xyz[3 * i + 1], z = xyz[3 * i + 2];
        static_for<0, 10>([&](auto lc) {
            constexpr int L = decltype(lc)::value;
            static_for<0, 2 * L + 1>([&](auto jc) {
                constexpr int M = decltype(jc)::value - L;
                constexpr int K = L * (L + 1) + M;
                real[100 * i + K] = shb200::sh_real_lm<L, M>(x, y, z);
                shb200::sh_complex_lm<L, M>(x, y, z, cplx[2 * (100 * i + K)], cplx[2 * (100 * i + K) + 1]);
            });
        });
    }
}

extern "C" float lm_real_7_m3_f32(float x, float y, float z) { return shb200::sh_real_lm<7, -3, float>(x, y, z); }
