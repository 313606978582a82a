// sh_ext.cu -- sh_real_ext / sh_complex_ext (include/shb200.h): lmax up to 32 by recurrence in l, SoA.
#include "sh_core.cuh"

namespace shb200 {

// ------------------------------------------------------------------------------------------------
// Extension beyond the explicit range, 10 <= l <= LMAX_EXT = 32 (the paper's conclusion: "could be easily
// extended using recurrence relationships for higher values of l").  The explicit l <= 9 block is evaluated as above
// and seeds, at fixed m, the upward recurrence in l of the normalized polar factors (tables from the generator):
//   q_lm = A_lm (z q_{l-1,m} - B_lm q_{l-2,m})   seeds q_8m, q_9m (m <= 9);      q_ll = SECT_l q_{l-1,l-1}  (l >= 10)
//   C_m + i S_m = (C_{m-1} + i S_{m-1}) (x + i y)                                 seeds C_9, S_9            (m >= 10)
// Loops run m-outer, l-inner, so a thread carries two q's and one (C_m, S_m) only; SoA planes make every store of a
// warp contiguous whatever the order of (l, m).  (AoS rows would be written 8 bytes at a time, columns l(l+1)+-m
// far apart: not offered for lmax > 9.)
template <int KIND>
struct SoAExtSink {
    double* p;        // out + i*ES
    int64_t stride;   // n*ES
    bool vec16;       // complex elements may be written by one 16-byte store
    double q8[9], q9[10];
    template <int K> __device__ __forceinline__ void put1(double v) { __stcs(p + K * stride, v); }
    template <int K> __device__ __forceinline__ void put2(double re, double im) { put_complex(K, re, im); }
    template <int L> __device__ __forceinline__ void end_l() {}
    template <int L> __device__ __forceinline__ void polar(const double (&q)[L + 1]) {
        if constexpr (L == 8) { static_for<0, 9>([&](auto mc) { q8[decltype(mc)::value] = q[decltype(mc)::value]; }); }
        if constexpr (L == 9) { static_for<0, 10>([&](auto mc) { q9[decltype(mc)::value] = q[decltype(mc)::value]; }); }
    }
    __device__ __forceinline__ void put_complex(int k, double re, double im) {
        double* q = p + k * stride;
        if (vec16) __stcs(reinterpret_cast<double2*>(q), make_double2(re, im));
        else { __stcs(q, re); __stcs(q + 1, im); }
    }
    // harmonics (l, +-m) from the polar factor q and the azimuthal pair (c, s); KIND_REAL: Eq. 6; KIND_COMPLEX: Eq. 5, 10
    __device__ __forceinline__ void emit(int l, int m, double q, double c, double s) {
        const int k0 = l * (l + 1);
        if constexpr (KIND == KIND_REAL) {
            if (m == 0) { __stcs(p + k0 * stride, q); return; }
            __stcs(p + (k0 + m) * stride, q * c);
            __stcs(p + (k0 - m) * stride, q * s);
        } else {
            if (m == 0) { put_complex(k0, q, 0.0); return; }
            const double a = q * c, b = q * s;
            put_complex(k0 - m, a, -b);
            if (m & 1) put_complex(k0 + m, -a, -b);
            else put_complex(k0 + m, a, b);
        }
    }
};

template <int KIND, bool ANGULAR>
__global__ void __launch_bounds__(256) sh_soa_ext_kernel(const double* __restrict__ xyz, int64_t n, double* __restrict__ out, int lmax, int coords, int vec16,
                                                          InputPrefetch pf) {
    constexpr int ES = elem_scalars(KIND);
    constexpr int IN_BYTES = (ANGULAR ? 2 : 3) * sizeof(double);
    constexpr int NT = shgen::LMAX_EXT + 1;
    prefetch_input_window(xyz, n * IN_BYTES, (int64_t)256 * IN_BYTES, pf);
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    RawPoint<double, ANGULAR> pt;
    pt.load(xyz, i);
    const UnitVec u = pt.unit(coords);
    const double z = u.z;
    SoAExtSink<KIND> sink;
    sink.p = out + i * ES;
    sink.stride = n * ES;
    sink.vec16 = vec16 != 0;
    const Azim<9, double> az(u.x, u.y);
    if constexpr (KIND == KIND_REAL) eval_real<9, double>(az, z, u.origin, sink);
    else eval_complex<9, double>(az, z, u.origin, sink);
    // m <= 9: the explicit factors C_m, S_m; l = 10 .. lmax by recurrence from the explicit q_8m, q_9m
    static_for<0, 10>([&](auto mc) {
        constexpr int M = decltype(mc)::value;
        double q2 = 0.0, q1 = sink.q9[M];
        if constexpr (M <= 8) q2 = sink.q8[M];
        for (int l = 10; l <= lmax; ++l) {
            const double q = shgen::REC_A[l * NT + M] * (z * q1 - shgen::REC_B[l * NT + M] * q2);
            sink.emit(l, M, q, az.C[M], az.S[M]);
            q2 = q1; q1 = q;
        }
    });
    // m >= 10: sectoral seed q_mm, azimuthal pair by complex multiplication, then the same recurrence in l
    double c = az.C[9], s = az.S[9], qmm = sink.q9[9];
    for (int m = 10; m <= lmax; ++m) {
        const double cn = c * u.x - s * u.y;
        s = c * u.y + s * u.x;
        c = cn;
        qmm *= shgen::REC_SECT[m];
        sink.emit(m, m, qmm, c, s);
        double q2 = 0.0, q1 = qmm;
        for (int l = m + 1; l <= lmax; ++l) {
            const double q = shgen::REC_A[l * NT + m] * (z * q1 - shgen::REC_B[l * NT + m] * q2);
            sink.emit(l, m, q, c, s);
            q2 = q1; q1 = q;
        }
    }
}


// l > 9 extension (sh_real_ext / sh_complex_ext): lmax <= 9 is the regular path; above, SoA only
template <int KIND>
int run_device_ext(const double* xyz, int64_t n, int lmax, double* out, int layout_bits, void* stream) {
    if (lmax <= shgen::LMAX_CAP)   // the regular path (kernels in sh_real.cu / sh_complex.cu)
        return KIND == KIND_REAL ? sh_real(xyz, n, lmax, out, layout_bits, stream) : sh_complex(xyz, n, lmax, out, layout_bits, stream);
    if (n < 0) return SH_ERR_COUNT;
    if (lmax > shgen::LMAX_EXT) return SH_ERR_LMAX;
    const int layout = layout_bits & 0xff, path = layout_bits & 0xff00, coords = layout_bits & 0x30000;
    if ((layout_bits & ~0x3ffff) || layout != SH_LAYOUT_SOA || (path != SH_STORE_AUTO && path != SH_STORE_DIRECT) || coords == 0x30000)
        return SH_ERR_LAYOUT;
    if (n == 0) return SH_OK;
    if (!xyz || !out) return SH_ERR_NULL;
    if (!aligned(out, sizeof(double)) || !aligned(xyz, sizeof(double))) return SH_ERR_ALIGNMENT;
    const int64_t blocks = (n + 255) / 256;
    if (blocks > 0x7fffffffLL) return SH_ERR_COUNT;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const int vec16 = aligned(out, 16) ? 1 : 0;   // complex element (k*n + i) sits 16 (k*n + i) bytes into `out`
    const InputPrefetch pf = prefetch_plan(n, 256);
    if (coords == SH_COORDS_ANGULAR) sh_soa_ext_kernel<KIND, true><<<(unsigned)blocks, 256, 0, st>>>(xyz, n, out, lmax, coords, vec16, pf);
    else sh_soa_ext_kernel<KIND, false><<<(unsigned)blocks, 256, 0, st>>>(xyz, n, out, lmax, coords, vec16, pf);
    return launch_status();
}


}  // namespace shb200

using namespace shb200;

extern "C" {

int sh_real_ext(const double* xyz, int64_t n, int lmax, double* out, int layout, void* stream) {
    return run_device_ext<KIND_REAL>(xyz, n, lmax, out, layout, stream);
}
int sh_complex_ext(const double* xyz, int64_t n, int lmax, double* out, int layout, void* stream) {
    return run_device_ext<KIND_COMPLEX>(xyz, n, lmax, out, layout, stream);
}
int sh_lmax_ext(void) { return shgen::LMAX_EXT; }

}  // extern "C"
