// sh_real.cu -- sh_real / sh_real_host: real harmonics R_l^m, fp64 (include/shb200.h); kernels and launchers in sh_store.cuh.
// Also sh_real_sum: the compute-only protocol of the paper's Table I.
#include "sh_store.cuh"

namespace shb200 {

// sh_real_sum: every R_l^m of a point is evaluated exactly as in sh_real (a1-a5) and ACCUMULATED; one double per point is stored.  This
// is how the paper times its library ("the results are accumulated and never stored"): with 32 B/point of traffic instead
// of 824 the path is bound by the FP64 pipe, so it measures the arithmetic side of the roofline of the factorized formulas.
struct SumSink {
    double s = 0.0;
    template <int K> __device__ __forceinline__ void put1(double v) { s += v; }
    template <int L> __device__ __forceinline__ void end_l() {}
    template <int L> __device__ __forceinline__ void polar(const double (&)[L + 1]) {}
};

template <int LMAX, bool ANGULAR>
__global__ void __launch_bounds__(256) sh_real_sum_kernel(const double* __restrict__ xyz, int64_t n, double* __restrict__ out, int coords) {
    const int64_t i = ((int64_t)blockIdx.x << 8) + threadIdx.x;
    if (i >= n) return;
    RawPoint<double, ANGULAR> pt;
    pt.load(xyz, i);
    SumSink sink;
    evaluate<KIND_REAL, LMAX, double>(pt.unit(coords), sink);
    out[i] = sink.s;
}

template <int LMAX>
int launch_real_sum(const double* xyz, int64_t n, double* out, int coords, cudaStream_t st) {
    const int64_t blocks = (n + 255) / 256;
    if (blocks > 0x7fffffffLL) return SH_ERR_COUNT;
    if (coords == SH_COORDS_ANGULAR) sh_real_sum_kernel<LMAX, true><<<(unsigned)blocks, 256, 0, st>>>(xyz, n, out, coords);
    else sh_real_sum_kernel<LMAX, false><<<(unsigned)blocks, 256, 0, st>>>(xyz, n, out, coords);
    return launch_status();
}

int run_real_sum(const double* xyz, int64_t n, int lmax, double* out, int coords, void* stream) {
    if (n < 0) return SH_ERR_COUNT;
    if (lmax < 0 || lmax > shgen::LMAX_CAP) return SH_ERR_LMAX;
    if (coords != SH_COORDS_CARTESIAN && coords != SH_COORDS_NORMALIZED && coords != SH_COORDS_ANGULAR) return SH_ERR_LAYOUT;
    if (n == 0) return SH_OK;
    if (!xyz || !out) return SH_ERR_NULL;
    if (!aligned(out, 8) || !aligned(xyz, 8)) return SH_ERR_ALIGNMENT;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    switch (lmax) {
#define SH_CASE(L) case L: return launch_real_sum<L>(xyz, n, out, coords, st);
        SH_CASE(0) SH_CASE(1) SH_CASE(2) SH_CASE(3) SH_CASE(4) SH_CASE(5) SH_CASE(6) SH_CASE(7) SH_CASE(8) SH_CASE(9)
#undef SH_CASE
    }
    return SH_ERR_LMAX;
}

}  // namespace shb200

using namespace shb200;

extern "C" {

int sh_real(const double* xyz, int64_t n, int lmax, double* out, int layout, void* stream) {
    return run_device<KIND_REAL, double, double>(xyz, n, lmax, out, layout, stream);
}
int sh_real_host(const double* xyz, int64_t n, int lmax, double* out, int layout) {
    return run_host<KIND_REAL, double, double>(xyz, n, lmax, out, layout);
}
int sh_real_sum(const double* xyz, int64_t n, int lmax, double* out, int coords, void* stream) {
    return run_real_sum(xyz, n, lmax, out, coords, stream);
}

}  // extern "C"
