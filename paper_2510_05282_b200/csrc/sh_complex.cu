// sh_complex.cu -- sh_complex / sh_complex_host: complex harmonics Y_l^m, fp64 (include/shb200.h); kernels and launchers in sh_store.cuh.
#include "sh_store.cuh"

using namespace shb200;

extern "C" {

int sh_complex(const double* xyz, int64_t n, int lmax, double* out, int layout, void* stream) {
    return run_device<KIND_COMPLEX, double, double>(xyz, n, lmax, out, layout, stream);
}
int sh_complex_host(const double* xyz, int64_t n, int lmax, double* out, int layout) {
    return run_host<KIND_COMPLEX, double, double>(xyz, n, lmax, out, layout);
}

}  // extern "C"
