// sh_real.cu -- sh_real / sh_real_host: real harmonics R_l^m, fp64 (include/shb200.h); kernels and launchers in sh_store.cuh.
#include "sh_store.cuh"

using namespace shb200;

extern "C" {

int sh_real(const double* xyz, int64_t n, int lmax, double* out, int layout, void* stream) {
    return run_device<KIND_REAL, double, double>(xyz, n, lmax, out, layout, stream);
}
int sh_real_host(const double* xyz, int64_t n, int lmax, double* out, int layout) {
    return run_host<KIND_REAL, double, double>(xyz, n, lmax, out, layout);
}

}  // extern "C"
