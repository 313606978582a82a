// sh_spinor.cu -- sh_spinor / sh_spinor_host: spin-1/2 spinor harmonics, fp64 (include/shb200.h); kernels and launchers in sh_store.cuh.
#include "sh_store.cuh"

using namespace shb200;

extern "C" {

int sh_spinor(const double* xyz, int64_t n, int lmax, double* out, int layout, void* stream) {
    return run_device<KIND_SPINOR, double, double>(xyz, n, lmax, out, layout, stream);
}
int sh_spinor_host(const double* xyz, int64_t n, int lmax, double* out, int layout) {
    return run_host<KIND_SPINOR, double, double>(xyz, n, lmax, out, layout);
}

}  // extern "C"
