// sh_real_f32.cu -- sh_real_f32 / sh_real_f32_host: real harmonics, fp32 variant (include/shb200.h); kernels and launchers in sh_store.cuh.
#include "sh_store.cuh"

using namespace shb200;

extern "C" {

int sh_real_f32(const float* xyz, int64_t n, int lmax, float* out, int layout, void* stream) {
    return run_device<KIND_REAL, float, float>(xyz, n, lmax, out, layout, stream);
}
int sh_real_f32_host(const float* xyz, int64_t n, int lmax, float* out, int layout) {
    return run_host<KIND_REAL, float, float>(xyz, n, lmax, out, layout);
}

}  // extern "C"
