// sh_abi.cu -- host state shared by the translation units of libshb200.so (launch counter, CUDA error text, tuning knobs,
// SM count, prefetch plan, tensor-map encoder lookup, host staging pool) and the small entry points of include/shb200.h
// that launch nothing.
#include "sh_store.cuh"   // HostPool

namespace shb200 {

std::atomic<int64_t> g_launches{0};
thread_local char g_cuda_error[256] = "";

int cuda_fail(cudaError_t e) {
    std::strncpy(g_cuda_error, cudaGetErrorString(e), sizeof(g_cuda_error) - 1);
    return SH_ERR_CUDA;
}

// SMs of the CURRENT device (cached per device; 148 on a B200)
int sm_count() {
    static PerDeviceInt cache;
    const int sms = cache.get([] {
        int dev = 0, v = 0;
        if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0) return v;
        return 0;
    });
    return sms > 0 ? sms : 148;
}

// launch-heuristic overrides (sh_set_tuning); 0 = default
std::atomic<int> g_tune[SH_TUNE_COUNT];

int tuned(int knob, int dflt) {
    const int v = g_tune[knob].load(std::memory_order_relaxed);
    return v > 0 ? v : dflt;
}

// window plan of the burst input prefetch for a launch whose CTAs own `points_per_cta` consecutive points each
InputPrefetch prefetch_plan(int64_t n, int64_t points_per_cta) {
    const int64_t win_points = tuned(SH_TUNE_PREFETCH_WINDOW_POINTS, 1 << 18);   // 6 MiB of fp64 xyz per burst
    InputPrefetch pf{0, 0};
    if (win_points <= 1 || n <= win_points) return pf;   // knob value 1 = off; one window: the first wave reads it all anyway
    int64_t win = win_points / points_per_cta;
    if (win < 1) win = 1;
    if (win > 0x3fffffff) return pf;
    pf.win_ctas = (int)win;
    pf.spread = win < sm_count() ? (int)win : sm_count();
    return pf;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point lookup (no link against libcuda); nullptr if unavailable
EncodeTiledFn encode_tiled() {
    static EncodeTiledFn fn = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) p = nullptr;
        return reinterpret_cast<EncodeTiledFn>(p);
    }();
    return fn;
}

HostPool g_pool;

}  // namespace shb200

using namespace shb200;

extern "C" {

void sh_host_release(void) {
    std::lock_guard<std::mutex> lock(g_pool.mu);
    g_pool.release();
}

int64_t sh_real_count(int lmax) { return (lmax < 0 || lmax > shgen::LMAX_EXT) ? -1 : (int64_t)(lmax + 1) * (lmax + 1); }
int64_t sh_complex_count(int lmax) { return (lmax < 0 || lmax > shgen::LMAX_EXT) ? -1 : 2 * (int64_t)(lmax + 1) * (lmax + 1); }
int64_t sh_spinor_count(int lmax) { return (lmax < 0 || lmax > 9) ? -1 : 8 * (int64_t)(lmax + 1) * (lmax + 1); }

int sh_index_real(int l, int m) {
    if (l < 0 || l > shgen::LMAX_EXT || m < -l || m > l) return -1;
    return l * (l + 1) + m;
}

int sh_index_spinor(int l, int twoj, int twomj) {
    if (l < 0 || l > 9) return -1;
    if (twoj != 2 * l - 1 && twoj != 2 * l + 1) return -1;
    if (twoj < 1) return -1;
    if (twomj < -twoj || twomj > twoj || ((twomj - twoj) & 1)) return -1;
    const int off = (twomj + twoj) / 2;   // m_j + j
    return 2 * l * l + (twoj == 2 * l - 1 ? off : 2 * l + off);
}

const char* sh_strerror(int code) {
    switch (code) {
        case SH_OK: return "ok";
        case SH_ERR_NULL: return "xyz or out is NULL with n > 0";
        case SH_ERR_COUNT: return "n is negative or too large for one launch";
        case SH_ERR_LMAX: return "lmax must be in [0, 9] (sh_real_ext / sh_complex_ext: [0, 32])";
        case SH_ERR_LAYOUT: return "unknown layout, store-path or front-end bits, or a layout this call does not offer";
        case SH_ERR_ALIGNMENT: return "pointer not aligned to its element type, or requested store path impossible for this alignment";
        case SH_ERR_CUDA: return "CUDA error (see sh_last_cuda_error)";
        case SH_ERR_PROJECTOR: return "bad projector arguments (nproj, proj_l, nr, dr, nvec or workspace size)";
        case SH_ERR_SCRATCH: return "sh_project_static: the request needs more than the 2 MiB static scratch array (see sh_project_static_bytes; use sh_project with a workspace)";
    }
    return "unknown error code";
}

const char* sh_last_cuda_error(void) { return g_cuda_error; }

int sh_set_tuning(int knob, int value) {
    if (knob < 0 || knob >= SH_TUNE_COUNT || value < 0) return SH_ERR_LAYOUT;
    g_tune[knob].store(value, std::memory_order_relaxed);
    return SH_OK;
}
int64_t sh_kernel_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }


}  // extern "C"
