// sh_peaks.cu -- ceilings microbenchmarks (SURVEY.md section 6 "the build should measure one (DFMA microbenchmark)" and
// section 8(d) denominator (ii) "a write-only fill kernel measured in the same run").  Built into its OWN library
// (libshb200_peaks.so) that only bench.py and the bandwidth-target test load: nothing here is on the product path, and
// libshb200.so does not link it.  No harmonic arithmetic in this file.
//
// The kernels of libshb200 write 97 % of their traffic and read 3 %, so the driver-measured copy bandwidth (half reads, half
// writes) is not their ceiling: a write stream pays no read/write bus turnarounds.  What bounds them is what the same store
// mechanism reaches with NO arithmetic in front of it:
//   shpeak_fill_flat        one flat stream of 32-byte streaming stores (st.global.cs.v4.f64), grid-stride
//   shpeak_fill_bulk_tiles  contiguous tiles, one TMA bulk copy (cp.async.bulk) per tile from shared memory: the AoS kernels' pattern
//   shpeak_fill_soa_planes  [K][n] planes, one TMA tensor store per {points x planes} box: the SoA kernels' pattern
// all with the L2 evict-first policy the library's stores carry.  And for the FP64-bound fused projection:
//   shpeak_dfma             independent DFMA chains at full occupancy: lane-instructions per second of the FP64 pipe
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>

namespace {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint64_t l2_evict_first_policy() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}

__global__ void __launch_bounds__(512) fill_flat_kernel(double* __restrict__ out, int64_t n4) {
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += stride)
        asm volatile("st.global.cs.v4.f64 [%0], {%1, %1, %1, %1};" ::"l"(out + 4 * i), "d"(1.0) : "memory");
}

// one warp per CTA, one tile per CTA (the AoS tile-bulk kernels' shape)
__global__ void __launch_bounds__(32) fill_bulk_tiles_kernel(unsigned char* __restrict__ out, int64_t bytes, int tile_bytes) {
    extern __shared__ __align__(128) unsigned char tile[];
    const int64_t off = (int64_t)blockIdx.x * tile_bytes;
    const int len = (bytes - off) < tile_bytes ? (int)(bytes - off) : tile_bytes;
    for (int e = threadIdx.x * 16; e < len; e += 32 * 16) *reinterpret_cast<double2*>(tile + e) = make_double2(1.0, 2.0);
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncwarp();
    if (threadIdx.x == 0) {
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(out + off), "r"(smem_u32(tile)), "r"(len),
                     "l"(l2_evict_first_policy())
                     : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    }
}

// CTA = one box {row_doubles, planes} at (tile * row_doubles, group * planes); block order: tile-major, plane group fastest
__global__ void __launch_bounds__(256) fill_soa_planes_kernel(const __grid_constant__ CUtensorMap tmap, int row_doubles, int planes, int ngroups) {
    extern __shared__ __align__(128) unsigned char smem[];
    double* t = reinterpret_cast<double*>(smem);
    const int tile = blockIdx.x / ngroups, group = blockIdx.x - tile * ngroups;
    for (int e = threadIdx.x; e < row_doubles * planes; e += blockDim.x) t[e] = (double)e;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
    if (threadIdx.x == 0) {
        asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group.L2::cache_hint [%0, {%1, %2}], [%3], %4;" ::"l"(&tmap), "r"(tile * row_doubles),
                     "r"(group * planes), "r"(smem_u32(t)), "l"(l2_evict_first_policy())
                     : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    }
}

// 8 independent DFMA chains per thread, `iters` rounds: 8 * iters DFMA lane-instructions per thread
__global__ void __launch_bounds__(256) dfma_kernel(double* __restrict__ sink, int64_t iters, double a, double b) {
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int64_t i = 0; i < iters; ++i) {
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
    const double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (s == 123.456) sink[0] = s;   // keeps the chains alive; never true for the arguments bench.py passes
}

using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                   const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int status() { return cudaGetLastError() == cudaSuccess ? 0 : -1; }

}  // namespace

extern "C" {

// `bytes` (a multiple of 32) of `out` (DEVICE, 32-byte aligned) written once by 32-byte streaming stores.  0 = launched.
int shpeak_fill_flat(void* out, int64_t bytes, void* stream) {
    if (!out || bytes <= 0 || bytes % 32) return -1;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    fill_flat_kernel<<<sms * 4, 512, 0, static_cast<cudaStream_t>(stream)>>>(static_cast<double*>(out), bytes / 32);
    return status();
}

// `bytes` of `out` (DEVICE, 16-byte aligned; bytes a multiple of 16) written as contiguous tiles of tile_bytes (a multiple of
// 16, <= 200 KB), one TMA bulk copy each, one warp per CTA.
int shpeak_fill_bulk_tiles(void* out, int64_t bytes, int tile_bytes, void* stream) {
    if (!out || bytes <= 0 || bytes % 16 || tile_bytes <= 0 || tile_bytes % 16 || tile_bytes > 200 * 1024) return -1;
    if (tile_bytes > 48 * 1024 && cudaFuncSetAttribute(fill_bulk_tiles_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, tile_bytes) != cudaSuccess) return -1;
    const int64_t blocks = (bytes + tile_bytes - 1) / tile_bytes;
    if (blocks > 0x7fffffffLL) return -1;
    fill_bulk_tiles_kernel<<<(unsigned)blocks, 32, tile_bytes, static_cast<cudaStream_t>(stream)>>>(static_cast<unsigned char*>(out), bytes, tile_bytes);
    return status();
}

// `out` (DEVICE, 16-byte aligned) viewed as k planes of row_total doubles ([k][row_total], row_total even): every box of
// {row_doubles <= 256, planes <= 256} written by one TMA tensor store; k must be a multiple of planes, row_total of row_doubles.
int shpeak_fill_soa_planes(void* out, int64_t row_total, int k, int row_doubles, int planes, void* stream) {
    if (!out || row_total <= 0 || k <= 0 || row_doubles <= 0 || row_doubles > 256 || planes <= 0 || planes > 256 || k % planes || row_total % row_doubles ||
        row_total % 2)
        return -1;
    static EncodeTiledFn enc = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) p = nullptr;
        return reinterpret_cast<EncodeTiledFn>(p);
    }();
    if (!enc) return -1;
    CUtensorMap tmap;
    const cuuint64_t gdim[2] = {(cuuint64_t)row_total, (cuuint64_t)k};
    const cuuint64_t gstride[1] = {(cuuint64_t)row_total * 8};
    const cuuint32_t box[2] = {(cuuint32_t)row_doubles, (cuuint32_t)planes}, estride[2] = {1, 1};
    if (enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, out, gdim, gstride, box, estride, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
            CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return -1;
    const size_t smem = (size_t)row_doubles * planes * 8;
    if (smem > 200 * 1024) return -1;
    if (smem > 48 * 1024 && cudaFuncSetAttribute(fill_soa_planes_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -1;
    const int ngroups = k / planes;
    const int64_t blocks = row_total / row_doubles * ngroups;
    if (blocks > 0x7fffffffLL) return -1;
    fill_soa_planes_kernel<<<(unsigned)blocks, 256, smem, static_cast<cudaStream_t>(stream)>>>(tmap, row_doubles, planes, ngroups);
    return status();
}

// blocks x 256 threads, each 8 * iters DFMA: returns the number of DFMA lane-instructions the launch executes (or -1)
int64_t shpeak_dfma(double* sink, int64_t iters, int blocks, void* stream) {
    if (!sink || iters <= 0 || blocks <= 0) return -1;
    dfma_kernel<<<blocks, 256, 0, static_cast<cudaStream_t>(stream)>>>(sink, iters, 0.999999, 1e-9);
    return status() == 0 ? (int64_t)blocks * 256 * 8 * iters : -1;
}

}  // extern "C"
