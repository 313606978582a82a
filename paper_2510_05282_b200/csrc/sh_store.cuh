// sh_store.cuh -- step a8 for the sh_real / sh_complex / sh_spinor / sh_real_f32 calls: store kernels (SoA by streaming
// stores or one TMA tensor store per tile, AoS by shared-memory staging and TMA bulk copies), their launchers, the
// dispatch over lmax / layout / alignment, and the host-buffer pipeline.  Included by one translation unit per kind.
#pragma once
#include "sh_core.cuh"

namespace shb200 {

// ------------------------------------------------------------------------------------------------
// ------------------------------------------------------------------------------------------------
// a8, SoA: element e of point i lives at out[(e*n + i) * ES .. +ES).  A warp writes 32*ES contiguous scalars
// per element; streaming (evict-first) stores since nothing is re-read.  VEC = widest store in bytes the
// alignment of `out` allows.
template <typename T, int VEC>
struct SoASink {
    T* p;             // out + i*ES
    int64_t stride;   // n*ES scalars between consecutive elements
    template <int K> __device__ __forceinline__ void put1(T v) { __stcs(p + K * stride, v); }
    template <int K> __device__ __forceinline__ void put2(T re, T im) {
        T* q = p + K * stride;
        if constexpr (VEC >= 16 && sizeof(T) == 8) {
            __stcs(reinterpret_cast<double2*>(q), make_double2(re, im));
        } else { __stcs(q, re); __stcs(q + 1, im); }
    }
    template <int S> __device__ __forceinline__ void put4(T a, T b, T c, T d) {
        T* q = p + S * stride;
        if constexpr (VEC >= 32 && sizeof(T) == 8) {
            asm volatile("st.global.cs.v4.f64 [%0], {%1, %2, %3, %4};" ::"l"(q), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
        } else if constexpr (VEC >= 16 && sizeof(T) == 8) {
            __stcs(reinterpret_cast<double2*>(q), make_double2(a, b));
            __stcs(reinterpret_cast<double2*>(q) + 1, make_double2(c, d));
        } else { __stcs(q, a); __stcs(q + 1, b); __stcs(q + 2, c); __stcs(q + 3, d); }
    }
    template <int L> __device__ __forceinline__ void end_l() {}
    template <int L> __device__ __forceinline__ void polar(const T (&)[L + 1]) {}
};

// One 256-point tile per CTA: with the burst L2 prefetch the input load is an L2 hit, and a deep grid lets the hardware CTA
// scheduler balance the SMs (251 vs 256 / 258 us for 1 / 2 / 4 tiles per CTA on the 128^3 grid at lmax = 9).
// Spinor, 16- and 32-byte store variants: ptxas takes 146 registers, i.e. ONE 256-thread CTA per SM.  Capped at 128 (two CTAs, 40-88 bytes
// of spills) the lmax = 9 kernel is SLOWER (3.88 vs 3.77 ms on 2^22 points): the 32-byte stores of 8 warps already saturate the write stream.
template <int KIND, int LMAX, typename T, typename TI, int VEC, bool ANGULAR>
__global__ void __launch_bounds__(256) sh_soa_kernel(const TI* __restrict__ xyz, int64_t n, T* __restrict__ out, int coords, InputPrefetch pf) {
    constexpr int ES = elem_scalars(KIND);
    constexpr int IN_BYTES = (ANGULAR ? 2 : 3) * sizeof(TI);
    prefetch_input_window(xyz, n * IN_BYTES, (int64_t)256 * IN_BYTES, pf);
    const int64_t i = ((int64_t)blockIdx.x << 8) + threadIdx.x;
    if (i >= n) return;
    RawPoint<TI, ANGULAR> pt;
    pt.load(xyz, i);
    SoASink<T, VEC> sink{out + i * ES, n * ES};
    evaluate<KIND, LMAX, T>(pt.unit(coords), sink);
}

// a8, SoA through the TMA tensor unit (sh_real fp64 and sh_real_f32).  One CTA = one tile of PTS points = SOA_TMA_WARPS groups
// of 32 points; thread i stages value k of its point at tile[k][i] (conflict-free 8-byte / 4-byte shared stores: consecutive
// lanes, consecutive words), and after a proxy fence and a CTA barrier thread 0 issues ONE cp.async.bulk.tensor.2d store of
// the box {PTS points, K planes} through a tensor map of `out` viewed as [K][n]: K rows of 1 KB (128 fp64 / 256 fp32 points).
// The LSU issues no global store at all (100 STG + their address arithmetic per point in sh_soa_kernel), and points past n
// in a ragged last tile are clipped by the tensor unit.
// Groups per tile: longer rows are what the tile buys -- 258 / 258 / 250 / 345 us for 1 / 2 / 4 / 8 groups (rows of
// 256 B .. 2 KB; 8 groups = one 205 KB tile per SM, nothing overlaps) on the 128^3 grid at lmax = 9.
constexpr int SOA_TMA_WARPS = 4;
// Warps sharing a 32-point group (lmax >= 4): two warps, each evaluating part of the l-blocks (block_part), shorten a tile's
// compute phase, so the two resident CTAs overlap their tensor stores better: 0.2499 -> 0.2477 ms on the 128^3 grid at
// lmax = 9 (with 64-point tiles the split changes nothing: 0.2585 ms either way -- row length, not compute, bounds those).
constexpr int SOA_SPLIT = 2;

template <int PTS, typename T = double>
struct TileSink {
    T* col;   // tile + this thread's point (complex: + 2 * point)
    template <int K> __device__ __forceinline__ void put1(T v) { col[K * PTS] = v; }
    template <int K> __device__ __forceinline__ void put2(T re, T im) { *reinterpret_cast<double2*>(col + K * 2 * PTS) = make_double2(re, im); }   // 16-byte stores, consecutive lanes: conflict-free
    template <int L> __device__ __forceinline__ void end_l() {}
    template <int L> __device__ __forceinline__ void polar(const T (&)[L + 1]) {}
};

// SPLIT warps share each 32-point group of the tile, each evaluating part of the l-blocks (block_part in sh_core.cuh)
// T = float (sh_real_f32): the same kernel on 256-point tiles (rows of 1 KB again), fp64 normalization, fp32 polynomials.
// Two CTAs per SM is what the 102 KB tile allows.  fp32 (512 threads with SPLIT = 2) needs the register cap of minBlocks = 2;
// for fp64 minBlocks stays unspecified (0): given a cap, ptxas spends registers up to it (64 -> 120 at minBlocks = 2, and 148,
// i.e. ONE resident CTA and 0.41 instead of 0.24 ms, at minBlocks = 1).
// KIND_COMPLEX (sh_complex): elements of 16 bytes, so 64-point tiles keep the 1 KB rows; `out` is seen as fp64 [K][2 n], box {128, K}.
template <typename T, int LMAX, int WARPS, int SPLIT, bool ANGULAR, int KIND = KIND_REAL>
__global__ void __launch_bounds__(32 * WARPS * SPLIT, sizeof(T) == 4 ? 2 : 0) sh_soa_tma_kernel(const T* __restrict__ xyz, int64_t n,
                                                                                                  const __grid_constant__ CUtensorMap tmap, int coords,
                                                                                                  InputPrefetch pf) {
    constexpr int PTS = 32 * WARPS, ES = elem_scalars(KIND);
    static_assert(KIND == KIND_REAL || (KIND == KIND_COMPLEX && sizeof(T) == 8), "real (fp64, fp32) and complex (fp64) harmonics");
    extern __shared__ __align__(128) unsigned char smem_tile[];
    constexpr int IN_BYTES = (ANGULAR ? 2 : 3) * sizeof(T);
    prefetch_input_window(xyz, n * IN_BYTES, (int64_t)PTS * IN_BYTES, pf);
    T* tile = reinterpret_cast<T*>(smem_tile);
    const int p = SPLIT == 1 ? threadIdx.x : threadIdx.x % PTS;   // point of the tile
    const int64_t base = (int64_t)blockIdx.x * PTS, i = base + p;
    if (i < n) {
        RawPoint<T, ANGULAR> pt;
        pt.load(xyz, i);
        TileSink<PTS, T> sink{tile + ES * p};
        const UnitVec u = pt.unit(coords);
        if constexpr (SPLIT == 1) evaluate<KIND, LMAX, T>(u, sink);
        else {
            const int part = threadIdx.x / PTS;   // warp-uniform
            static_for<0, SPLIT>([&](auto pc) {
                constexpr int PART = decltype(pc)::value;
                if (part == PART) {
                    if constexpr (KIND == KIND_REAL) eval_real_part<LMAX, SPLIT, PART>((T)u.x, (T)u.y, (T)u.z, u.origin, sink);   // fp32: rounded once, after the fp64 normalization
                    else eval_complex_part<LMAX, SPLIT, PART>((T)u.x, (T)u.y, (T)u.z, u.origin, sink);
                }
            });
        }
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // every thread: its staging stores -> async proxy
    if constexpr (WARPS * SPLIT == 1) __syncwarp();
    else __syncthreads();
    if (threadIdx.x == 0) {
        asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group.L2::cache_hint [%0, {%1, %2}], [%3], %4;" ::"l"(&tmap), "r"((int)(ES * base)), "r"(0),
                     "r"(smem_u32(tile)), "l"(l2_evict_first_policy())
                     : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // shared memory is released when the CTA exits
    }
}

// fp32 SoA, two ADJACENT points (2j, 2j+1) per thread: 8-byte stores (a warp store covers 256 B of a plane),
// half the store and address instructions per point, packed-fp32 arithmetic.  Needs even n and 8-byte aligned out.
struct SoAPairSink {
    float* p;         // out + 2j
    int64_t stride;   // n
    template <int K> __device__ __forceinline__ void put1(f2 v) { __stcs(reinterpret_cast<float2*>(p + K * stride), v.v); }
    template <int L> __device__ __forceinline__ void end_l() {}
    template <int L> __device__ __forceinline__ void polar(const f2 (&)[L + 1]) {}
};

template <int LMAX>
__global__ void __launch_bounds__(256) sh_soa_pair_kernel(const float* __restrict__ xyz, int64_t n, float* __restrict__ out, int coords, InputPrefetch pf) {
    prefetch_input_window(xyz, n * 12, (int64_t)512 * 12, pf);
    const int64_t j = ((int64_t)blockIdx.x << 8) + threadIdx.x;   // pair index
    if (j >= (n >> 1)) return;
    const float2* q = reinterpret_cast<const float2*>(xyz + 6 * j);   // 24 B per pair: three 8-byte loads
    const float2 ca = __ldg(q), cb = __ldg(q + 1), cc = __ldg(q + 2);
    SoAPairSink sink{out + 2 * j, n};
    // one copy of the polynomial code: only the front end branches (straight-line code size is instruction-fetch traffic)
    UnitVec u0, u1;
    if (coords == SH_COORDS_CARTESIAN) { u0 = normalize_f32in(ca.x, ca.y, cb.x); u1 = normalize_f32in(cb.y, cc.x, cc.y); }
    else { u0 = as_given(ca.x, ca.y, cb.x); u1 = as_given(cb.y, cc.x, cc.y); }
    evaluate_pair<LMAX>(u0, u1, sink);
}


// ------------------------------------------------------------------------------------------------
// ------------------------------------------------------------------------------------------------
// a8, AoS: a point's row of SP = scalars_per_point scalars is contiguous in `out`.  Each lane stages its row
// (or a segment of whole l-blocks of it, at most CAP scalars) in its own shared-memory row, then
//   MODE_ROWBULK: the lane issues ONE TMA bulk copy (cp.async.bulk.global.shared::cta) for its segment;
//                 needs 16-byte aligned global segments.  No warp-level synchronization at all.
//   MODE_TILEBULK: whole rows are staged DENSELY (pitch = row), so the warp's 32-row tile is one contiguous span of
//                 `out`; after a __syncwarp one lane issues ONE bulk copy for the whole tile (25.6 KB at lmax = 9).
//                 One large TMA request per tile instead of 32 small ones: 7.4 vs 6.3-6.7 TB/s on a store-only model.
//                 Dense rows cost 2-way bank conflicts on the 16-byte staging stores when the row is 32 (mod 128) bytes
//                 (lmax = 9: 800 B); layouts where it would be worse (tile_bulk_ok) stay on MODE_ROWBULK.
//   MODE_PLAIN:   the warp copies the staged tile out with coalesced streaming stores (any alignment).
template <int KIND, int LMAX, int TSIZE, int CAP, int MODE>
struct Segments {
    static constexpr int SP = scalars_per_point(KIND, LMAX);
    // a cut before block l is allowed where the row offset keeps the copy granularity (16 B for bulk)
    static constexpr bool cut_ok(int l) { return l == LMAX + 1 || MODE == MODE_PLAIN || (MODE == MODE_ROWBULK && (cum_scalars(KIND, l) * TSIZE) % 16 == 0); }
    // greedy: the segment starting at block s ends before block seg_end(s)
    static constexpr int seg_end(int s) {
        int best = -1;
        for (int c = s + 1; c <= LMAX + 1; ++c)
            if (cut_ok(c) && cum_scalars(KIND, c) - cum_scalars(KIND, s) <= CAP) best = c;
        return best;
    }
    static constexpr int first_l(int l) {
        int s = 0;
        while (seg_end(s) <= l) s = seg_end(s);
        return s;
    }
    static constexpr bool valid() {
        for (int s = 0; s <= LMAX;) {
            int e = seg_end(s);
            if (e < 0) return false;
            s = e;
        }
        return true;
    }
    static constexpr int max_len() {
        int m = 0;
        for (int s = 0; s <= LMAX; s = seg_end(s)) {
            int len = cum_scalars(KIND, seg_end(s)) - cum_scalars(KIND, s);
            if (len > m) m = len;
        }
        return m;
    }
    // row pitch in scalars: conflict-free staging stores.  bulk: 16-byte stores, odd number of 16-byte chunks;
    // plain: scalar stores, odd number of 8-byte (fp64) / 4-byte (fp32) words.
    static constexpr int pitch() {
        if (MODE == MODE_TILEBULK) return SP;
        if (MODE == MODE_ROWBULK) {
            int chunks = (max_len() * TSIZE + 15) / 16;
            return (chunks | 1) * 16 / TSIZE;
        }
        return max_len() | 1;
    }
};

template <int KIND, int LMAX, typename T, int CAP, int MODE>
struct RowSink {
    using Seg = Segments<KIND, LMAX, sizeof(T), CAP, MODE>;
    static constexpr int SP = Seg::SP;
    static constexpr int PITCH = Seg::pitch();
    static constexpr int VPC = 16 / sizeof(T);   // scalars per 16-byte chunk
    // 16-byte staging stores: always in row-bulk mode (padded, aligned rows); in tile-bulk mode when dense rows keep 16-byte alignment
    static constexpr bool VSTAGE = MODE == MODE_ROWBULK || (MODE == MODE_TILEBULK && (SP * sizeof(T)) % 16 == 0);

    T* row;          // this lane's staging row (shared memory)
    T* tile;         // the warp's staging tile (32 rows)
    T* gout;         // global `out`
    int64_t i;       // this lane's point
    int64_t base;    // first point of the warp's tile
    int rows;        // valid rows of the tile (plain mode)
    int lane;
    T hold[VPC > 1 ? VPC - 1 : 1];

    // scalar offset of row scalar J inside the staging row
    template <int J, int L> static constexpr int off() { return J - cum_scalars(KIND, Seg::first_l(L)); }
    template <int K> static constexpr int l_of_real() { int l = 0; while ((l + 1) * (l + 1) <= K) ++l; return l; }
    template <int S> static constexpr int l_of_spinor() { int l = 0; while (2 * (l + 1) * (l + 1) <= S) ++l; return l; }

    __device__ __forceinline__ void st16(T* dst, T a, T b) { *reinterpret_cast<double2*>(dst) = make_double2(a, b); }

    template <int K> __device__ __forceinline__ void put1(T v) {
        constexpr int O = off<K, l_of_real<K>()>();
        if constexpr (!VSTAGE) {
            row[O] = v;
        } else if constexpr (sizeof(T) == 8) {
            if constexpr (K % 2 == 0) hold[0] = v;
            else st16(row + O - 1, hold[0], v);
        } else {
            if constexpr (K % 4 != 3) hold[K % 4] = v;
            else *reinterpret_cast<float4*>(row + O - 3) = make_float4(hold[0], hold[1], hold[2], v);
        }
    }
    template <int K> __device__ __forceinline__ void put2(T re, T im) {
        constexpr int O = off<2 * K, l_of_real<K>()>();
        if constexpr (!VSTAGE) { row[O] = re; row[O + 1] = im; }
        else st16(row + O, re, im);
    }
    template <int S> __device__ __forceinline__ void put4(T a, T b, T c, T d) {
        constexpr int O = off<4 * S, l_of_spinor<S>()>();
        if constexpr (!VSTAGE) { row[O] = a; row[O + 1] = b; row[O + 2] = c; row[O + 3] = d; }
        else { st16(row + O, a, b); st16(row + O + 2, c, d); }
    }

    template <int L> __device__ __forceinline__ void polar(const T (&)[L + 1]) {}

    __device__ __forceinline__ void wait_reads() {
        if constexpr (MODE != MODE_PLAIN) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        if constexpr (MODE == MODE_TILEBULK) __syncwarp();   // lane 0 owns the tile's bulk group; nobody restages before it has been read
    }

    // coalesced copy-out of `rows` staged rows (tile-contiguous in `out` when whole rows are staged)
    __device__ __forceinline__ void copy_out_whole_rows() {
        T* g = gout + base * SP;
        const int total = rows * SP;
        int r = 0, c = lane;
        while (c >= SP) { c -= SP; ++r; }
        for (int e = lane; e < total; e += 32) {
            __stcs(g + e, tile[r * PITCH + c]);
            c += 32;
            while (c >= SP) { c -= SP; ++r; }
        }
    }

    template <int L> __device__ __forceinline__ void end_l() {
        constexpr int S0 = Seg::first_l(L);
        if constexpr (Seg::seg_end(S0) == L + 1) {
            constexpr int BEGIN = cum_scalars(KIND, S0);
            constexpr int LEN = cum_scalars(KIND, L + 1) - BEGIN;
            if constexpr (MODE == MODE_ROWBULK) {
                static_assert((LEN * sizeof(T)) % 16 == 0 && (BEGIN * sizeof(T)) % 16 == 0, "bulk granularity");
                // generic-proxy staging stores -> visible to the async proxy, then one bulk copy for this row segment
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                bulk_store(gout + i * SP + BEGIN, row, LEN * (int)sizeof(T));
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                if constexpr (L < LMAX) wait_reads();   // the row is reused by the next segment
            } else if constexpr (MODE == MODE_TILEBULK) {
                static_assert(LEN == SP && PITCH == SP, "tile-bulk mode stages whole dense rows");
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // every lane: its staging stores -> async proxy
                __syncwarp();
                const int bytes = rows * SP * (int)sizeof(T);
                if (bytes % 16 == 0) {   // always for a full tile; a ragged last tile with an odd scalar count is copied by the warp
                    if (lane == 0) {
                        bulk_store(gout + base * SP, tile, bytes);
                        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                    }
                } else {
                    copy_out_whole_rows();
                    __syncwarp();
                }
            } else {
                __syncwarp();
                if constexpr (LEN == SP) {
                    // whole rows staged: the tile is one contiguous span of rows*SP scalars in `out`
                    copy_out_whole_rows();
                } else {
                    for (int r = 0; r < rows; ++r) {
                        T* g = gout + (base + r) * SP + BEGIN;
                        for (int c = lane; c < LEN; c += 32) __stcs(g + c, tile[r * PITCH + c]);
                    }
                }
                __syncwarp();
            }
        }
    }
};

// One 32-point tile per warp: measured fastest on every bulk path now that the input arrives by the burst L2 prefetch (real
// tile-bulk 238 / 242 / 249 us, spinor row-bulk 1002 / 1028 / 1064 us for 1 / 2 / 4 tiles per warp).
template <int KIND, int LMAX, typename T, typename TI, int CAP, int MODE, int WARPS, bool ANGULAR>
__global__ void __launch_bounds__(WARPS * 32) sh_aos_kernel(const TI* __restrict__ xyz, int64_t n, T* __restrict__ out, int coords, InputPrefetch pf) {
    using Sink = RowSink<KIND, LMAX, T, CAP, MODE>;
    constexpr int IN_BYTES = (ANGULAR ? 2 : 3) * sizeof(TI);
    prefetch_input_window(xyz, n * IN_BYTES, (int64_t)WARPS * 32 * IN_BYTES, pf);
    static_assert(Sink::Seg::valid(), "CAP too small for one l-block group");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    T* tile = reinterpret_cast<T*>(smem_raw) + (size_t)warp * 32 * Sink::PITCH;
    const int64_t base = ((int64_t)blockIdx.x * WARPS + warp) << 5;   // first point of the warp's tile
    if (base >= n) return;
    int64_t i = base + lane;
    // plain / tile-bulk mode: every lane takes part in the warp-level copy-out, so idle lanes of the last tile evaluate a clamped point
    if (i >= n) {
        if constexpr (MODE == MODE_ROWBULK) return;
        i = n - 1;
    }
    RawPoint<TI, ANGULAR> pt;
    pt.load(xyz, i);
    const int64_t left = n - base;
    Sink sink;
    sink.row = tile + lane * Sink::PITCH;
    sink.tile = tile;
    sink.gout = out;
    sink.base = base;
    sink.rows = left < 32 ? (int)left : 32;
    sink.lane = lane;
    sink.i = i;
    evaluate<KIND, LMAX, T>(pt.unit(coords), sink);
    if constexpr (MODE != MODE_PLAIN) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // shared memory is released when the CTA exits
}


// ------------------------------------------------------------------------------------------------
// launchers
template <int KIND, int LMAX, typename T, typename TI, int VEC, bool ANGULAR = false>
int launch_soa(const TI* xyz, int64_t n, T* out, int coords, cudaStream_t st) {
    const int64_t blocks = (n + 255) / 256;
    if (blocks > 0x7fffffffLL) return SH_ERR_COUNT;
    sh_soa_kernel<KIND, LMAX, T, TI, VEC, ANGULAR><<<(unsigned)blocks, 256, 0, st>>>(xyz, n, out, coords, prefetch_plan(n, 256));
    return launch_status();
}

// SoA through the tensor unit: `out` as a 2-D tensor [K][n] of fp64 / fp32 (row pitch must be a multiple of 16 bytes: n even /
// a multiple of 4), box {points per tile, K}, tiles of 1 KB rows (128 / 256 points).  Returns SH_ERR_ALIGNMENT when this launch
// cannot use the path (the caller then takes the LSU-store kernels).
template <int LMAX, bool ANGULAR = false, typename T = double, int KIND = KIND_REAL>
int launch_soa_tma(const T* xyz, int64_t n, T* out, int coords, cudaStream_t st) {
    constexpr int K = (LMAX + 1) * (LMAX + 1), ES = elem_scalars(KIND);
    constexpr int TMA_WARPS = SOA_TMA_WARPS * (int)(sizeof(double) / sizeof(T)) / ES;   // rows of 1 KB: 128 fp64, 256 fp32, 64 complex128 points
    constexpr int PTS = 32 * TMA_WARPS;
    EncodeTiledFn enc = encode_tiled();
    if (!enc || (n * ES * sizeof(T)) % 16 != 0 || n < PTS || n * ES > 0x7fffff00LL || !aligned(out, 16)) return SH_ERR_ALIGNMENT;
    CUtensorMap tmap;
    const cuuint64_t gdim[2] = {(cuuint64_t)n * ES, (cuuint64_t)K};
    const cuuint64_t gstride[1] = {(cuuint64_t)n * ES * sizeof(T)};
    const cuuint32_t box[2] = {PTS * ES, (cuuint32_t)K}, estride[2] = {1, 1};
    if (enc(&tmap, sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, out, gdim, gstride, box, estride, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
            CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return SH_ERR_ALIGNMENT;
    const int64_t blocks = (n + PTS - 1) / PTS;
    constexpr size_t smem = (size_t)K * PTS * ES * sizeof(T);
    static_assert(smem <= 227 * 1024, "tile exceeds shared memory");
    auto launch = [&](auto kern, int split, SmemOptIn& opted_in) -> int {
        const int rc = ensure_dynamic_smem(kern, smem, opted_in);
        if (rc != SH_OK) return rc;
        kern<<<(unsigned)blocks, PTS * split, smem, st>>>(xyz, n, tmap, coords, prefetch_plan(n, PTS));
        return launch_status();
    };
    static SmemOptIn opted_in[2];
    if constexpr (LMAX >= 4) {
        if (tuned(SH_TUNE_SOA_SPLIT, SOA_SPLIT) >= 2) return launch(sh_soa_tma_kernel<T, LMAX, TMA_WARPS, 2, ANGULAR, KIND>, 2, opted_in[1]);
    }
    return launch(sh_soa_tma_kernel<T, LMAX, TMA_WARPS, 1, ANGULAR, KIND>, 1, opted_in[0]);
}

// staging capacity per row, in scalars: whole rows for real (800 B at lmax = 9) and complex (1600 B);
// spinor rows (6400 B) are staged in groups of l-blocks of at most 1600 B
template <int KIND, int LMAX>
constexpr int aos_cap() {
    return KIND == KIND_SPINOR ? (200 > 8 * (2 * LMAX + 1) ? 200 : 8 * (2 * LMAX + 1)) : scalars_per_point(KIND, LMAX);
}

template <int KIND, int LMAX, typename T>
constexpr bool tile_bulk_ok() {
    constexpr int row_bytes = scalars_per_point(KIND, LMAX) * (int)sizeof(T);
    if (KIND == KIND_SPINOR || TILEBULK_WARPS * 32 * row_bytes > 55 * 1024) return false;
    if (row_bytes % 16 != 0) return true;
    int chunks = row_bytes / 16, g = 8;
    while (chunks % g) g >>= 1;
    return g <= TILEBULK_MAX_CONFLICT;
}

template <int KIND, int LMAX, typename T, typename TI, int MODE, bool ANGULAR = false>
int launch_aos(const TI* xyz, int64_t n, T* out, int coords, cudaStream_t st) {
    constexpr int CAP = aos_cap<KIND, LMAX>();
    constexpr int WARPS = MODE == MODE_TILEBULK ? TILEBULK_WARPS : 4;
    using Sink = RowSink<KIND, LMAX, T, CAP, MODE>;
    constexpr size_t smem = (size_t)WARPS * 32 * Sink::PITCH * sizeof(T);
    static_assert(smem <= 227 * 1024, "staging tile exceeds shared memory");
    auto kern = sh_aos_kernel<KIND, LMAX, T, TI, CAP, MODE, WARPS, ANGULAR>;
    static SmemOptIn opted_in;
    if (const int rc = ensure_dynamic_smem(kern, smem, opted_in); rc != SH_OK) return rc;
    const int64_t blocks = ((n + 31) / 32 + WARPS - 1) / WARPS;
    if (blocks > 0x7fffffffLL) return SH_ERR_COUNT;
    kern<<<(unsigned)blocks, WARPS * 32, smem, st>>>(xyz, n, out, coords, prefetch_plan(n, (int64_t)WARPS * 32));
    return launch_status();
}

template <int LMAX>
int launch_soa_pair(const float* xyz, int64_t n, float* out, int coords, cudaStream_t st) {
    const int64_t blocks = ((n >> 1) + 255) / 256;
    if (blocks > 0x7fffffffLL) return SH_ERR_COUNT;
    sh_soa_pair_kernel<LMAX><<<(unsigned)blocks, 256, 0, st>>>(xyz, n, out, coords, prefetch_plan(n, 512));
    return launch_status();
}

template <int KIND, int LMAX, typename T, typename TI>
int dispatch_lmax(const TI* xyz, int64_t n, T* out, int layout, int path, int coords, cudaStream_t st) {
    constexpr int SP = scalars_per_point(KIND, LMAX);
    constexpr bool F32 = std::is_same<T, float>::value && KIND == KIND_REAL;
    if (coords == SH_COORDS_ANGULAR) {
        // angular front end: served by the generic store paths (scalar SoA stores, AoS staging + coalesced copy-out), which
        // are valid for every alignment -- except sh_real SoA, which takes the tensor-store path where `out` allows it
        if (path == SH_STORE_BULK) return SH_ERR_ALIGNMENT;
        if constexpr (KIND == KIND_REAL && std::is_same<T, double>::value) {
            if (layout == SH_LAYOUT_SOA && path == SH_STORE_AUTO && tuned(SH_TUNE_SOA_TMA, 0) != 1) {   // the tensor-store path of sh_real SoA
                const int rc = launch_soa_tma<LMAX, true>(reinterpret_cast<const double*>(xyz), n, reinterpret_cast<double*>(out), coords, st);
                if (rc != SH_ERR_ALIGNMENT) return rc;
            }
        }
        if (layout == SH_LAYOUT_SOA) return launch_soa<KIND, LMAX, T, TI, 8, true>(xyz, n, out, coords, st);
        return launch_aos<KIND, LMAX, T, TI, MODE_PLAIN, true>(xyz, n, out, coords, st);
    }
    if (layout == SH_LAYOUT_SOA) {
        if (path == SH_STORE_BULK) return SH_ERR_ALIGNMENT;   // bulk path is AoS only
        constexpr int ES = elem_scalars(KIND);
        if constexpr (KIND == KIND_REAL && std::is_same<T, double>::value) {
            // one tensor-map store per 128-point tile where `out` allows it (16-byte aligned, even n)
            if (path == SH_STORE_AUTO && tuned(SH_TUNE_SOA_TMA, 0) != 1) {
                const int rc = launch_soa_tma<LMAX>(reinterpret_cast<const double*>(xyz), n, reinterpret_cast<double*>(out), coords, st);
                if (rc != SH_ERR_ALIGNMENT) return rc;
            }
        }
        if constexpr (KIND == KIND_COMPLEX && std::is_same<T, double>::value) {
            // one tensor store per 64-point tile where `out` allows it (16-byte aligned)
            if (path == SH_STORE_AUTO && tuned(SH_TUNE_SOA_TMA, 0) != 1) {
                const int rc = launch_soa_tma<LMAX, false, double, KIND_COMPLEX>(reinterpret_cast<const double*>(xyz), n, reinterpret_cast<double*>(out), coords, st);
                if (rc != SH_ERR_ALIGNMENT) return rc;
            }
        }
        if constexpr (F32) {
            // one tensor store per 256-point tile where `out` allows it (16-byte aligned, n a multiple of 4)
            if (path == SH_STORE_AUTO && tuned(SH_TUNE_SOA_TMA, 0) != 1) {
                const int rc = launch_soa_tma<LMAX, false, float>(reinterpret_cast<const float*>(xyz), n, reinterpret_cast<float*>(out), coords, st);
                if (rc != SH_ERR_ALIGNMENT) return rc;
            }
            // two adjacent points per thread (packed fp32, 8-byte stores) when every plane keeps 8-byte alignment
            if (n >= 2 && n % 2 == 0 && aligned(out, 8) && aligned(xyz, 8) && path != SH_STORE_DIRECT)
                return launch_soa_pair<LMAX>(reinterpret_cast<const float*>(xyz), n, reinterpret_cast<float*>(out), coords, st);
        }
        // plane e starts at out + e*n*ES scalars: vector stores need that to stay aligned for every e
        const size_t plane_bytes = (size_t)n * ES * sizeof(T);
        if constexpr (ES * sizeof(T) >= 32) {
            if (aligned(out, 32) && plane_bytes % 32 == 0) return launch_soa<KIND, LMAX, T, TI, 32>(xyz, n, out, coords, st);
        }
        if constexpr (ES * sizeof(T) >= 16) {
            if (aligned(out, 16) && plane_bytes % 16 == 0) return launch_soa<KIND, LMAX, T, TI, 16>(xyz, n, out, coords, st);
        }
        return launch_soa<KIND, LMAX, T, TI, 8>(xyz, n, out, coords, st);
    }
    // bulk (TMA) paths need a 16-byte aligned `out`: one copy per warp tile where dense staging is cheap (every row size),
    // else one copy per row (rows that are multiples of 16 B)
    if (aligned(out, 16) && path != SH_STORE_DIRECT) {
        if constexpr (tile_bulk_ok<KIND, LMAX, T>()) return launch_aos<KIND, LMAX, T, TI, MODE_TILEBULK>(xyz, n, out, coords, st);
        else if constexpr ((SP * sizeof(T)) % 16 == 0) return launch_aos<KIND, LMAX, T, TI, MODE_ROWBULK>(xyz, n, out, coords, st);
    }
    if (path == SH_STORE_BULK) return SH_ERR_ALIGNMENT;
    return launch_aos<KIND, LMAX, T, TI, MODE_PLAIN>(xyz, n, out, coords, st);
}

template <int KIND, typename T, typename TI>
int run_device(const TI* xyz, int64_t n, int lmax, T* out, int layout_bits, void* stream) {
    if (n < 0) return SH_ERR_COUNT;
    if (lmax < 0 || lmax > shgen::LMAX_CAP) return SH_ERR_LMAX;
    const int layout = layout_bits & 0xff, path = layout_bits & 0xff00, coords = layout_bits & 0x30000;
    if ((layout_bits & ~0x3ffff) || (layout != SH_LAYOUT_AOS && layout != SH_LAYOUT_SOA) ||
        (path != SH_STORE_AUTO && path != SH_STORE_DIRECT && path != SH_STORE_BULK) || coords == 0x30000)
        return SH_ERR_LAYOUT;
    if (n == 0) return SH_OK;
    if (!xyz || !out) return SH_ERR_NULL;
    if (!aligned(out, sizeof(T)) || !aligned(xyz, sizeof(TI))) return SH_ERR_ALIGNMENT;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    switch (lmax) {
#define SH_CASE(L) case L: return dispatch_lmax<KIND, L, T, TI>(xyz, n, out, layout, path, coords, st);
        SH_CASE(0) SH_CASE(1) SH_CASE(2) SH_CASE(3) SH_CASE(4) SH_CASE(5) SH_CASE(6) SH_CASE(7) SH_CASE(8) SH_CASE(9)
#undef SH_CASE
    }
    return SH_ERR_LMAX;
}


// Host-buffer pipeline: chunks of points go host -> device -> kernel -> host on two streams (double buffering):
// the device->host copy of chunk c overlaps the host->device copy and the kernel of chunk c+1.
// The two staging slots (64 MiB input + 256 MiB output each) and their streams are created on first use and
// kept for later calls (cudaMalloc/cudaFree per call cost milliseconds and cudaFree synchronizes the device);
// sh_host_release() frees them.  One host call at a time uses the pool (mutex); device calls never touch it.
struct HostPool {
    std::mutex mu;
    int device = -1;
    cudaStream_t st[2] = {nullptr, nullptr};
    void* din[2] = {nullptr, nullptr};
    void* dout[2] = {nullptr, nullptr};
    static constexpr size_t IN_CAP = (size_t)64 << 20, OUT_CAP = (size_t)256 << 20;
    void release() {
        for (int b = 0; b < 2; ++b) {
            if (st[b]) cudaStreamDestroy(st[b]);
            if (din[b]) cudaFree(din[b]);
            if (dout[b]) cudaFree(dout[b]);
            st[b] = nullptr; din[b] = nullptr; dout[b] = nullptr;
        }
        device = -1;
    }
    cudaError_t ensure() {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        if (device == dev && st[1] && dout[1]) return cudaSuccess;
        release();
        for (int b = 0; b < 2; ++b) {
            if ((e = cudaStreamCreateWithFlags(&st[b], cudaStreamNonBlocking)) != cudaSuccess) return e;
            if ((e = cudaMalloc(&din[b], IN_CAP)) != cudaSuccess) return e;
            if ((e = cudaMalloc(&dout[b], OUT_CAP)) != cudaSuccess) return e;
        }
        device = dev;
        return cudaSuccess;
    }
};
extern HostPool g_pool;   // defined in sh_abi.cu

template <int KIND, typename T, typename TI>
int run_host(const TI* xyz, int64_t n, int lmax, T* out, int layout_bits) {
    if (n < 0) return SH_ERR_COUNT;
    if (lmax < 0 || lmax > shgen::LMAX_CAP) return SH_ERR_LMAX;
    const int layout = layout_bits & 0xff, coords = layout_bits & 0x30000;
    if ((layout_bits & ~0x3ffff) || (layout != SH_LAYOUT_AOS && layout != SH_LAYOUT_SOA) || coords == 0x30000) return SH_ERR_LAYOUT;
    if (n == 0) return SH_OK;
    if (!xyz || !out) return SH_ERR_NULL;
    const int64_t w = coords == SH_COORDS_ANGULAR ? 2 : 3;   // input scalars per point
    const int64_t sp = (int64_t)elem_scalars(KIND) * elems_per_point(KIND, lmax);   // scalars per point
    const int64_t es = elem_scalars(KIND), ne = sp / es;
    // chunk: what fits a staging slot, a multiple of 256 points
    int64_t chunk = (int64_t)(HostPool::OUT_CAP / (size_t)(sp * (int64_t)sizeof(T)));
    const int64_t chunk_in = (int64_t)(HostPool::IN_CAP / (size_t)(w * (int64_t)sizeof(TI)));
    if (chunk > chunk_in) chunk = chunk_in;
    chunk = chunk / 256 * 256;
    if (chunk > n) chunk = n;
    std::lock_guard<std::mutex> lock(g_pool.mu);
    int rc = SH_OK;
    auto check = [&](cudaError_t e) { if (e != cudaSuccess && rc == SH_OK) rc = cuda_fail(e); return e == cudaSuccess; };
    if (!check(g_pool.ensure())) { g_pool.release(); return rc; }
    for (int64_t c0 = 0, it = 0; c0 < n && rc == SH_OK; c0 += chunk, ++it) {
        const int b = (int)(it & 1);
        cudaStream_t st = g_pool.st[b];
        TI* dxyz = static_cast<TI*>(g_pool.din[b]);
        T* dout = static_cast<T*>(g_pool.dout[b]);
        const int64_t m = (n - c0) < chunk ? (n - c0) : chunk;
        // stream order makes slot b safe to reuse: its previous device->host copy precedes this host->device copy
        if (!check(cudaMemcpyAsync(dxyz, xyz + w * c0, (size_t)m * w * sizeof(TI), cudaMemcpyHostToDevice, st))) break;
        int r = run_device<KIND, T, TI>(dxyz, m, lmax, dout, layout_bits, st);
        if (r != SH_OK) { rc = r; break; }
        if (layout == SH_LAYOUT_AOS) {
            check(cudaMemcpyAsync(out + c0 * sp, dout, (size_t)m * sp * sizeof(T), cudaMemcpyDeviceToHost, st));
        } else {
            // device chunk is [ne][m] elements; host array is [ne][n]: one strided 2-D copy
            check(cudaMemcpy2DAsync(out + c0 * es, (size_t)n * es * sizeof(T), dout, (size_t)m * es * sizeof(T),
                                    (size_t)m * es * sizeof(T), (size_t)ne, cudaMemcpyDeviceToHost, st));
        }
    }
    for (int b = 0; b < 2; ++b) check(cudaStreamSynchronize(g_pool.st[b]));
    return rc;
}


}  // namespace shb200
