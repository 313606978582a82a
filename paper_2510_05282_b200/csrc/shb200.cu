// shb200.cu -- sm_100a kernels + C ABI (include/shb200.h) for batched spherical harmonics, l <= 9.
//
// Hot path per point (P:n = /root/reference/PAPER.md line n):
//   a1 load xyz (AoS [N][3])
//   a2 normalize: x, y, z <- (x, y, z)/r, r = 0 flag          P:58-69, Eq. 8
//   a3 azimuthal factors C_m, S_m (root-pair products)        Eq. 16, App. B
//   a4 polar factors Qhat_l^m(z) (root-pair products)         Eq. 14-15
//   a5 combine -> R_l^m, r = 0 convention                     Eq. 6
//   a6 complex Y_l^m                                          Eq. 5, 9, 10 P:42
//   a7 spinor harmonics                                       Eq. 7
//   a8 store: SoA planes by coalesced streaming stores; AoS rows staged in shared memory and written
//      by TMA bulk copies (cp.async.bulk.global.shared::cta) or by coalesced stores.
// a3/a4 building blocks and all constants come from the build-time generator (sh_generated.cuh).
//
// One thread evaluates one point; all (lmax+1)^2 values of a point are produced in ascending k by
// straight-line code, so the store sinks below see compile-time offsets only.
#include <cuda.h>   // CUtensorMap and the cuTensorMapEncodeTiled prototype only: the entry point is fetched through the runtime, libcuda is not linked
#include <cuda_runtime.h>

#include <atomic>
#include <cfloat>
#include <cstdint>
#include <cstring>
#include <mutex>
#include <type_traits>

#include "../../include/shb200.h"
#define SHGEN_FN __device__ __forceinline__
#define SHGEN_TABLE __constant__   /* recurrence tables of the l > 9 extension live in constant memory */
#include "sh_generated.cuh"

namespace {

constexpr int KIND_REAL = 0, KIND_COMPLEX = 1, KIND_SPINOR = 2;
constexpr int MODE_PLAIN = 0, MODE_ROWBULK = 1, MODE_TILEBULK = 2;

// ------------------------------------------------------------------------------------------------
// compile-time loop
template <int B, int E, class F>
__device__ __forceinline__ void static_for(F&& f) {
    if constexpr (B < E) {
        f(std::integral_constant<int, B>{});
        static_for<B + 1, E>(f);
    }
}

// ------------------------------------------------------------------------------------------------
// f2: two fp32 lanes = two POINTS per thread, on Blackwell's packed-fp32 pipe (PTX fma/mul/add .f32x2, SASS
// FFMA2/FMUL2/FADD2, sm_100+): one issue slot does the arithmetic of two points.  The generated templates are
// written against a generic T, so T = f2 needs only these operators.
struct f2 {
    float2 v;
    f2() = default;
    __device__ __forceinline__ explicit f2(float a, float b) : v(make_float2(a, b)) {}
    __device__ __forceinline__ explicit f2(double s) : v(make_float2((float)s, (float)s)) {}
    __device__ __forceinline__ explicit f2(int s) : v(make_float2((float)s, (float)s)) {}
};
__device__ __forceinline__ f2 operator*(f2 a, f2 b) { f2 r; r.v = __fmul2_rn(a.v, b.v); return r; }
__device__ __forceinline__ f2 operator+(f2 a, f2 b) { f2 r; r.v = __fadd2_rn(a.v, b.v); return r; }
__device__ __forceinline__ f2 operator-(f2 a, f2 b) { f2 r; r.v = __ffma2_rn(b.v, make_float2(-1.f, -1.f), a.v); return r; }  // exact: one rounding
__device__ __forceinline__ f2 operator-(f2 a) { return f2(-a.v.x, -a.v.y); }

// r = 0 flags of the point(s) a thread evaluates, and "zero where the point is the origin"
struct Origin2 { bool a, b; };
__device__ __forceinline__ double zero_where(bool o, double q) { return o ? 0.0 : q; }
__device__ __forceinline__ float zero_where(bool o, float q) { return o ? 0.f : q; }
__device__ __forceinline__ f2 zero_where(Origin2 o, f2 q) { return f2(o.a ? 0.f : q.v.x, o.b ? 0.f : q.v.y); }

// scalars (T) per element, elements per point
__host__ __device__ constexpr int elem_scalars(int kind) { return kind == KIND_REAL ? 1 : kind == KIND_COMPLEX ? 2 : 4; }
__host__ __device__ constexpr int elems_per_point(int kind, int lmax) {
    return (kind == KIND_SPINOR ? 2 : 1) * (lmax + 1) * (lmax + 1);
}
__host__ __device__ constexpr int scalars_per_point(int kind, int lmax) { return elem_scalars(kind) * elems_per_point(kind, lmax); }
// scalars of a point's row that precede the l-block
__host__ __device__ constexpr int cum_scalars(int kind, int l) { return (kind == KIND_REAL ? 1 : kind == KIND_COMPLEX ? 2 : 8) * l * l; }

// ------------------------------------------------------------------------------------------------
// a2: normalization.  fp64 always (also for the fp32 variant).
struct UnitVec {
    double x, y, z;
    bool origin;
};

__device__ __forceinline__ UnitVec normalize(double x, double y, double z) {
    // keep r^2 finite and normal over the whole fp64 range: scale by an exact power of two when needed
    const double s = fmax(fmax(fabs(x), fabs(y)), fabs(z));
    if (s < 0x1p-500) {
        x *= 0x1p600; y *= 0x1p600; z *= 0x1p600;
    } else if (s > 0x1p500) {
        x *= 0x1p-600; y *= 0x1p-600; z *= 0x1p-600;
    }
    const double r2 = x * x + y * y + z * z;
    UnitVec u;
    u.origin = (r2 == 0.0);
    double inv = 1.0 / sqrt(r2);                          // IEEE sqrt and divide
    if (u.origin) inv = 0.0;                              // r = 0: (0, 0, 0), handled by the evaluators
    if (!(r2 <= DBL_MAX)) inv = __longlong_as_double(0x7ff8000000000000LL);  // NaN / Inf input -> NaN outputs
    u.x = x * inv; u.y = y * inv; u.z = z * inv;
    return u;
}

// Normalized-Cartesian front end (the paper's fastest interface): the caller guarantees x^2+y^2+z^2 = 1
// (Eq. 8); a2 is skipped.  A zero vector selects the r = 0 convention.
__device__ __forceinline__ UnitVec as_given(double x, double y, double z) {
    UnitVec u;
    u.x = x; u.y = y; u.z = z;
    u.origin = (x == 0.0 && y == 0.0 && z == 0.0);
    return u;
}

// Angular front end: x = sin(theta) cos(phi), y = sin(theta) sin(phi), z = cos(theta).
__device__ __forceinline__ UnitVec from_angles(double theta, double phi) {
    double st, ct, sp, cp;
    sincos(theta, &st, &ct);
    sincos(phi, &sp, &cp);
    UnitVec u;
    u.x = st * cp; u.y = st * sp; u.z = ct;
    u.origin = false;
    return u;
}

// a1: one point of the AoS input.  Loaded one tile ahead of its use (software prefetch): under a saturated
// write stream the read latency is several microseconds, and nothing else in a warp's tile depends on memory.
template <typename TI, bool ANGULAR = false>
struct RawPoint {
    TI x, y, z;
    // coords: Cartesian / normalized Cartesian points are [n][3]; angular points are [n][2] = (theta, phi).
    // ANGULAR is a compile-time switch: the fp64 sincos slow path is a real function call, and kernels that contain
    // it get a much larger register allocation, so the Cartesian kernels must not.
    __device__ __forceinline__ void load(const TI* __restrict__ in, int64_t i) {
        if constexpr (ANGULAR) {
            const TI* p = in + 2 * i;
            x = __ldg(p); y = __ldg(p + 1); z = TI(0);
        } else {
            const TI* p = in + 3 * i;
            x = __ldg(p); y = __ldg(p + 1); z = __ldg(p + 2);
        }
    }
    __device__ __forceinline__ UnitVec unit(int coords) const {
        if constexpr (ANGULAR) return from_angles((double)x, (double)y);
        if (coords == SH_COORDS_NORMALIZED) return as_given((double)x, (double)y, (double)z);
        return normalize((double)x, (double)y, (double)z);
    }
};

// a1, second half: burst prefetch of the input into L2.  The 24 B/point of input are 3 % of the traffic, but read
// requests sprinkled into a saturated write stream cost ~4x their share (each one turns DRAM channels around:
// 241 -> 274 us on a store-only model of the lmax = 9 SoA kernel).  So reads are issued in bursts, far ahead of use:
// the grid is cut into windows of `win_ctas` consecutive CTAs; the first `spread` CTAs of window w (they start at about
// the same time on different SMs) prefetch the whole input of window w + 1 (window 0: of windows 0 and 1) into L2
// with evict_last priority -- the streaming evict-first stores of the outputs then do not push it out before the
// demand loads arrive (with normal priority they do: no gain measured).  A hint only: results never depend on it.
struct InputPrefetch {
    int win_ctas;   // 0 = off
    int spread;
};

__device__ __forceinline__ void prefetch_input_window(const void* in, int64_t total_bytes, int64_t bytes_per_cta, InputPrefetch pf) {
    if (pf.win_ctas <= 0) return;
    const int w = blockIdx.x / pf.win_ctas, r = blockIdx.x - w * pf.win_ctas;
    if (r >= pf.spread) return;
    const int64_t wbytes = (int64_t)pf.win_ctas * bytes_per_cta;
    int64_t lo = (int64_t)(w + 1) * wbytes;
    const int64_t hi = lo + wbytes < total_bytes ? lo + wbytes : total_bytes;
    if (w == 0) lo = 0;
    const char* base = static_cast<const char*>(in);
    const int64_t step = (int64_t)pf.spread * blockDim.x * 128;
    for (int64_t o = lo + ((int64_t)r * blockDim.x + threadIdx.x) * 128; o < hi; o += step)
        asm volatile("prefetch.global.L2::evict_last [%0];" ::"l"(base + o));
}

// ------------------------------------------------------------------------------------------------
// a3-a7: evaluators.  Sink interface: put1<K>(v) real element K; put2<K>(re, im) complex element K;
// put4<S>(ur, ui, dr, di) spinor element S; end_l<L>() after the last element of block l.
// REC = false: the factorized forms (root-pair products, Eq. 16).  REC = true: C_m + i S_m = (C_{m-1} + i S_{m-1})(x + i y),
// four instructions per m instead of ~17; used only by the FP64-bound projection when its fast form is requested.
template <int LMAX, typename T, bool REC = false>
struct Azim {
    T C[LMAX + 1], S[LMAX + 1];
    __device__ __forceinline__ Azim(T x, T y) {
        if constexpr (REC) {
            C[0] = T(1); S[0] = T(0);
            static_for<1, LMAX + 1>([&](auto mc) {
                constexpr int M = decltype(mc)::value;
                if constexpr (M == 1) { C[1] = x; S[1] = y; }
                else {
                    C[M] = C[M - 1] * x - S[M - 1] * y;
                    S[M] = C[M - 1] * y + S[M - 1] * x;
                }
            });
        } else {
            static_for<0, LMAX + 1>([&](auto mc) {
                constexpr int M = decltype(mc)::value;
                shgen::Azimuthal<M, T>::eval(x, y, C[M], S[M]);
            });
        }
    }
};

template <int LMAX, typename T, class O, class Sink>
__device__ __forceinline__ void eval_real(const Azim<LMAX, T>& az, T z, O origin, Sink& sink) {
    static_for<0, LMAX + 1>([&](auto lc) {
        constexpr int L = decltype(lc)::value;
        T q[L + 1];
        static_for<0, L + 1>([&](auto mc) {
            constexpr int M = decltype(mc)::value;
            constexpr double A = shgen::A_REAL[L][M];
            q[M] = T(A) * shgen::Polar<L, M, T>::eval(z);
        });
        // r = 0: x = y = z = 0 zeroes everything except the even-l, m = 0 polynomials (P_l(0) != 0)
        if constexpr (L > 0 && L % 2 == 0) q[0] = zero_where(origin, q[0]);
        sink.template polar<L>(q);   // the normalized polar factors of block l (seeds of the l > 9 recurrence)
        static_for<0, L>([&](auto jc) {
            constexpr int M = L - decltype(jc)::value;
            sink.template put1<L * (L + 1) - M>(q[M] * az.S[M]);
        });
        sink.template put1<L * (L + 1)>(q[0]);
        static_for<1, L + 1>([&](auto mc) {
            constexpr int M = decltype(mc)::value;
            sink.template put1<L * (L + 1) + M>(q[M] * az.C[M]);
        });
        sink.template end_l<L>();
    });
}

template <int LMAX, typename T, class O, class Sink>
__device__ __forceinline__ void eval_real(T x, T y, T z, O origin, Sink& sink) {
    const Azim<LMAX, T> az(x, y);
    eval_real<LMAX, T>(az, z, origin, sink);
}

// a[M] + i b[M] = B_lm Qhat_lm (C_M + i S_M);  Y_l^{-M} = (a, -b),  Y_l^{+M} = (-1)^M (a, b)
template <int L, int LMAX, typename T, class Sink>
__device__ __forceinline__ void complex_block(const Azim<LMAX, T>& az, T z, bool origin, T (&a)[L + 1], T (&b)[L + 1], Sink& sink) {
    T u[L + 1];
    static_for<0, L + 1>([&](auto mc) {
        constexpr int M = decltype(mc)::value;
        constexpr double B = shgen::B_CPLX[L][M];
        u[M] = T(B) * shgen::Polar<L, M, T>::eval(z);
    });
    if constexpr (L > 0 && L % 2 == 0) u[0] = zero_where(origin, u[0]);
    sink.template polar<L>(u);
    static_for<0, L + 1>([&](auto mc) {
        constexpr int M = decltype(mc)::value;
        a[M] = u[M] * az.C[M];
        b[M] = u[M] * az.S[M];
    });
}

template <int LMAX, typename T, class Sink>
__device__ __forceinline__ void eval_complex(const Azim<LMAX, T>& az, T z, bool origin, Sink& sink) {
    static_for<0, LMAX + 1>([&](auto lc) {
        constexpr int L = decltype(lc)::value;
        T a[L + 1], b[L + 1];
        complex_block<L>(az, z, origin, a, b, sink);
        static_for<0, L>([&](auto jc) {
            constexpr int M = L - decltype(jc)::value;
            sink.template put2<L * (L + 1) - M>(a[M], -b[M]);
        });
        sink.template put2<L * (L + 1)>(a[0], T(0));
        static_for<1, L + 1>([&](auto mc) {
            constexpr int M = decltype(mc)::value;
            if constexpr (M % 2) sink.template put2<L * (L + 1) + M>(-a[M], -b[M]);
            else sink.template put2<L * (L + 1) + M>(a[M], b[M]);
        });
        sink.template end_l<L>();
    });
}

template <int LMAX, typename T, class Sink>
__device__ __forceinline__ void eval_complex(T x, T y, T z, bool origin, Sink& sink) {
    const Azim<LMAX, T> az(x, y);
    eval_complex<LMAX, T>(az, z, origin, sink);
}

// component c * Y_l^m from the block's (a, b); c and the signs fold into one compile-time constant
template <int L, int M_SIGNED, typename T>
__device__ __forceinline__ void scaled_y(double c, const T (&a)[L + 1], const T (&b)[L + 1], T& re, T& im) {
    constexpr int M = M_SIGNED < 0 ? -M_SIGNED : M_SIGNED;
    if constexpr (M > L) {
        re = T(0); im = T(0);
    } else if constexpr (M_SIGNED < 0) {
        re = T(c) * a[M]; im = T(-c) * b[M];
    } else if constexpr (M_SIGNED == 0) {
        re = T(c) * a[0]; im = T(0);
    } else {
        const double s = (M % 2) ? -c : c;
        re = T(s) * a[M]; im = T(s) * b[M];
    }
}

template <int LMAX, typename T, class Sink>
__device__ __forceinline__ void eval_spinor(T x, T y, T z, bool origin, Sink& sink) {
    const Azim<LMAX, T> az(x, y);
    static_for<0, LMAX + 1>([&](auto lc) {
        constexpr int L = decltype(lc)::value;
        T a[L + 1], b[L + 1];
        complex_block<L>(az, z, origin, a, b, sink);
        static_for<2 * L * L, 2 * (L + 1) * (L + 1)>([&](auto sc) {
            constexpr int S = decltype(sc)::value;
            constexpr shgen::SpinorEntry e = shgen::SPINOR[S];
            static_assert(e.l == L, "spinor table order");
            T ur, ui, dr, di;
            scaled_y<L, e.m_up>(e.cu, a, b, ur, ui);
            scaled_y<L, e.m_dn>(e.cd, a, b, dr, di);
            sink.template put4<S>(ur, ui, dr, di);
        });
        sink.template end_l<L>();
    });
}

template <int KIND, int LMAX, typename T, class Sink>
__device__ __forceinline__ void evaluate(const UnitVec& u, Sink& sink) {
    const T x = (T)u.x, y = (T)u.y, z = (T)u.z;   // fp32 variant: rounded once, after the fp64 normalization
    if constexpr (KIND == KIND_REAL) eval_real<LMAX, T>(x, y, z, u.origin, sink);
    else if constexpr (KIND == KIND_COMPLEX) eval_complex<LMAX, T>(x, y, z, u.origin, sink);
    else eval_spinor<LMAX, T>(x, y, z, u.origin, sink);
}

// two points per thread (fp32 variant): fp64 normalization of each, rounded once, then packed-fp32 polynomials
template <int LMAX, class Sink>
__device__ __forceinline__ void evaluate_pair(const UnitVec& u0, const UnitVec& u1, Sink& sink) {
    const f2 x((float)u0.x, (float)u1.x), y((float)u0.y, (float)u1.y), z((float)u0.z, (float)u1.z);
    eval_real<LMAX, f2>(x, y, z, Origin2{u0.origin, u1.origin}, sink);
}

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

template <int KIND, int LMAX, typename T, typename TI, int VEC, bool ANGULAR>
__global__ void __launch_bounds__(256) sh_soa_kernel(const TI* __restrict__ xyz, int64_t n, T* __restrict__ out, int tiles_per_cta, int coords, InputPrefetch pf) {
    constexpr int ES = elem_scalars(KIND);
    constexpr int IN_BYTES = (ANGULAR ? 2 : 3) * sizeof(TI);
    prefetch_input_window(xyz, n * IN_BYTES, (int64_t)tiles_per_cta * 256 * IN_BYTES, pf);
    const int64_t ntiles = (n + 255) >> 8;
    int64_t t = (int64_t)blockIdx.x * tiles_per_cta;
    const int64_t tend = (t + tiles_per_cta < ntiles) ? t + tiles_per_cta : ntiles;
    int64_t i = (t << 8) + threadIdx.x;
    RawPoint<TI, ANGULAR> cur, nxt;
    bool have = i < n;
    if (have) cur.load(xyz, i);
    for (; t < tend; ++t, i += 256) {
        const bool have_next = (t + 1 < tend) && (i + 256 < n);
        if (have_next) nxt.load(xyz, i + 256);
        if (have) {
            SoASink<T, VEC> sink{out + i * ES, n * ES};
            evaluate<KIND, LMAX, T>(cur.unit(coords), sink);
        }
        cur = nxt;
        have = have_next;
    }
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// a8, SoA through the TMA tensor unit (real fp64).  One warp = one 32-point tile; lane i stages value k of its point at
// tile[k][i] (8-byte stores, 32 consecutive doubles per plane: conflict-free), and after a proxy fence lane 0 issues ONE
// cp.async.bulk.tensor.2d store of the box {32 points, K planes} through a tensor map of `out` viewed as [K][n]: K rows of
// 256 contiguous bytes, each two full 128-byte lines.  The LSU issues no global store at all (100 STG + their address
// arithmetic per point in sh_soa_kernel), and points past n in a ragged last tile are clipped by the tensor unit.
// One warp per CTA for the same reason as the AoS tile-bulk path (fence.proxy.async is CTA-scoped).
#ifndef SHB200_SOA_TMA_WARPS
#define SHB200_SOA_TMA_WARPS 4
#endif
// warps per CTA = 32-point groups per tile.  Longer rows are what the tile buys: 258 / 258 / 250 / 345 us for 1 / 2 / 4 / 8 warps
// (rows of 256 B .. 2 KB; 8 warps = one 205 KB tile per SM, nothing overlaps) on the 128^3 grid at lmax = 9.
// (The fp32 variant gains nothing from it -- 255 vs 257 us on 2^22 points -- and stays on sh_soa_pair_kernel.)
constexpr int SOA_TMA_WARPS = SHB200_SOA_TMA_WARPS;

template <int PTS>
struct TileSink {
    double* col;   // tile + this thread's point
    template <int K> __device__ __forceinline__ void put1(double v) { col[K * PTS] = v; }
    template <int L> __device__ __forceinline__ void end_l() {}
    template <int L> __device__ __forceinline__ void polar(const double (&)[L + 1]) {}
};

template <int LMAX, int WARPS>
__global__ void __launch_bounds__(32 * WARPS) sh_soa_tma_kernel(const double* __restrict__ xyz, int64_t n, const __grid_constant__ CUtensorMap tmap, int coords,
                                                                 InputPrefetch pf) {
    constexpr int PTS = 32 * WARPS;
    extern __shared__ __align__(128) unsigned char smem_tile[];
    prefetch_input_window(xyz, n * 24, (int64_t)PTS * 24, pf);
    double* tile = reinterpret_cast<double*>(smem_tile);
    const int64_t base = (int64_t)blockIdx.x * PTS, i = base + threadIdx.x;
    if (i < n) {
        RawPoint<double> pt;
        pt.load(xyz, i);
        TileSink<PTS> sink{tile + threadIdx.x};
        evaluate<KIND_REAL, LMAX, double>(pt.unit(coords), sink);
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // every thread: its staging stores -> async proxy
    if constexpr (WARPS == 1) __syncwarp();
    else __syncthreads();
    if (threadIdx.x == 0) {
        asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];" ::"l"(&tmap), "r"((int)base), "r"(0),
                     "r"(smem_u32(tile))
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
__global__ void __launch_bounds__(256) sh_soa_pair_kernel(const float* __restrict__ xyz, int64_t n, float* __restrict__ out, int tiles_per_cta, int coords, InputPrefetch pf) {
    prefetch_input_window(xyz, n * 12, (int64_t)tiles_per_cta * 512 * 12, pf);
    const int64_t npairs = n >> 1;
    const int64_t ntiles = (npairs + 255) >> 8;
    int64_t t = (int64_t)blockIdx.x * tiles_per_cta;
    const int64_t tend = (t + tiles_per_cta < ntiles) ? t + tiles_per_cta : ntiles;
    int64_t j = (t << 8) + threadIdx.x;
    auto load6 = [&](int64_t jj, float2& a, float2& b, float2& c) {
        const float2* q = reinterpret_cast<const float2*>(xyz + 6 * jj);   // 24 B per pair: three 8-byte loads
        a = __ldg(q); b = __ldg(q + 1); c = __ldg(q + 2);
    };
    float2 ca, cb, cc, na, nb, nc;
    bool have = j < npairs;
    if (have) load6(j, ca, cb, cc);
    for (; t < tend; ++t, j += 256) {
        const bool have_next = (t + 1 < tend) && (j + 256 < npairs);
        if (have_next) load6(j + 256, na, nb, nc);
        if (have) {
            SoAPairSink sink{out + 2 * j, n};
            if (coords == SH_COORDS_CARTESIAN) evaluate_pair<LMAX>(normalize(ca.x, ca.y, cb.x), normalize(cb.y, cc.x, cc.y), sink);
            else evaluate_pair<LMAX>(as_given(ca.x, ca.y, cb.x), as_given(cb.y, cc.x, cc.y), sink);
        }
        ca = na; cb = nb; cc = nc;
        have = have_next;
    }
}

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
                asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gout + i * SP + BEGIN),
                             "r"(smem_u32(row)), "r"(LEN * (int)sizeof(T))
                             : "memory");
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                if constexpr (L < LMAX) wait_reads();   // the row is reused by the next segment
            } else if constexpr (MODE == MODE_TILEBULK) {
                static_assert(LEN == SP && PITCH == SP, "tile-bulk mode stages whole dense rows");
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // every lane: its staging stores -> async proxy
                __syncwarp();
                const int bytes = rows * SP * (int)sizeof(T);
                if (bytes % 16 == 0) {   // always for a full tile; a ragged last tile with an odd scalar count is copied by the warp
                    if (lane == 0) {
                        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gout + base * SP),
                                     "r"(smem_u32(tile)), "r"(bytes)
                                     : "memory");
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

template <int KIND, int LMAX, typename T, typename TI, int CAP, int MODE, int WARPS, bool ANGULAR>
__global__ void __launch_bounds__(WARPS * 32) sh_aos_kernel(const TI* __restrict__ xyz, int64_t n, T* __restrict__ out, int tiles_per_warp, int coords, InputPrefetch pf) {
    using Sink = RowSink<KIND, LMAX, T, CAP, MODE>;
    constexpr int IN_BYTES = (ANGULAR ? 2 : 3) * sizeof(TI);
    prefetch_input_window(xyz, n * IN_BYTES, (int64_t)tiles_per_warp * WARPS * 32 * IN_BYTES, pf);
    static_assert(Sink::Seg::valid(), "CAP too small for one l-block group");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    T* tile = reinterpret_cast<T*>(smem_raw) + (size_t)warp * 32 * Sink::PITCH;
    const int64_t ntiles = (n + 31) >> 5;
    // warp w of CTA b owns tiles [(b*WARPS + w) * tiles_per_warp, +tiles_per_warp): a contiguous span of `out`
    int64_t t = ((int64_t)blockIdx.x * WARPS + warp) * tiles_per_warp;
    const int64_t tend = (t + tiles_per_warp < ntiles) ? t + tiles_per_warp : ntiles;
    // plain / tile-bulk mode: every lane takes part in the warp-level copy-out, so idle lanes of the last tile evaluate a clamped point
    auto point_of = [&](int64_t tt) {
        const int64_t i = (tt << 5) + lane;
        return (MODE != MODE_ROWBULK && i >= n) ? n - 1 : i;
    };
    RawPoint<TI, ANGULAR> cur, nxt;
    bool have = t < tend && point_of(t) < n;
    if (have) cur.load(xyz, point_of(t));
    for (; t < tend; ++t) {
        const bool have_next = (t + 1 < tend) && point_of(t + 1) < n;
        if (have_next) nxt.load(xyz, point_of(t + 1));
        if (have) {
            const int64_t base = t << 5;
            const int64_t left = n - base;
            Sink sink;
            sink.row = tile + lane * Sink::PITCH;
            sink.tile = tile;
            sink.gout = out;
            sink.base = base;
            sink.rows = left < 32 ? (int)left : 32;
            sink.lane = lane;
            sink.i = point_of(t);
            sink.wait_reads();   // bulk mode: the previous tile's copy has finished reading this lane's row
            evaluate<KIND, LMAX, T>(cur.unit(coords), sink);
        }
        cur = nxt;
        have = have_next;
    }
    if constexpr (MODE != MODE_PLAIN) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}

// ------------------------------------------------------------------------------------------------
// Fused projector consumer (the use case of P:14; include/shb200.h "Fused projector
// consumer"): beta_{p,m}(r_vec) = f_p(|r_vec|) R_{l_p}^m(r_vec/|r_vec|) with f_p piecewise linear on a uniform radial grid.
// The l-blocks are produced as above (a3-a5) and consumed in registers: each block is scaled by the radial value of
// every channel of that l and either stored (sh_projectors: only the requested columns, 8 ncols B/point) or contracted
// with the weight vectors (sh_project: nothing per point is written -- the path is then bound by the FP64 pipe).
// l-blocks no channel asks for are skipped by a warp-uniform branch.
struct ProjPlan {
    int ncols;                             // columns of this launch
    int nr;                                // radial table length
    double inv_dr;
    unsigned char first[shgen::LMAX_CAP + 2];   // channel slots of block l: [first[l], first[l+1])  (slots sorted by l)
    unsigned char chan[SH_MAX_PROJ];       // slot -> row of `radial`
    unsigned short col[SH_MAX_PROJ];       // slot -> first column of the channel in this launch's output
};

// position of |r| in the radial table: j = floor(r/dr), u = r/dr - j; beyond the table (and for NaN) `in` is false
struct RadialPos {
    int j;
    double u;
    bool in;
    __device__ __forceinline__ RadialPos(double x, double y, double z, const ProjPlan& plan) {
        const double r = sqrt(x * x + y * y + z * z);   // unscaled: 0 for r < 1e-162 (table start), +Inf beyond 1e154 (past any table)
        const double t = r * plan.inv_dr;
        in = t < (double)(plan.nr - 1);
        j = in ? (int)t : 0;
        u = in ? t - (double)j : 0.0;
    }
    __device__ __forceinline__ double f(const double* __restrict__ radial, int nr, int channel) const {
        const double* tab = radial + (int64_t)channel * nr + j;
        const double a = __ldg(tab), b = __ldg(tab + 1);
        return in ? fma(u, b - a, a) : 0.0;
    }
};

// Radial values of EVERY channel slot at this lane's point, computed up front and parked in shared memory as
// fs[slot*32 + lane] (times `scale`).  The table loads of different slots are independent, so their latencies overlap;
// loaded one l-block at a time instead, a warp pays one dependent L2 round trip per channel (the staging tiles leave
// little L1), which is what bounds the low-occupancy staging kernels (AoS sh_projectors 0.41 -> see DESIGN.md section 6).
__device__ __forceinline__ void stage_radial(const RadialPos& pos, const double* __restrict__ radial, const ProjPlan& plan, double* fs, int lane,
                                             double scale) {
    const int nslots = plan.first[shgen::LMAX_CAP + 1];
#pragma unroll 4
    for (int s = 0; s < nslots; ++s) fs[s * 32 + lane] = pos.f(radial, plan.nr, plan.chan[s]) * scale;
}

// the real harmonics of block l in ascending m (a3-a5), handed to the sink one block at a time
// FAST: Horner-in-z^2 polar factors and the azimuthal recurrence instead of the factorized forms -- ~35 % fewer FP64
// instructions, accuracy still two orders inside the tolerance; sh_project only, on request.
template <int LMAX, bool FAST = false, class Sink>
__device__ __forceinline__ void eval_projector_blocks(const UnitVec& u, const ProjPlan& plan, Sink& sink) {
    const Azim<LMAX, double, FAST> az(u.x, u.y);
    [[maybe_unused]] const double z2 = u.z * u.z;
    static_for<0, LMAX + 1>([&](auto lc) {
        constexpr int L = decltype(lc)::value;
        if (plan.first[L] != plan.first[L + 1]) {
            double blk[2 * L + 1];
            static_for<0, L + 1>([&](auto mc) {
                constexpr int M = decltype(mc)::value;
                constexpr double A = shgen::A_REAL[L][M];
                double q;
                if constexpr (FAST) q = A * shgen::PolarHorner<L, M, double>::eval(u.z, z2);
                else q = A * shgen::Polar<L, M, double>::eval(u.z);
                if constexpr (M == 0) {
                    if constexpr (L > 0 && L % 2 == 0) q = zero_where(u.origin, q);   // P_l(0) != 0: the r = 0 convention needs it
                    blk[L] = q;
                } else {
                    blk[L - M] = q * az.S[M];
                    blk[L + M] = q * az.C[M];
                }
            });
            sink.template block<L>(blk);
        }
    });
}

struct ProjSoASink {
    double* p;         // out + i
    int64_t n;
    const double* radial;
    const ProjPlan& plan;
    const RadialPos& pos;
    template <int L> __device__ __forceinline__ void block(const double (&blk)[2 * L + 1]) {
        for (int s = plan.first[L]; s < plan.first[L + 1]; ++s) {
            const double f = pos.f(radial, plan.nr, plan.chan[s]);
            double* q = p + (int64_t)plan.col[s] * n;
            static_for<0, 2 * L + 1>([&](auto mc) { __stcs(q + decltype(mc)::value * n, f * blk[decltype(mc)::value]); });
        }
    }
};

template <int LMAX>
__global__ void __launch_bounds__(256) sh_proj_soa_kernel(const double* __restrict__ xyz, int64_t n, const double* __restrict__ radial,
                                                           const __grid_constant__ ProjPlan plan, double* __restrict__ out, InputPrefetch pf) {
    prefetch_input_window(xyz, n * 24, (int64_t)256 * 24, pf);
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i >= n) return;
    RawPoint<double> pt;
    pt.load(xyz, i);
    const RadialPos pos(pt.x, pt.y, pt.z, plan);
    ProjSoASink sink{out + i, n, radial, plan, pos};
    eval_projector_blocks<LMAX>(pt.unit(SH_COORDS_CARTESIAN), plan, sink);
}

// sh_projectors, AoS: one warp = one 32-point tile.  Each lane stages its point's row in the warp's shared-memory tile
// with 8-byte stores at runtime column offsets; the tile is one contiguous span of `out`.  Copy-out, by `mode`:
//   PROJ_AOS_TILEBULK (`out` 16-byte aligned, ncols not a multiple of 8): rows staged densely (pitch = ncols; the 8-byte
//       staging stores conflict gcd(ncols, 16)-way, i.e. not at all for odd ncols), one TMA bulk copy
//       (cp.async.bulk.global.shared::cta) of the whole tile by lane 0; one warp per CTA (see TILEBULK_WARPS);
//   PROJ_AOS_ROWBULK (ncols a multiple of 8, `out` 16-byte aligned): pitch = ncols + 2 (rows stay 16-byte aligned, staging
//       stores conflict 2-way), one bulk copy per row by its lane (32 copies issued one after the other);
//   PROJ_AOS_PLAIN: pitch odd, the warp copies the tile out with coalesced streaming stores (any alignment, any width).
// A ragged last tile is always copied out by the warp.
constexpr int PROJ_AOS_PLAIN = 0, PROJ_AOS_ROWBULK = 1, PROJ_AOS_TILEBULK = 2;
struct ProjRowSink {
    double* row;
    const double* fs;   // this lane's radial values: fs[slot*32]
    const ProjPlan& plan;
    template <int L> __device__ __forceinline__ void block(const double (&blk)[2 * L + 1]) {
        for (int s = plan.first[L]; s < plan.first[L + 1]; ++s) {
            const double f = fs[s * 32];
            double* q = row + plan.col[s];
            static_for<0, 2 * L + 1>([&](auto mc) { q[decltype(mc)::value] = f * blk[decltype(mc)::value]; });
        }
    }
};

template <int LMAX>
__global__ void __launch_bounds__(128) sh_proj_aos_kernel(const double* __restrict__ xyz, int64_t n, const double* __restrict__ radial,
                                                           const __grid_constant__ ProjPlan plan, double* __restrict__ out, int pitch, int mode,
                                                           InputPrefetch pf) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, warps = blockDim.x >> 5;
    prefetch_input_window(xyz, n * 24, (int64_t)warps * 32 * 24, pf);
    const int ncols = plan.ncols;
    const int nslots = plan.first[shgen::LMAX_CAP + 1];
    double* tile = reinterpret_cast<double*>(smem_raw) + (size_t)warp * 32 * (pitch + nslots);
    double* fs = tile + 32 * pitch;   // radial values [slot][lane]
    const int64_t base = ((int64_t)blockIdx.x * warps + warp) << 5;
    if (base >= n) return;
    const int64_t i = base + lane;
    const int rows = (n - base) < 32 ? (int)(n - base) : 32;
    if (i < n) {
        RawPoint<double> pt;
        pt.load(xyz, i);
        const RadialPos pos(pt.x, pt.y, pt.z, plan);
        stage_radial(pos, radial, plan, fs, lane, 1.0);
        ProjRowSink sink{tile + lane * pitch, fs + lane, plan};
        eval_projector_blocks<LMAX>(pt.unit(SH_COORDS_CARTESIAN), plan, sink);
    }
    double* g = out + base * ncols;
    if (mode != PROJ_AOS_PLAIN && rows == 32) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // every lane: its staging stores -> async proxy
        if (mode == PROJ_AOS_TILEBULK) {
            __syncwarp();
            if (lane == 0)
                asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(g), "r"(smem_u32(tile)), "r"(32 * ncols * 8) : "memory");
        } else {
            asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(g + (int64_t)lane * ncols),
                         "r"(smem_u32(tile + lane * pitch)), "r"(ncols * 8)
                         : "memory");
        }
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // shared memory is released when the CTA exits
        return;
    }
    __syncwarp();
    const int total = rows * ncols;
    int r = 0, c = lane;
    while (c >= ncols) { c -= ncols; ++r; }
    for (int e = lane; e < total; e += 32) {
        __stcs(g + e, tile[r * pitch + c]);
        c += 32;
        while (c >= ncols) { c -= ncols; ++r; }
    }
}

// sh_project: coeff[v][col] = sum_i w[v][i] beta_col(r_i).  Nothing per point is written, so the FP64 pipe is the bound.
// One warp = one 32-point tile at a time, tiles dealt round-robin over all warps of a grid that fills the machine once;
// the next tile's point and weights are loaded before the current tile is evaluated.  The l-blocks a lane produces are
// staged, scaled by the radial values, in SEGMENTS of at most 32 columns (whole channels, packed in the order of
// production; segment plan in ProjSegments) in the warp's shared-memory tile, TRANSPOSED: tile[column][point], pitch 34
// doubles, so a lane's staging stores are conflict-free 8-byte stores (32 consecutive doubles per column) and, when a
// segment is complete, lane c sums column c over the 32 points with 16-byte loads (rows 272 B apart: eight lanes per
// 128-byte wavefront, conflict-free) and adds the result to the warp's running sums in shared memory.
//   NV = 1: the weight is folded into the radial value (beta w is staged), the column sum is 32 additions;
//   NV = 4: up to four weight vectors; the tile's weights sit in shared memory as [point][4] and are read as broadcasts.
// Idle lanes of a ragged last tile evaluate the point (0, 0, 1) with weight 0, so every column sum runs over 32 rows.
// Running sums are kept in the order of production ("slot order"); at the end a CTA adds its four warps in a fixed order
// and writes one row of `partial` [cta][nvec][ncols]; sh_project_reduce_kernel adds the rows in a fixed order and
// scatters to the caller's column order.
#ifndef SHB200_PROJ_CTAS_NV1
#define SHB200_PROJ_CTAS_NV1 4
#endif
#ifndef SHB200_PROJ_CTAS_NV4
#define SHB200_PROJ_CTAS_NV4 3
#endif
constexpr int PROJ_CTAS_NV1 = SHB200_PROJ_CTAS_NV1, PROJ_CTAS_NV4 = SHB200_PROJ_CTAS_NV4;   // resident CTAs per SM (__launch_bounds__): register budget
constexpr int PROJ_NV = 4;          // weight vectors contracted per launch
constexpr int PROJ_MAX_COLS = 128;  // columns per launch (whole channels); wider channel lists run as several launches
constexpr int PROJ_SEG_PITCH = 34;  // doubles between consecutive columns of the transposed segment tile
template <int NV> constexpr int project_smem_doubles_per_warp() {
    return 32 * PROJ_SEG_PITCH + NV * PROJ_MAX_COLS + (NV > 1 ? 32 * PROJ_NV : 0);   // tile, running sums, weights
}

struct ProjSegments {
    unsigned short scol[SH_MAX_PROJ];   // slot -> its first column in slot order
    unsigned short sbeg[SH_MAX_PROJ];   // slot -> first column (slot order) of the segment the slot belongs to
    unsigned char flush[SH_MAX_PROJ];   // slot -> 1 if the segment is complete after this slot
};

template <int NV>
struct ProjectSink {
    double* tile;        // the warp's [32][PROJ_SEG_PITCH] transposed segment tile
    double* sums;        // the warp's running sums [NV][PROJ_MAX_COLS]
    const double* wt;    // NV > 1: the tile's weights [32][PROJ_NV]
    const double* fs;    // this lane's radial values fs[slot*32] (NV = 1: times the lane's weight)
    const ProjPlan& plan;
    const ProjSegments& seg;
    int lane;

    __device__ __forceinline__ void flush(int begin, int len) {
        __syncwarp();
        if (lane < len) {
            const double2* t = reinterpret_cast<const double2*>(tile + lane * PROJ_SEG_PITCH);
            if constexpr (NV == 1) {
                double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
                for (int r = 0; r < 16; r += 2) {
                    const double2 a = t[r], b = t[r + 1];
                    s0 += a.x; s1 += a.y; s2 += b.x; s3 += b.y;
                }
                sums[begin + lane] += (s0 + s1) + (s2 + s3);
            } else {
                const double2* wv = reinterpret_cast<const double2*>(wt);   // row r: (w0, w1), (w2, w3)
                double e[PROJ_NV], o[PROJ_NV];
                static_for<0, PROJ_NV>([&](auto vc) { e[decltype(vc)::value] = 0.0; o[decltype(vc)::value] = 0.0; });
#pragma unroll
                for (int r = 0; r < 16; ++r) {
                    const double2 a = t[r];   // points 2r, 2r+1
                    const double2 w01 = wv[4 * r], w23 = wv[4 * r + 1], x01 = wv[4 * r + 2], x23 = wv[4 * r + 3];
                    e[0] = fma(a.x, w01.x, e[0]); e[1] = fma(a.x, w01.y, e[1]); e[2] = fma(a.x, w23.x, e[2]); e[3] = fma(a.x, w23.y, e[3]);
                    o[0] = fma(a.y, x01.x, o[0]); o[1] = fma(a.y, x01.y, o[1]); o[2] = fma(a.y, x23.x, o[2]); o[3] = fma(a.y, x23.y, o[3]);
                }
                static_for<0, PROJ_NV>([&](auto vc) {
                    constexpr int V = decltype(vc)::value;
                    sums[V * PROJ_MAX_COLS + begin + lane] += e[V] + o[V];
                });
            }
        }
        __syncwarp();
    }

    template <int L> __device__ __forceinline__ void block(const double (&blk)[2 * L + 1]) {
        for (int s = plan.first[L]; s < plan.first[L + 1]; ++s) {
            const double f = fs[s * 32];
            const int c0 = seg.scol[s], b0 = seg.sbeg[s];
            double* q = tile + (c0 - b0) * PROJ_SEG_PITCH + lane;
            static_for<0, 2 * L + 1>([&](auto mc) { q[decltype(mc)::value * PROJ_SEG_PITCH] = f * blk[decltype(mc)::value]; });
            if (seg.flush[s]) flush(b0, c0 + 2 * L + 1 - b0);
        }
    }
};

template <int LMAX, int NV, bool FAST>
__global__ void __launch_bounds__(128, NV == 1 ? PROJ_CTAS_NV1 : PROJ_CTAS_NV4) sh_project_kernel(const double* __restrict__ xyz, int64_t n, const double* __restrict__ radial,
                                                                          const __grid_constant__ ProjPlan plan, const __grid_constant__ ProjSegments seg,
                                                                          const double* __restrict__ w, int nvec, double* __restrict__ partial) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nslots = plan.first[shgen::LMAX_CAP + 1];
    double* s_tile = reinterpret_cast<double*>(smem_raw) + (size_t)warp * (project_smem_doubles_per_warp<NV>() + 32 * nslots);
    double* s_sums = s_tile + 32 * PROJ_SEG_PITCH;
    double* s_wt = s_sums + NV * PROJ_MAX_COLS;
    double* s_fs = s_tile + project_smem_doubles_per_warp<NV>();   // radial values [slot][lane]
    const int ncols = plan.ncols;
    for (int e = lane; e < NV * PROJ_MAX_COLS; e += 32) s_sums[e] = 0.0;
    const int64_t ntiles = (n + 31) >> 5;
    const int64_t gw = (int64_t)blockIdx.x * 4 + warp, nw = (int64_t)gridDim.x * 4;
    struct Item { double x, y, z, w[NV]; };
    auto load = [&](int64_t t, Item& it) {
        const int64_t i = (t << 5) + lane;
        if (i < n) {
            const double* p = xyz + 3 * i;
            it.x = __ldg(p); it.y = __ldg(p + 1); it.z = __ldg(p + 2);
            static_for<0, NV>([&](auto vc) {
                constexpr int V = decltype(vc)::value;
                it.w[V] = V < nvec ? __ldg(w + (int64_t)V * n + i) : 0.0;
            });
        } else {   // idle lane of the ragged last tile: a harmless point with weight 0
            it.x = 0.0; it.y = 0.0; it.z = 1.0;
            static_for<0, NV>([&](auto vc) { it.w[decltype(vc)::value] = 0.0; });
        }
    };
    Item cur, nxt;
    int64_t t = gw;
    if (t < ntiles) load(t, cur);
    for (; t < ntiles; t += nw) {
        if (t + nw < ntiles) load(t + nw, nxt);
        if constexpr (NV > 1) {
            // the previous tile's last column sum ended with __syncwarp: the weights may be overwritten
            reinterpret_cast<double2*>(s_wt)[2 * lane] = make_double2(cur.w[0], cur.w[1]);
            reinterpret_cast<double2*>(s_wt)[2 * lane + 1] = make_double2(cur.w[2], cur.w[3]);
        }
        const RadialPos pos(cur.x, cur.y, cur.z, plan);
        stage_radial(pos, radial, plan, s_fs, lane, NV == 1 ? cur.w[0] : 1.0);   // only this lane reads its column back
        ProjectSink<NV> sink{s_tile, s_sums, s_wt, s_fs + lane, plan, seg, lane};
        eval_projector_blocks<LMAX, FAST>(normalize(cur.x, cur.y, cur.z), plan, sink);
        cur = nxt;
    }
    // the CTA's four warps are added in a fixed order: one row of `partial` per CTA
    __syncthreads();
    const size_t wstride = project_smem_doubles_per_warp<NV>() + 32 * nslots;
    const double* s0 = reinterpret_cast<const double*>(smem_raw) + 32 * PROJ_SEG_PITCH;
    for (int e = threadIdx.x; e < nvec * ncols; e += 128) {
        const int v = e / ncols, c = e - v * ncols;
        const double* q = s0 + v * PROJ_MAX_COLS + c;
        partial[(int64_t)blockIdx.x * nvec * ncols + e] = ((q[0] + q[wstride]) + q[2 * wstride]) + q[3 * wstride];
    }
}

// coeff[v*coeff_stride + user column] = sum over CTAs of partial[cta][v][slot-order column], the rows added in a fixed
// order (reproducible): 32 lanes = 32 consecutive (v, column) elements; the block's 32 warps each add every 32nd row of
// `partial` (coalesced, four loads in flight), then the 32 sums are added in order.
__global__ void __launch_bounds__(1024) sh_project_reduce_kernel(const double* __restrict__ partial, int nrows, int nvec, const __grid_constant__ ProjPlan plan,
                                                                  const __grid_constant__ ProjSegments seg, double* __restrict__ coeff, int coeff_stride) {
    __shared__ double s[32][33];
    const int ncols = plan.ncols, ne = nvec * ncols;
    const int y = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int e = blockIdx.x * 32 + lane;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    if (e < ne) {
        int g = y;
        for (; g + 96 < nrows; g += 128) {
            a0 += partial[(int64_t)g * ne + e];
            a1 += partial[(int64_t)(g + 32) * ne + e];
            a2 += partial[(int64_t)(g + 64) * ne + e];
            a3 += partial[(int64_t)(g + 96) * ne + e];
        }
        for (; g < nrows; g += 32) a0 += partial[(int64_t)g * ne + e];
    }
    s[y][lane] = (a0 + a1) + (a2 + a3);
    __syncthreads();
    if (y == 0 && e < ne) {
        double t = 0.0;
        for (int k = 0; k < 32; ++k) t += s[k][lane];
        // slot-order column -> the caller's column
        const int v = e / ncols, c = e - v * ncols;
        int slot = 0;
        const int nslots = plan.first[shgen::LMAX_CAP + 1];
        while (slot + 1 < nslots && seg.scol[slot + 1] <= c) ++slot;
        coeff[v * coeff_stride + plan.col[slot] + (c - seg.scol[slot])] = t;
    }
}

// ------------------------------------------------------------------------------------------------
// host side
std::atomic<int64_t> g_launches{0};
thread_local char g_cuda_error[256] = "";

int cuda_fail(cudaError_t e) {
    std::strncpy(g_cuda_error, cudaGetErrorString(e), sizeof(g_cuda_error) - 1);
    return SH_ERR_CUDA;
}

int sm_count() {
    static int sms = 0;
    if (!sms) {
        int dev = 0, v = 0;
        if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0)
            sms = v;
        else
            return 148;
    }
    return sms;
}

// launch-heuristic overrides (sh_set_tuning); 0 = default
std::atomic<int> g_tune[8];

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

template <int KIND, int LMAX, typename T, typename TI, int VEC, bool ANGULAR = false>
int launch_soa(const TI* xyz, int64_t n, T* out, int coords, cudaStream_t st) {
    const int64_t tiles = (n + 255) / 256;
    // one 256-point tile per CTA: with the burst L2 prefetch the input load is an L2 hit, and a deep grid lets the
    // hardware CTA scheduler balance the SMs (251 vs 256 / 258 us for 1 / 2 / 4 tiles on the 128^3 grid at lmax = 9).
    // With more tiles per CTA the next tile's input is loaded before the current tile is evaluated.
    int tpc = tuned(SH_TUNE_SOA_TILES_PER_CTA, 1);
    while (tpc > 1 && tiles / tpc < (int64_t)sm_count() * 16) tpc >>= 1;
    const int64_t blocks = (tiles + tpc - 1) / tpc;
    if (blocks > 0x7fffffffLL) return SH_ERR_COUNT;
    sh_soa_kernel<KIND, LMAX, T, TI, VEC, ANGULAR><<<(unsigned)blocks, 256, 0, st>>>(xyz, n, out, tpc, coords, prefetch_plan(n, (int64_t)tpc * 256));
    g_launches.fetch_add(1, std::memory_order_relaxed);
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SH_OK : cuda_fail(e);
}

inline bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

// cuTensorMapEncodeTiled through the runtime's driver entry point lookup (no link against libcuda); nullptr if unavailable
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                   const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled() {
    static EncodeTiledFn fn = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess) p = nullptr;
        return reinterpret_cast<EncodeTiledFn>(p);
    }();
    return fn;
}

// SoA through the tensor unit: `out` as a 2-D tensor [K][n] of fp64 (row pitch 8n bytes must be a multiple of 16: n even),
// box {points per tile, K}.  Returns SH_ERR_ALIGNMENT when this launch cannot use the path (the caller then takes sh_soa_kernel).
template <int LMAX>
int launch_soa_tma(const double* xyz, int64_t n, double* out, int coords, cudaStream_t st) {
    constexpr int K = (LMAX + 1) * (LMAX + 1);
    constexpr int PTS = 32 * SOA_TMA_WARPS;
    EncodeTiledFn enc = encode_tiled();
    if (!enc || (n & 1) || n < PTS || n > 0x7fffff00LL || !aligned(out, 16)) return SH_ERR_ALIGNMENT;
    CUtensorMap tmap;
    const cuuint64_t gdim[2] = {(cuuint64_t)n, (cuuint64_t)K};
    const cuuint64_t gstride[1] = {(cuuint64_t)n * sizeof(double)};
    const cuuint32_t box[2] = {PTS, (cuuint32_t)K}, estride[2] = {1, 1};
    if (enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, out, gdim, gstride, box, estride, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
            CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return SH_ERR_ALIGNMENT;
    const int64_t blocks = (n + PTS - 1) / PTS;
    constexpr size_t smem = (size_t)K * PTS * sizeof(double);
    static_assert(smem <= 227 * 1024, "tile exceeds shared memory");
    auto kern = sh_soa_tma_kernel<LMAX, SOA_TMA_WARPS>;
    if constexpr (smem > 48 * 1024) {
        static bool opted_in = false;
        if (!opted_in) {
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (e != cudaSuccess) return cuda_fail(e);
            opted_in = true;
        }
    }
    kern<<<(unsigned)blocks, PTS, smem, st>>>(xyz, n, tmap, coords, prefetch_plan(n, PTS));
    g_launches.fetch_add(1, std::memory_order_relaxed);
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SH_OK : cuda_fail(e);
}

// staging capacity per row, in scalars: whole rows for real (800 B at lmax = 9) and complex (1600 B);
// spinor rows (6400 B) are staged in groups of l-blocks of at most 1600 B
template <int KIND, int LMAX>
constexpr int aos_cap() {
    return KIND == KIND_SPINOR ? (200 > 8 * (2 * LMAX + 1) ? 200 : 8 * (2 * LMAX + 1)) : scalars_per_point(KIND, LMAX);
}

// tile-bulk mode: ONE warp per CTA (fence.proxy.async is CTA-scoped: with several warps per CTA each warp's fence also
// waits for the other warps' copies in flight -- 4.3 vs 7.4 TB/s on a store-only model with 51.2 KB tiles), at least
// four CTAs per SM, i.e. whole rows of a 32-point tile staged densely in <= 55 KB (complex lmax = 9: 51.2 KB), and
// staging stores that conflict at most 4-way: 16-byte stores of a quarter warp land gcd(row_bytes/16, 8) deep; rows that
// are not multiples of 16 B are staged with scalar stores, conflict-free because the row is then an odd number of words
#ifndef SHB200_TILEBULK_WARPS
#define SHB200_TILEBULK_WARPS 1
#endif
#ifndef SHB200_TILEBULK_MAX_CONFLICT
#define SHB200_TILEBULK_MAX_CONFLICT 4
#endif
constexpr int TILEBULK_WARPS = SHB200_TILEBULK_WARPS;
template <int KIND, int LMAX, typename T>
constexpr bool tile_bulk_ok() {
    constexpr int row_bytes = scalars_per_point(KIND, LMAX) * (int)sizeof(T);
    if (KIND == KIND_SPINOR || TILEBULK_WARPS * 32 * row_bytes > 55 * 1024) return false;
    if (row_bytes % 16 != 0) return true;
    int chunks = row_bytes / 16, g = 8;
    while (chunks % g) g >>= 1;
    return g <= SHB200_TILEBULK_MAX_CONFLICT;
}

template <int KIND, int LMAX, typename T, typename TI, int MODE, bool ANGULAR = false>
int launch_aos(const TI* xyz, int64_t n, T* out, int coords, cudaStream_t st) {
    constexpr int CAP = aos_cap<KIND, LMAX>();
    constexpr int WARPS = MODE == MODE_TILEBULK ? TILEBULK_WARPS : 4;
    using Sink = RowSink<KIND, LMAX, T, CAP, MODE>;
    constexpr size_t smem = (size_t)WARPS * 32 * Sink::PITCH * sizeof(T);
    static_assert(smem <= 227 * 1024, "staging tile exceeds shared memory");
    auto kern = sh_aos_kernel<KIND, LMAX, T, TI, CAP, MODE, WARPS, ANGULAR>;
    static int ctas_per_sm = 0;   // idempotent cache of a pure function of the kernel
    if (!ctas_per_sm) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return cuda_fail(e);
        int occ = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, WARPS * 32, smem);
        if (e != cudaSuccess) return cuda_fail(e);
        ctas_per_sm = occ > 0 ? occ : 1;
    }
    const int64_t ntiles = (n + 31) / 32;
    // one tile per warp measured fastest on every bulk path now that the input arrives by the burst L2 prefetch
    // (real tile-bulk 238 / 242 / 249 us, spinor row-bulk 1002 / 1028 / 1064 us for 1 / 2 / 4 tiles per warp); with more
    // tiles per warp the next tile's input is loaded before the current tile is evaluated
    int tpw = tuned(SH_TUNE_AOS_TILES_PER_WARP, 1);
    while (tpw > 1 && ntiles / ((int64_t)WARPS * tpw) < (int64_t)sm_count() * ctas_per_sm * 4) tpw >>= 1;
    const int64_t blocks = (ntiles + (int64_t)WARPS * tpw - 1) / ((int64_t)WARPS * tpw);
    if (blocks > 0x7fffffffLL) return SH_ERR_COUNT;
    kern<<<(unsigned)blocks, WARPS * 32, smem, st>>>(xyz, n, out, tpw, coords, prefetch_plan(n, (int64_t)tpw * WARPS * 32));
    g_launches.fetch_add(1, std::memory_order_relaxed);
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SH_OK : cuda_fail(e);
}

template <int LMAX>
int launch_soa_pair(const float* xyz, int64_t n, float* out, int coords, cudaStream_t st) {
    const int64_t tiles = ((n >> 1) + 255) / 256;
    int tpc = tuned(SH_TUNE_SOA_TILES_PER_CTA, 1);
    while (tpc > 1 && tiles / tpc < (int64_t)sm_count() * 16) tpc >>= 1;
    const int64_t blocks = (tiles + tpc - 1) / tpc;
    if (blocks > 0x7fffffffLL) return SH_ERR_COUNT;
    sh_soa_pair_kernel<LMAX><<<(unsigned)blocks, 256, 0, st>>>(xyz, n, out, tpc, coords, prefetch_plan(n, (int64_t)tpc * 512));
    g_launches.fetch_add(1, std::memory_order_relaxed);
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SH_OK : cuda_fail(e);
}

template <int KIND, int LMAX, typename T, typename TI>
int dispatch_lmax(const TI* xyz, int64_t n, T* out, int layout, int path, int coords, cudaStream_t st) {
    constexpr int SP = scalars_per_point(KIND, LMAX);
    constexpr bool F32 = std::is_same<T, float>::value && KIND == KIND_REAL;
    if (coords == SH_COORDS_ANGULAR) {
        // angular front end: trigonometry dominates; it is served by the generic store paths only (scalar SoA stores,
        // AoS staging + coalesced copy-out), which are valid for every alignment
        if (path == SH_STORE_BULK) return SH_ERR_ALIGNMENT;
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
        if constexpr (F32) {
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
#ifndef SHB200_DEV_ONLY_LMAX9   /* development builds may compile the lmax = 9 kernels only */
        SH_CASE(0) SH_CASE(1) SH_CASE(2) SH_CASE(3) SH_CASE(4) SH_CASE(5) SH_CASE(6) SH_CASE(7) SH_CASE(8)
#endif
        SH_CASE(9)
#undef SH_CASE
    }
    return SH_ERR_LMAX;
}

// l > 9 extension (sh_real_ext / sh_complex_ext): lmax <= 9 is the regular path; above, SoA only
template <int KIND>
int run_device_ext(const double* xyz, int64_t n, int lmax, double* out, int layout_bits, void* stream) {
    if (lmax <= shgen::LMAX_CAP) return run_device<KIND, double, double>(xyz, n, lmax, out, layout_bits, stream);
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
    g_launches.fetch_add(1, std::memory_order_relaxed);
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SH_OK : cuda_fail(e);
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
HostPool g_pool;

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

// ---- fused projector consumer, host side ----
// ncols of a channel list, or -1
int projector_count(int nproj, const int* proj_l) {
    if (nproj < 0 || nproj > SH_MAX_PROJ || (nproj > 0 && !proj_l)) return -1;
    int ncols = 0;
    for (int p = 0; p < nproj; ++p) {
        if (proj_l[p] < 0 || proj_l[p] > shgen::LMAX_CAP) return -1;
        ncols += 2 * proj_l[p] + 1;
    }
    return ncols;
}

// plan for the channels [p0, p1): slots sorted by l, columns relative to the first column of channel p0; returns the largest l
int make_plan(const int* proj_l, int p0, int p1, int nr, double dr, ProjPlan& plan) {
    std::memset(&plan, 0, sizeof(plan));
    plan.nr = nr;
    plan.inv_dr = 1.0 / dr;
    int col0[SH_MAX_PROJ], ncols = 0, lmax = 0;
    for (int p = p0; p < p1; ++p) {
        col0[p] = ncols;
        ncols += 2 * proj_l[p] + 1;
        if (proj_l[p] > lmax) lmax = proj_l[p];
    }
    plan.ncols = ncols;
    int slot = 0;
    for (int l = 0; l <= shgen::LMAX_CAP; ++l) {
        plan.first[l] = (unsigned char)slot;
        for (int p = p0; p < p1; ++p)
            if (proj_l[p] == l) {
                plan.chan[slot] = (unsigned char)p;
                plan.col[slot] = (unsigned short)col0[p];
                ++slot;
            }
    }
    plan.first[shgen::LMAX_CAP + 1] = (unsigned char)slot;
    return lmax;
}

int check_projector_args(const double* xyz, int64_t n, int nproj, const int* proj_l, const double* radial, int nr, double dr) {
    if (n < 0) return SH_ERR_COUNT;
    if (projector_count(nproj, proj_l) < 0 || nr < 2 || !(dr > 0.0) || !(1.0 / dr > 0.0) || !(1.0 / dr <= DBL_MAX)) return SH_ERR_PROJECTOR;
    if (n > 0 && (!xyz || (nproj > 0 && !radial))) return SH_ERR_NULL;
    if (!aligned(xyz, 8) || !aligned(radial, 8)) return SH_ERR_ALIGNMENT;
    return SH_OK;
}

constexpr int PROJ_CTAS_PER_SM = PROJ_CTAS_NV1 > PROJ_CTAS_NV4 ? PROJ_CTAS_NV1 : PROJ_CTAS_NV4;   // grid cap of sh_project_kernel: the machine filled once (what the workspace is sized for)

template <int LMAX>
int launch_proj_aos(const double* xyz, int64_t n, const double* radial, const ProjPlan& plan, double* out, cudaStream_t st) {
    auto kern = sh_proj_aos_kernel<LMAX>;
    const int ncols = plan.ncols;
    // store mode (see the kernel): bulk copies need a 16-byte aligned `out` and a tile that leaves room for >= 4 CTAs per SM
    int mode = PROJ_AOS_PLAIN, pitch = ncols | 1, warps = 4;
    if (aligned(out, 16) && (size_t)32 * (ncols + 2 + plan.first[shgen::LMAX_CAP + 1]) * sizeof(double) <= (size_t)55 * 1024) {
        // dense rows conflict gcd(ncols, 16)-way on the 8-byte staging stores (16 lanes per wavefront, rows ncols words apart)
        int g = 16;
        while (ncols % g) g >>= 1;
        mode = g <= 4 ? PROJ_AOS_TILEBULK : PROJ_AOS_ROWBULK;
        const int force = tuned(SH_TUNE_PROJ_AOS_MODE, 0);
        if (force == 1) mode = PROJ_AOS_PLAIN;
        else if (force == 2 && ncols % 2 == 0) mode = PROJ_AOS_ROWBULK;
        else if (force == 3) mode = PROJ_AOS_TILEBULK;
        if (mode == PROJ_AOS_TILEBULK) pitch = ncols;
        else if (mode == PROJ_AOS_ROWBULK) pitch = (ncols / 2) & 1 ? ncols : ncols + 2;
        if (mode != PROJ_AOS_PLAIN) warps = TILEBULK_WARPS;   // fence.proxy.async is CTA-scoped: one warp per CTA keeps the warps' copies independent
    }
    const size_t per_warp = (size_t)32 * (pitch + plan.first[shgen::LMAX_CAP + 1]) * sizeof(double);   // row tile + radial values
    while (warps > 1 && warps * per_warp > (size_t)56 * 1024) warps >>= 1;   // four CTAs per SM while the row width allows it
    const size_t smem = warps * per_warp;
    if (smem > (size_t)227 * 1024) return SH_ERR_PROJECTOR;
    static size_t smem_set = 0;   // the opt-in limit only ever grows
    if (smem > 48 * 1024 && smem > smem_set) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return cuda_fail(e);
        smem_set = smem;
    }
    const int64_t ntiles = (n + 31) / 32;
    const int64_t blocks = (ntiles + warps - 1) / warps;
    if (blocks > 0x7fffffffLL) return SH_ERR_COUNT;
    kern<<<(unsigned)blocks, warps * 32, smem, st>>>(xyz, n, radial, plan, out, pitch, mode, prefetch_plan(n, (int64_t)warps * 32));
    g_launches.fetch_add(1, std::memory_order_relaxed);
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SH_OK : cuda_fail(e);
}

template <int LMAX>
int launch_proj_soa(const double* xyz, int64_t n, const double* radial, const ProjPlan& plan, double* out, cudaStream_t st) {
    const int64_t blocks = (n + 255) / 256;
    if (blocks > 0x7fffffffLL) return SH_ERR_COUNT;
    sh_proj_soa_kernel<LMAX><<<(unsigned)blocks, 256, 0, st>>>(xyz, n, radial, plan, out, prefetch_plan(n, 256));
    g_launches.fetch_add(1, std::memory_order_relaxed);
    cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SH_OK : cuda_fail(e);
}

int run_projectors(const double* xyz, int64_t n, int nproj, const int* proj_l, const double* radial, int nr, double dr, double* out,
                   int layout_bits, void* stream) {
    int rc = check_projector_args(xyz, n, nproj, proj_l, radial, nr, dr);
    if (rc != SH_OK) return rc;
    if (layout_bits != SH_LAYOUT_AOS && layout_bits != SH_LAYOUT_SOA) return SH_ERR_LAYOUT;   // Cartesian points, automatic store path
    if (n == 0 || nproj == 0) return SH_OK;
    if (!out) return SH_ERR_NULL;
    if (!aligned(out, 8)) return SH_ERR_ALIGNMENT;
    ProjPlan plan;
    const int lmax = make_plan(proj_l, 0, nproj, nr, dr, plan);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    switch (lmax) {
#define SH_CASE(L) case L: return layout_bits == SH_LAYOUT_SOA ? launch_proj_soa<L>(xyz, n, radial, plan, out, st) \
                                                             : launch_proj_aos<L>(xyz, n, radial, plan, out, st);
#ifndef SHB200_DEV_ONLY_LMAX9
        SH_CASE(0) SH_CASE(1) SH_CASE(2) SH_CASE(4) SH_CASE(5) SH_CASE(6) SH_CASE(7) SH_CASE(8)
#endif
        SH_CASE(3) SH_CASE(9)
#undef SH_CASE
    }
    return SH_ERR_PROJECTOR;
}

// segments of at most 32 columns, whole channels, packed greedily in slot order (the order of production)
void make_segments(const int* proj_l, const ProjPlan& plan, ProjSegments& seg) {
    std::memset(&seg, 0, sizeof(seg));
    const int nslots = plan.first[shgen::LMAX_CAP + 1];
    int col = 0, beg = 0;
    for (int s = 0; s < nslots; ++s) {
        const int len = 2 * proj_l[plan.chan[s]] + 1;
        if (col + len - beg > 32) {
            seg.flush[s - 1] = 1;
            beg = col;
        }
        seg.scol[s] = (unsigned short)col;
        seg.sbeg[s] = (unsigned short)beg;
        col += len;
    }
    if (nslots > 0) seg.flush[nslots - 1] = 1;
}

int64_t project_workspace_bytes(int ncols, int nvec) {
    if (ncols < 0 || nvec < 0) return -1;
    const int64_t cols = ncols < PROJ_MAX_COLS ? ncols : PROJ_MAX_COLS, vecs = nvec < PROJ_NV ? nvec : PROJ_NV;
    return (int64_t)sm_count() * PROJ_CTAS_PER_SM * vecs * cols * (int64_t)sizeof(double);   // one row per CTA of the largest grid
}

template <int LMAX>
int launch_project(const double* xyz, int64_t n, const double* radial, const ProjPlan& plan, const ProjSegments& seg, const double* w, int nvec,
                   double* partial, double* coeff, int coeff_stride, cudaStream_t st) {
    const int64_t ntiles = (n + 31) / 32;
    int64_t blocks = (ntiles + 3) / 4;
    const int64_t cap = (int64_t)sm_count() * (nvec == 1 ? PROJ_CTAS_NV1 : PROJ_CTAS_NV4);   // resident CTAs per SM (__launch_bounds__)
    if (blocks > cap) blocks = cap;
    // per warp: segment tile, running sums, (weights,) and the radial values of every slot: 38 / 54 KB + 1 KB per slot per CTA
    const size_t slots_bytes = (size_t)4 * 32 * plan.first[shgen::LMAX_CAP + 1] * sizeof(double);
    constexpr size_t smem_max = (size_t)4 * (project_smem_doubles_per_warp<PROJ_NV>() + 32 * SH_MAX_PROJ) * sizeof(double);   // 86 KB
    const bool fast = tuned(SH_TUNE_PROJECT_FORM, 0) == 1;   // Horner / recurrence forms instead of the factorized ones
    auto launch = [&](auto kern, size_t warp_doubles, bool& opted_in) -> int {
        if (!opted_in) {
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_max);
            if (e != cudaSuccess) return cuda_fail(e);
            opted_in = true;
        }
        kern<<<(unsigned)blocks, 128, (size_t)4 * warp_doubles * sizeof(double) + slots_bytes, st>>>(xyz, n, radial, plan, seg, w, nvec, partial);
        return SH_OK;
    };
    static bool opted_in[4] = {false, false, false, false};
    int rc;
    if (nvec == 1) {
        rc = fast ? launch(sh_project_kernel<LMAX, 1, true>, project_smem_doubles_per_warp<1>(), opted_in[1])
                  : launch(sh_project_kernel<LMAX, 1, false>, project_smem_doubles_per_warp<1>(), opted_in[0]);
    } else {
        rc = fast ? launch(sh_project_kernel<LMAX, PROJ_NV, true>, project_smem_doubles_per_warp<PROJ_NV>(), opted_in[3])
                  : launch(sh_project_kernel<LMAX, PROJ_NV, false>, project_smem_doubles_per_warp<PROJ_NV>(), opted_in[2]);
    }
    if (rc != SH_OK) return rc;
    g_launches.fetch_add(1, std::memory_order_relaxed);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    const int elems = nvec * plan.ncols;
    sh_project_reduce_kernel<<<(elems + 31) / 32, 1024, 0, st>>>(partial, (int)blocks, nvec, plan, seg, coeff, coeff_stride);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    e = cudaGetLastError();
    return e == cudaSuccess ? SH_OK : cuda_fail(e);
}

int run_project(const double* xyz, int64_t n, int nproj, const int* proj_l, const double* radial, int nr, double dr, const double* w,
                int nvec, double* coeff, void* workspace, int64_t workspace_bytes, void* stream) {
    int rc = check_projector_args(xyz, n, nproj, proj_l, radial, nr, dr);
    if (rc != SH_OK) return rc;
    if (nvec < 0) return SH_ERR_PROJECTOR;
    const int ncols = projector_count(nproj, proj_l);
    if (nvec == 0 || ncols == 0) return SH_OK;
    if (!coeff || (n > 0 && !w)) return SH_ERR_NULL;
    if (!aligned(coeff, 8) || !aligned(w, 8) || !aligned(workspace, 8)) return SH_ERR_ALIGNMENT;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (n == 0) {   // the empty sum
        cudaError_t e = cudaMemsetAsync(coeff, 0, (size_t)nvec * ncols * sizeof(double), st);
        return e == cudaSuccess ? SH_OK : cuda_fail(e);
    }
    if (!workspace || workspace_bytes < project_workspace_bytes(ncols, nvec)) return SH_ERR_PROJECTOR;
    double* partial = static_cast<double*>(workspace);
    // a launch covers at most PROJ_MAX_COLS columns (whole channels) and PROJ_NV weight vectors; the workspace is reused in stream order
    for (int p0 = 0, c0 = 0; p0 < nproj;) {
        int p1 = p0, cols = 0;
        while (p1 < nproj && cols + 2 * proj_l[p1] + 1 <= PROJ_MAX_COLS) cols += 2 * proj_l[p1++] + 1;
        ProjPlan plan;
        ProjSegments seg;
        const int lmax = make_plan(proj_l, p0, p1, nr, dr, plan);
        make_segments(proj_l, plan, seg);
        for (int v0 = 0; v0 < nvec; v0 += PROJ_NV) {
            const int nv = nvec - v0 < PROJ_NV ? nvec - v0 : PROJ_NV;
            switch (lmax) {
#define SH_CASE(L) case L: rc = launch_project<L>(xyz, n, radial, plan, seg, w + (int64_t)v0 * n, nv, partial, coeff + (int64_t)v0 * ncols + c0, ncols, st); break;
#ifndef SHB200_DEV_ONLY_LMAX9
                SH_CASE(0) SH_CASE(1) SH_CASE(2) SH_CASE(4) SH_CASE(5) SH_CASE(6) SH_CASE(7) SH_CASE(8)
#endif
                SH_CASE(3) SH_CASE(9)
#undef SH_CASE
            }
            if (rc != SH_OK) return rc;
        }
        p0 = p1;
        c0 += cols;
    }
    return SH_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------------
extern "C" {

int sh_real(const double* xyz, int64_t n, int lmax, double* out, int layout, void* stream) {
    return run_device<KIND_REAL, double, double>(xyz, n, lmax, out, layout, stream);
}
int sh_complex(const double* xyz, int64_t n, int lmax, double* out, int layout, void* stream) {
    return run_device<KIND_COMPLEX, double, double>(xyz, n, lmax, out, layout, stream);
}
int sh_spinor(const double* xyz, int64_t n, int lmax, double* out, int layout, void* stream) {
    return run_device<KIND_SPINOR, double, double>(xyz, n, lmax, out, layout, stream);
}
int sh_real_f32(const float* xyz, int64_t n, int lmax, float* out, int layout, void* stream) {
    return run_device<KIND_REAL, float, float>(xyz, n, lmax, out, layout, stream);
}

int sh_real_ext(const double* xyz, int64_t n, int lmax, double* out, int layout, void* stream) {
    return run_device_ext<KIND_REAL>(xyz, n, lmax, out, layout, stream);
}
int sh_complex_ext(const double* xyz, int64_t n, int lmax, double* out, int layout, void* stream) {
    return run_device_ext<KIND_COMPLEX>(xyz, n, lmax, out, layout, stream);
}
int sh_lmax_ext(void) { return shgen::LMAX_EXT; }

int sh_projector_count(int nproj, const int* proj_l) { return projector_count(nproj, proj_l); }
int64_t sh_project_workspace_bytes(int ncols, int nvec) { return project_workspace_bytes(ncols, nvec); }
int sh_projectors(const double* xyz, int64_t n, int nproj, const int* proj_l, const double* radial, int nr, double dr, double* out,
                  int layout, void* stream) {
    return run_projectors(xyz, n, nproj, proj_l, radial, nr, dr, out, layout, stream);
}
int sh_project(const double* xyz, int64_t n, int nproj, const int* proj_l, const double* radial, int nr, double dr, const double* w,
               int nvec, double* coeff, void* workspace, int64_t workspace_bytes, void* stream) {
    return run_project(xyz, n, nproj, proj_l, radial, nr, dr, w, nvec, coeff, workspace, workspace_bytes, stream);
}

int sh_real_host(const double* xyz, int64_t n, int lmax, double* out, int layout) {
    return run_host<KIND_REAL, double, double>(xyz, n, lmax, out, layout);
}
int sh_complex_host(const double* xyz, int64_t n, int lmax, double* out, int layout) {
    return run_host<KIND_COMPLEX, double, double>(xyz, n, lmax, out, layout);
}
int sh_spinor_host(const double* xyz, int64_t n, int lmax, double* out, int layout) {
    return run_host<KIND_SPINOR, double, double>(xyz, n, lmax, out, layout);
}
int sh_real_f32_host(const float* xyz, int64_t n, int lmax, float* out, int layout) {
    return run_host<KIND_REAL, float, float>(xyz, n, lmax, out, layout);
}

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
