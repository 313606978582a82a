// sh_core.cuh -- shared by every translation unit of libshb200.so (include/shb200.h): the per-point evaluation (steps
// a1-a7 of SURVEY.md section 8a) and the small host-side state the launchers share.
//
// Hot path per point (P:n = /root/reference/PAPER.md line n):
//   a1 load xyz (AoS [N][3])
//   a2 normalize: x, y, z <- (x, y, z)/r, r = 0 flag          P:58-69, Eq. 8
//   a3 azimuthal factors C_m, S_m (root-pair products)        Eq. 16, App. B
//   a4 polar factors Qhat_l^m(z) (root-pair products)         Eq. 14-15
//   a5 combine -> R_l^m, r = 0 convention                     Eq. 6
//   a6 complex Y_l^m                                          Eq. 5, 9, 10 P:42
//   a7 spinor harmonics                                       Eq. 7
//   a8 store                                                  sh_store.cuh (sh_real / sh_complex / sh_spinor / sh_real_f32),
//                                                             sh_ext.cu (l > 9), sh_projector.cu (fused consumer)
// a3/a4 building blocks and all constants come from the build-time generator (sh_generated.cuh).
//
// One thread evaluates one point; all (lmax+1)^2 values of a point are produced in ascending k by
// straight-line code, so the store sinks see compile-time offsets only.
//
// Translation units (compiled in parallel by build.py): sh_real.cu, sh_complex.cu, sh_spinor.cu, sh_real_f32.cu (one kind
// each), sh_ext.cu, sh_projector.cu, sh_abi.cu (shared host state and the small entry points).
#pragma once
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
#define SHGEN_TABLE static __constant__   /* recurrence tables of the l > 9 extension live in constant memory (of the unit that uses them) */
#include "sh_generated.cuh"

namespace shb200 {

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

// a2 for the fp32 variant (fp32 coordinates in, unit vector rounded once to fp32).  The fp64 range scaling is not needed (the square of
// any fp32 value, subnormals included, is a normal fp64 number), and 1/sqrt comes from the fp64 rsqrt (reciprocal-square-root seed + Newton
// steps, <= 2 ulp in fp64: nine orders below the rounding to fp32 that follows) instead of an IEEE sqrt and an IEEE divide, which together
// are ~150 instructions -- a third of this variant's instruction stream when two warps share a point group.  Results are defined by
// SURVEY.md 8c #21 ("normalization in fp64, rounded once to fp32") and by the 1e-5 tolerance; r = 0, NaN and Inf as in normalize().
__device__ __forceinline__ UnitVec normalize_f32in(float xf, float yf, float zf) {
    const double x = xf, y = yf, z = zf;
    const double r2 = x * x + y * y + z * z;
    UnitVec u;
    u.origin = (r2 == 0.0);
    double inv = rsqrt(r2);
    if (u.origin) inv = 0.0;
    if (!(r2 <= DBL_MAX)) inv = __longlong_as_double(0x7ff8000000000000LL);
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
        if constexpr (std::is_same<TI, float>::value) return normalize_f32in(x, y, z);
        else return normalize((double)x, (double)y, (double)z);
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

// block l of the real harmonics, m = -l..l, from the azimuthal factors (MAZ >= L of them)
template <int L, int MAZ, typename T, class O, class Sink>
__device__ __forceinline__ void real_block(const Azim<MAZ, T>& az, T z, O origin, Sink& sink) {
    static_assert(MAZ >= L, "azimuthal factors up to m = l");
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
}

template <int LMAX, typename T, class O, class Sink>
__device__ __forceinline__ void eval_real(const Azim<LMAX, T>& az, T z, O origin, Sink& sink) {
    static_for<0, LMAX + 1>([&](auto lc) { real_block<decltype(lc)::value>(az, z, origin, sink); });
}

template <int LMAX, typename T, class O, class Sink>
__device__ __forceinline__ void eval_real(T x, T y, T z, O origin, Sink& sink) {
    const Azim<LMAX, T> az(x, y);
    eval_real<LMAX, T>(az, z, origin, sink);
}

// Several warps may share the points of one tile, warp `PART` of `SPLIT` evaluating the l-blocks with
// block_part<SPLIT>(l) == PART: a2/a3 are repeated per warp, the chain of dependent instructions per tile is cut SPLIT-fold.
// The parts are balanced in work (~l^2 per block) and in values (2l+1): for two warps {0, 3, 4, 7, 8} | {1, 2, 5, 6, 9},
// 49 | 51 values at lmax = 9.
template <int SPLIT>
__host__ __device__ constexpr int block_part(int l) {
    if (SPLIT == 2) return ((l + 1) >> 1) & 1;
    if (SPLIT == 4) { constexpr int t[10] = {2, 1, 1, 3, 2, 3, 3, 2, 1, 0}; return t[l % 10]; }   // {9} {8,2,1} {7,4,0} {6,5,3}
    return 0;
}
template <int SPLIT, int PART, int LMAX>
constexpr int part_mmax() {   // largest m the part's blocks need
    int m = 0;
    for (int l = 0; l <= LMAX; ++l)
        if (block_part<SPLIT>(l) == PART) m = l;
    return m;
}

template <int LMAX, int SPLIT, int PART, typename T, class O, class Sink>
__device__ __forceinline__ void eval_real_part(T x, T y, T z, O origin, Sink& sink) {
    const Azim<part_mmax<SPLIT, PART, LMAX>(), T> az(x, y);
    static_for<0, LMAX + 1>([&](auto lc) {
        constexpr int L = decltype(lc)::value;
        if constexpr (block_part<SPLIT>(L) == PART) real_block<L>(az, z, origin, sink);
    });
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

// block l of the complex harmonics, m = -l..l, from the azimuthal factors (MAZ >= L of them)
template <int L, int MAZ, typename T, class Sink>
__device__ __forceinline__ void complex_emit_block(const Azim<MAZ, T>& az, T z, bool origin, Sink& sink) {
    static_assert(MAZ >= L, "azimuthal factors up to m = l");
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
}

template <int LMAX, typename T, class Sink>
__device__ __forceinline__ void eval_complex(const Azim<LMAX, T>& az, T z, bool origin, Sink& sink) {
    static_for<0, LMAX + 1>([&](auto lc) { complex_emit_block<decltype(lc)::value>(az, z, origin, sink); });
}

// warp part PART of SPLIT (block_part, as eval_real_part)
template <int LMAX, int SPLIT, int PART, typename T, class Sink>
__device__ __forceinline__ void eval_complex_part(T x, T y, T z, bool origin, Sink& sink) {
    const Azim<part_mmax<SPLIT, PART, LMAX>(), T> az(x, y);
    static_for<0, LMAX + 1>([&](auto lc) {
        constexpr int L = decltype(lc)::value;
        if constexpr (block_part<SPLIT>(L) == PART) complex_emit_block<L>(az, z, origin, sink);
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

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// TMA bulk store shared -> global (cp.async.bulk, one bulk group per call site's commit).  The output is never re-read,
// so its lines carry the L2 evict-first policy, like the st.global.cs of the LSU store paths: they leave L2 ahead of the
// evict-last input prefetch and in the order they were written (without the hint: +1-3 % time).
__device__ __forceinline__ uint64_t l2_evict_first_policy() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void bulk_store(void* gdst, const void* ssrc, int bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(gdst), "r"(smem_u32(ssrc)), "r"(bytes),
                 "l"(l2_evict_first_policy())
                 : "memory");
}

// ------------------------------------------------------------------------------------------------
// host side, shared by the translation units (defined in sh_abi.cu)
extern std::atomic<int64_t> g_launches;   // kernels launched (sh_kernel_launch_count)
int cuda_fail(cudaError_t e);             // records the CUDA error text, returns SH_ERR_CUDA
int sm_count();
int tuned(int knob, int dflt);            // launch-heuristic overrides (sh_set_tuning); 0 = default
InputPrefetch prefetch_plan(int64_t n, int64_t points_per_cta);   // window plan of the burst input prefetch
inline bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

// counts the launch just issued and maps its status
inline int launch_status() {
    g_launches.fetch_add(1, std::memory_order_relaxed);
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? SH_OK : cuda_fail(e);
}

// A small per-device cache of a pure function of (kernel, device): 0 = not computed yet.  Racing threads compute the same value.
struct PerDeviceInt {
    std::atomic<int> v[64];   // static storage: zero-initialised
    template <class F> int get(F&& compute) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess) return compute();
        std::atomic<int>& slot = v[dev & 63];
        int x = slot.load(std::memory_order_relaxed);
        if (x <= 0) {
            x = compute();
            if (x > 0) slot.store(x, std::memory_order_relaxed);
        }
        return x;
    }
};

// Dynamic shared memory above 48 KB is an opt-in per kernel AND per device (cudaFuncSetAttribute acts on the current device):
// the largest size granted so far is remembered per device, so a process that drives several GPUs opts in on each.
struct SmemOptIn {
    std::atomic<size_t> granted[64];   // static storage: zero-initialised
};
template <class Kernel>
inline int ensure_dynamic_smem(Kernel kern, size_t bytes, SmemOptIn& state) {
    if (bytes <= 48 * 1024) return SH_OK;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e);
    std::atomic<size_t>& slot = state.granted[dev & 63];
    if (slot.load(std::memory_order_relaxed) >= bytes) return SH_OK;
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
    if (e != cudaSuccess) return cuda_fail(e);
    slot.store(bytes, std::memory_order_relaxed);
    return SH_OK;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point lookup (no link against libcuda); nullptr if unavailable
using EncodeTiledFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                   const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled();

// tile-bulk mode: ONE warp per CTA (fence.proxy.async is CTA-scoped: with several warps per CTA each warp's fence also
// waits for the other warps' copies in flight -- 4.3 vs 7.4 TB/s on a store-only model with 51.2 KB tiles), at least
// four CTAs per SM, i.e. whole rows of a 32-point tile staged densely in <= 55 KB (complex lmax = 9: 51.2 KB), and
// staging stores that conflict at most 4-way: 16-byte stores of a quarter warp land gcd(row_bytes/16, 8) deep; rows that
// are not multiples of 16 B are staged with scalar stores, conflict-free because the row is then an odd number of words
constexpr int TILEBULK_WARPS = 1;
constexpr int TILEBULK_MAX_CONFLICT = 4;

}  // namespace shb200
