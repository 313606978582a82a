// sh_projector.cu -- sh_projectors / sh_project (include/shb200.h): the fused projector consumer.
#include "sh_core.cuh"

namespace shb200 {

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
// little L1).  sh_project uses this; sh_proj_aos_kernel shares the slots among the warps of its tile the same way.
__device__ __forceinline__ void stage_radial(const RadialPos& pos, const double* __restrict__ radial, const ProjPlan& plan, double* fs, int lane,
                                             double scale) {
    const int nslots = plan.first[shgen::LMAX_CAP + 1];
#pragma unroll 4
    for (int s = 0; s < nslots; ++s) fs[s * 32 + lane] = pos.f(radial, plan.nr, plan.chan[s]) * scale;
}

// the real harmonics of block l in ascending m (a3-a5), handed to the sink one block at a time
// FAST: Horner-in-z^2 polar factors and the azimuthal recurrence instead of the factorized forms -- ~35 % fewer FP64
// instructions, accuracy still two orders inside the tolerance; sh_project only, on request.
template <int LMAX, bool FAST = false, int SPLIT = 1, int PART = 0, class Sink>
__device__ __forceinline__ void eval_projector_blocks(const UnitVec& u, const ProjPlan& plan, Sink& sink) {
    constexpr int MMAX = part_mmax<SPLIT, PART, LMAX>();
    const Azim<MMAX, double, FAST> az(u.x, u.y);
    [[maybe_unused]] const double z2 = u.z * u.z;
    static_for<0, LMAX + 1>([&](auto lc) {
        constexpr int L = decltype(lc)::value;
        if constexpr (block_part<SPLIT>(L) == PART) {
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
#pragma unroll 1   // code size is instruction-fetch traffic (see ProjRowSink)
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

// sh_projectors, AoS: one CTA = one 32-point tile = SPLIT warps; lane i of every warp takes point i of the tile, and warp w
// evaluates the l-blocks of part w (block_part): a2/a3 are repeated per warp, but a tile's chain of dependent FP64
// instructions is cut SPLIT-fold.  That chain, not the store, is what bounds this kernel: shared memory caps an SM at
// eight 25.6 KB tiles (100 columns), and with one warp per tile that is two warps per scheduler running ~2200
// instructions per tile at one issue every ~6 cycles.  Each lane stages its point's columns in the tile with 8-byte
// stores at runtime column offsets; the tile is one contiguous span of `out`.  Copy-out, by `mode`:
//   PROJ_AOS_TILEBULK (`out` 16-byte aligned, ncols not a multiple of 8): rows staged densely (pitch = ncols; the 8-byte
//       staging stores conflict gcd(ncols, 16)-way, i.e. not at all for odd ncols), one TMA bulk copy
//       (cp.async.bulk.global.shared::cta) of the whole tile by thread 0; one tile per CTA, so the CTA-scoped
//       fence.proxy.async never waits for another tile's copy;
//   PROJ_AOS_ROWBULK (ncols a multiple of 8, `out` 16-byte aligned): pitch = ncols + 2 (rows stay 16-byte aligned, staging
//       stores conflict 2-way), one bulk copy per row by the lanes of warp 0 (32 copies issued one after the other);
//   PROJ_AOS_PLAIN: pitch odd, the CTA copies the tile out with coalesced streaming stores (any alignment, any width).
// A ragged last tile is always copied out by the CTA; its idle lanes evaluate the last point.
constexpr int PROJ_AOS_PLAIN = 0, PROJ_AOS_ROWBULK = 1, PROJ_AOS_TILEBULK = 2;
struct ProjRowSink {
    double* row;
    const double* fs;   // this lane's radial values: fs[slot*32]
    const ProjPlan& plan;
    template <int L> __device__ __forceinline__ void block(const double (&blk)[2 * L + 1]) {
        // not unrolled: the kernel is straight-line code that every warp runs through once per tile, so its size is
        // instruction-fetch traffic (4096 -> ~2300 SASS instructions at lmax = 9)
#pragma unroll 1
        for (int s = plan.first[L]; s < plan.first[L + 1]; ++s) {
            const double f = fs[s * 32];
            double* q = row + plan.col[s];
            static_for<0, 2 * L + 1>([&](auto mc) { q[decltype(mc)::value] = f * blk[decltype(mc)::value]; });
        }
    }
};

template <int LMAX, int SPLIT>
__global__ void __launch_bounds__(32 * SPLIT) sh_proj_aos_kernel(const double* __restrict__ xyz, int64_t n, const double* __restrict__ radial,
                                                                  const __grid_constant__ ProjPlan plan, double* __restrict__ out, int pitch, int mode,
                                                                  InputPrefetch pf) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    prefetch_input_window(xyz, n * 24, (int64_t)32 * 24, pf);
    const int ncols = plan.ncols;
    const int nslots = plan.first[shgen::LMAX_CAP + 1];
    double* tile = reinterpret_cast<double*>(smem_raw);
    double* fs = tile + 32 * pitch;   // radial values [slot][lane]
    const int64_t base = (int64_t)blockIdx.x << 5;
    const int rows = (n - base) < 32 ? (int)(n - base) : 32;
    const int64_t i = lane < rows ? base + lane : n - 1;
    RawPoint<double> pt;
    pt.load(xyz, i);
    const RadialPos pos(pt.x, pt.y, pt.z, plan);
    // radial values of every channel slot at this lane's point: the warps share the slots (independent table loads overlap)
#pragma unroll 4
    for (int s = warp; s < nslots; s += SPLIT) fs[s * 32 + lane] = pos.f(radial, plan.nr, plan.chan[s]);
    if constexpr (SPLIT > 1) __syncthreads();
    else __syncwarp();
    const UnitVec u = pt.unit(SH_COORDS_CARTESIAN);
    ProjRowSink sink{tile + lane * pitch, fs + lane, plan};
    static_for<0, SPLIT>([&](auto pc) {
        constexpr int PART = decltype(pc)::value;
        if (warp == PART) eval_projector_blocks<LMAX, false, SPLIT, PART>(u, plan, sink);
    });
    double* g = out + base * ncols;
    const bool bulk = mode != PROJ_AOS_PLAIN && rows == 32;
    if (bulk) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // every thread: its staging stores -> async proxy
    if constexpr (SPLIT > 1) __syncthreads();
    else __syncwarp();
    if (bulk) {
        if (warp != 0) return;
        if (mode == PROJ_AOS_TILEBULK) {
            if (lane == 0)
                bulk_store(g, tile, 32 * ncols * 8);
        } else {
            bulk_store(g + (int64_t)lane * ncols, tile + lane * pitch, ncols * 8);
        }
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // shared memory is released when the CTA exits
        return;
    }
    const int total = rows * ncols;
    int r = 0, c = threadIdx.x;
    while (c >= ncols) { c -= ncols; ++r; }
    for (int e = threadIdx.x; e < total; e += 32 * SPLIT) {
        __stcs(g + e, tile[r * pitch + c]);
        c += 32 * SPLIT;
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
constexpr int PROJ_CTAS_NV1 = 4, PROJ_CTAS_NV4 = 3;   // resident CTAs per SM (__launch_bounds__): register budget
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

// column sums of a complete segment, added to the warp's running sums
template <int NV>
__device__ __forceinline__ void project_flush(double* tile, double* sums, const double* wt, int lane, int begin, int len) {
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

__device__ __noinline__ void project_flush_call(double* tile, double* sums, const double* wt, int lane, int begin, int len) {
    project_flush<PROJ_NV>(tile, sums, wt, lane, begin, len);
}

template <int NV>
struct ProjectSink {
    double* tile;        // the warp's [32][PROJ_SEG_PITCH] transposed segment tile
    double* sums;        // the warp's running sums [NV][PROJ_MAX_COLS]
    const double* wt;    // NV > 1: the tile's weights [32][PROJ_NV]
    const double* fs;    // this lane's radial values fs[slot*32] (NV = 1: times the lane's weight)
    const ProjPlan& plan;
    const ProjSegments& seg;
    int lane;

    // NV = 4: out of line.  Inlined after every l-block its 210 instructions stand ten times in code that a warp runs through
    // once per tile (4744 -> 2552 SASS instructions at lmax 9; 0.334 -> 0.327 ms on the 128^3 grid).  The 36 instructions of
    // NV = 1 stay inline (the call costs more than the fetches: 0.189 -> 0.202 ms out of line).
    __device__ __forceinline__ void flush(int begin, int len) {
        if constexpr (NV == 1) project_flush<1>(tile, sums, wt, lane, begin, len);
        else project_flush_call(tile, sums, wt, lane, begin, len);
    }

    template <int L> __device__ __forceinline__ void block(const double (&blk)[2 * L + 1]) {
#pragma unroll 1   // code size is instruction-fetch traffic (see ProjRowSink)
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

// warps per tile (block_part): the default comes from the 128^3-grid measurements in DESIGN.md section 6
constexpr int PROJ_AOS_SPLIT = 2;

template <int LMAX, int SPLIT>
int launch_proj_aos_split(const double* xyz, int64_t n, const double* radial, const ProjPlan& plan, double* out, int pitch, int mode, size_t smem,
                          cudaStream_t st) {
    auto kern = sh_proj_aos_kernel<LMAX, SPLIT>;
    static SmemOptIn opted_in;   // the opt-in limit only ever grows
    if (const int rc = ensure_dynamic_smem(kern, smem, opted_in); rc != SH_OK) return rc;
    const int64_t ntiles = (n + 31) / 32;
    if (ntiles > 0x7fffffffLL) return SH_ERR_COUNT;
    kern<<<(unsigned)ntiles, 32 * SPLIT, smem, st>>>(xyz, n, radial, plan, out, pitch, mode, prefetch_plan(n, 32));
    return launch_status();
}

template <int LMAX>
int launch_proj_aos(const double* xyz, int64_t n, const double* radial, const ProjPlan& plan, double* out, cudaStream_t st) {
    const int ncols = plan.ncols;
    // store mode (see the kernel): bulk copies need a 16-byte aligned `out` and a tile that leaves room for >= 4 CTAs per SM
    int mode = PROJ_AOS_PLAIN, pitch = ncols | 1;
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
    }
    const size_t smem = (size_t)32 * (pitch + plan.first[shgen::LMAX_CAP + 1]) * sizeof(double);   // row tile + radial values
    if (smem > (size_t)227 * 1024) return SH_ERR_PROJECTOR;
    // warps per tile: splitting pays once there are several l-blocks to share
    int split = LMAX >= 4 ? tuned(SH_TUNE_PROJ_AOS_SPLIT, PROJ_AOS_SPLIT) : 1;
    if constexpr (LMAX >= 4) {
        if (split >= 4) return launch_proj_aos_split<LMAX, 4>(xyz, n, radial, plan, out, pitch, mode, smem, st);
        if (split >= 2) return launch_proj_aos_split<LMAX, 2>(xyz, n, radial, plan, out, pitch, mode, smem, st);
    }
    (void)split;
    return launch_proj_aos_split<LMAX, 1>(xyz, n, radial, plan, out, pitch, mode, smem, st);
}

template <int LMAX>
int launch_proj_soa(const double* xyz, int64_t n, const double* radial, const ProjPlan& plan, double* out, cudaStream_t st) {
    const int64_t blocks = (n + 255) / 256;
    if (blocks > 0x7fffffffLL) return SH_ERR_COUNT;
    sh_proj_soa_kernel<LMAX><<<(unsigned)blocks, 256, 0, st>>>(xyz, n, radial, plan, out, prefetch_plan(n, 256));
    return launch_status();
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
        SH_CASE(0) SH_CASE(1) SH_CASE(2) SH_CASE(3) SH_CASE(4) SH_CASE(5) SH_CASE(6) SH_CASE(7) SH_CASE(8) SH_CASE(9)
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
    const bool fast = tuned(SH_TUNE_PROJECT_FORM, 1) != 2;   // Horner / recurrence forms (default) or the factorized ones (knob value 2)
    auto launch = [&](auto kern, size_t warp_doubles, SmemOptIn& opted_in) -> int {
        if (const int rc = ensure_dynamic_smem(kern, smem_max, opted_in); rc != SH_OK) return rc;
        kern<<<(unsigned)blocks, 128, (size_t)4 * warp_doubles * sizeof(double) + slots_bytes, st>>>(xyz, n, radial, plan, seg, w, nvec, partial);
        return SH_OK;
    };
    static SmemOptIn opted_in[4];
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
                SH_CASE(0) SH_CASE(1) SH_CASE(2) SH_CASE(3) SH_CASE(4) SH_CASE(5) SH_CASE(6) SH_CASE(7) SH_CASE(8) SH_CASE(9)
#undef SH_CASE
            }
            if (rc != SH_OK) return rc;
        }
        p0 = p1;
        c0 += cols;
    }
    return SH_OK;
}


}  // namespace shb200

using namespace shb200;

extern "C" {

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

}  // extern "C"
