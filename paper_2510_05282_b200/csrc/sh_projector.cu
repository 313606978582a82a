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
    unsigned char part_first[5];           // sh_project: slots of warp part p are part_slots[part_first[p] .. part_first[p+1])
    unsigned char part_slots[SH_MAX_PROJ];
    int row[SH_MAX_PROJ];                  // slot -> offset of its row in `radial` (chan * nr)
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
    __device__ __forceinline__ double f_row(const double* __restrict__ tab) const {
        const double a = __ldg(tab + j), b = __ldg(tab + j + 1);
        return in ? fma(u, b - a, a) : 0.0;
    }
    __device__ __forceinline__ double f(const double* __restrict__ radial, int nr, int channel) const {
        const double* tab = radial + (int64_t)channel * nr + j;
        const double a = __ldg(tab), b = __ldg(tab + 1);
        return in ? fma(u, b - a, a) : 0.0;
    }
};

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
// PAIRS (rows of an even number of doubles: every row keeps 16-byte alignment): the 2l + 1 values of a channel go out as l 16-byte
// stores and one 8-byte store, from an even or an odd start column (warp-uniform branch).  With dense 800-byte rows the 32 lanes of an
// 8-byte staging store land on 4 bank pairs -- 8 wavefronts instead of 2, ~800 per tile, and ncu showed the shared-memory pipe (7.6-way
// conflicts on 7.2 M store requests), not the store stream, bounding this kernel; a 16-byte store of the same lanes takes 8 wavefronts
// for twice the data: 0.258 -> 0.237 ms on the 128^3 grid with 100 columns, the rate of sh_real AoS.
template <bool PAIRS>
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
            const int c = plan.col[s];
            double* q = row + c;
            if constexpr (!PAIRS || L == 0) {
                static_for<0, 2 * L + 1>([&](auto mc) { q[decltype(mc)::value] = f * blk[decltype(mc)::value]; });
            } else if ((c & 1) == 0) {
                static_for<0, L>([&](auto jc) {
                    constexpr int J = 2 * decltype(jc)::value;
                    *reinterpret_cast<double2*>(q + J) = make_double2(f * blk[J], f * blk[J + 1]);
                });
                q[2 * L] = f * blk[2 * L];
            } else {
                q[0] = f * blk[0];
                static_for<0, L>([&](auto jc) {
                    constexpr int J = 1 + 2 * decltype(jc)::value;
                    *reinterpret_cast<double2*>(q + J) = make_double2(f * blk[J], f * blk[J + 1]);
                });
            }
        }
    }
};

template <int LMAX, int SPLIT, bool PAIRS>
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
    ProjRowSink<PAIRS> sink{tile + lane * pitch, fs + lane, plan};
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

constexpr int PROJ_NV = 8;           // weight vectors contracted per launch
constexpr int PROJ_MAX_COLS = 104;   // columns per launch (whole channels); wider channel lists run as several launches
constexpr int PROJ_RING_MAX = 8;     // tile slots in flight (ring kernel)

// ------------------------------------------------------------------------------------------------
// sh_project with ONE weight vector: sh_project_seg_kernel.  One warp = one 32-point tile at a time, tiles dealt round-robin
// over all warps of a grid that fills the machine once; the next tile's point and weight are loaded before the current tile is
// evaluated.  The weight is folded into the radial values (w beta is what a lane produces), so the contraction is a plain column
// sum: the l-blocks are staged in SEGMENTS of at most 32 columns (whole channels, packed in the order of production; plan in
// ProjSegments) in the warp's shared-memory tile, TRANSPOSED: tile[column][point], pitch 34 doubles, so a lane's staging stores are
// conflict-free 8-byte stores and, when a segment is complete, lane c sums column c over the 32 points with 16-byte loads (rows
// 272 B apart: conflict-free) and adds the result to the warp's running sums in shared memory.  With one vector this beats the
// ring kernel below (0.158 vs 0.175 ms on the 128^3 grid, 100 columns): there is no weight traffic to save, and sixteen warps each
// own a whole tile.  Idle lanes of a ragged last tile evaluate the point (0, 0, 1) with weight 0.  Running sums are kept in the
// order of production ("slot order"); at the end a CTA adds its four warps in a fixed order and writes one row of `partial`
// [cta][ncols] in the caller's column order.
constexpr int PROJ_SEG_CTAS = 4;    // resident CTAs per SM (__launch_bounds__): register budget
constexpr int PROJ_SEG_PITCH = 34;  // doubles between consecutive columns of the transposed segment tile
constexpr int project_seg_doubles_per_warp() { return 32 * PROJ_SEG_PITCH + PROJ_MAX_COLS; }   // tile, running sums

struct ProjSegments {
    unsigned short scol[SH_MAX_PROJ];   // slot -> its first column in slot order
    unsigned short sbeg[SH_MAX_PROJ];   // slot -> first column (slot order) of the segment the slot belongs to
    unsigned char flush[SH_MAX_PROJ];   // slot -> 1 if the segment is complete after this slot
};

struct ProjectSegSink {
    double* tile;        // the warp's [32][PROJ_SEG_PITCH] transposed segment tile
    double* sums;        // the warp's running sums [PROJ_MAX_COLS]
    const double* fs;    // this lane's radial values times its weight: fs[slot*32]
    const ProjPlan& plan;
    const ProjSegments& seg;
    int lane;

    // column sums of a complete segment, added to the warp's running sums
    __device__ __forceinline__ void flush(int begin, int len) {
        __syncwarp();
        if (lane < len) {
            const double2* t = reinterpret_cast<const double2*>(tile + lane * PROJ_SEG_PITCH);
            double s0 = 0.0, s1 = 0.0, s2 = 0.0, s3 = 0.0;
#pragma unroll
            for (int r = 0; r < 16; r += 2) {
                const double2 a = t[r], b = t[r + 1];
                s0 += a.x; s1 += a.y; s2 += b.x; s3 += b.y;
            }
            sums[begin + lane] += (s0 + s1) + (s2 + s3);
        }
        __syncwarp();
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

template <int LMAX, bool FAST>
__global__ void __launch_bounds__(128, PROJ_SEG_CTAS) sh_project_seg_kernel(const double* __restrict__ xyz, int64_t n, const double* __restrict__ radial,
                                                                            const __grid_constant__ ProjPlan plan, const __grid_constant__ ProjSegments seg,
                                                                            const double* __restrict__ w, double* __restrict__ partial) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nslots = plan.first[shgen::LMAX_CAP + 1];
    const size_t wstride = project_seg_doubles_per_warp() + 32 * nslots;
    double* s_tile = reinterpret_cast<double*>(smem_raw) + (size_t)warp * wstride;
    double* s_sums = s_tile + 32 * PROJ_SEG_PITCH;
    double* s_fs = s_tile + project_seg_doubles_per_warp();   // radial values [slot][lane]
    const int ncols = plan.ncols;
    for (int e = lane; e < PROJ_MAX_COLS; e += 32) s_sums[e] = 0.0;
    const int64_t ntiles = (n + 31) >> 5;
    const int64_t gw = (int64_t)blockIdx.x * 4 + warp, nw = (int64_t)gridDim.x * 4;
    struct Item { double x, y, z, w; };
    auto load = [&](int64_t t, Item& it) {
        const int64_t i = (t << 5) + lane;
        if (i < n) {
            const double* p = xyz + 3 * i;
            it.x = __ldg(p); it.y = __ldg(p + 1); it.z = __ldg(p + 2);
            it.w = __ldg(w + i);
        } else {   // idle lane of the ragged last tile: a harmless point with weight 0
            it.x = 0.0; it.y = 0.0; it.z = 1.0; it.w = 0.0;
        }
    };
    Item cur, nxt;
    int64_t t = gw;
    if (t < ntiles) load(t, cur);
    for (; t < ntiles; t += nw) {
        if (t + nw < ntiles) load(t + nw, nxt);
        const RadialPos pos(cur.x, cur.y, cur.z, plan);
        // radial values of EVERY channel slot, times the lane's weight, computed up front (independent table loads overlap; loaded one
        // l-block at a time a warp pays one dependent L2 round trip per channel) and parked as fs[slot*32 + lane]
#pragma unroll 4
        for (int s = 0; s < nslots; ++s) s_fs[s * 32 + lane] = pos.f_row(radial + plan.row[s]) * cur.w;
        ProjectSegSink sink{s_tile, s_sums, s_fs + lane, plan, seg, lane};
        eval_projector_blocks<LMAX, FAST>(normalize(cur.x, cur.y, cur.z), plan, sink);
        cur = nxt;
    }
    // the CTA's four warps are added in a fixed order: one row of `partial` per CTA, in the caller's column order
    __syncthreads();
    const double* s0 = reinterpret_cast<const double*>(smem_raw) + 32 * PROJ_SEG_PITCH;
    for (int c = threadIdx.x; c < ncols; c += 128) {
        const double* q = s0 + c;
        int slot = 0;
        while (slot + 1 < nslots && seg.scol[slot + 1] <= c) ++slot;   // slot-order column -> the caller's column
        partial[(int64_t)blockIdx.x * ncols + plan.col[slot] + (c - seg.scol[slot])] = ((q[0] + q[wstride]) + q[2 * wstride]) + q[3 * wstride];
    }
}

// sh_project with 2 to 8 weight vectors per launch: sh_project_kernel.  coeff[v][col] = sum_i w[v][i] beta_col(r_i).  Nothing per point is written, so the FP64 pipe is the bound --
// provided the contraction does not spend the shared-memory bandwidth first (the previous design transposed every tile
// through shared memory and re-read the tile's weights as broadcasts per 32-column segment: ~710 shared-memory wavefronts
// per tile against 500 FP64-pipe cycles).  Here a lane IS a point on both sides of the hand-off, so nothing is transposed:
//
//   one persistent CTA per SM = NPW producer warps + NCW consumer warps around a ring of tile slots in shared memory
//   (slot = vals[ncols][32] + wts[NV][32] doubles; mbarrier full/empty pair per slot).
//   PRODUCERS: SPLIT warps per 32-point tile (lane i = point i; SPLIT = 1 in both shipped shapes: one warp evaluates the whole tile.
//     With SPLIT > 1 warp `part` evaluates the l-blocks of block_part and a2/a3 are repeated) stage beta_col = f_p(r) R_l^m at
//     vals[col][lane] (conflict-free 8-byte stores); the tile's weights go to wts[v][lane].  The radial values of a warp's own
//     channel slots are fetched up front (independent table loads overlap) and parked in the first column cell of each channel
//     until the block is produced.
//   CONSUMERS: every consumer warp visits every tile, but owns only some columns: a lane keeps acc[v][j] for its point
//     position and its columns IN REGISTERS across all tiles of the CTA (acc += wts[v][lane] * vals[col][lane]: one 8-byte
//     conflict-free load per NV FMAs, no broadcast, no transpose, every lane busy), and the cross-lane sum is taken once,
//     at the end, by a butterfly.  The accumulators are what bounds the shape: NV x ncols x 32 lanes doubles per CTA
//     (NV = 4, 104 columns: 26.6 K of the SM's 64 K registers), hence separate consumer warps that never evaluate a
//     polynomial, and lane GROUPS: G groups of 32/G lanes own different columns and take G points each per tile (group g
//     reads the point quarters in the rotated order (k + g) % G, so the G groups hit different banks), which divides the
//     accumulators per lane by G.
//   The consumers' FMAs are independent and fill the FP64-pipe bubbles of the producers' dependent polynomial chains.
// Tiles are dealt round-robin to the CTAs (static: the summation order is fixed, results are reproducible); idle lanes of a
// ragged last tile stage the point (0, 0, 1) with weight 0.  One row of `partial` [cta][nvec][ncols] per CTA, then
// sh_project_reduce_kernel adds the rows in a fixed order.

template <int NV> struct ProjCfg;
//                                   producer warps, warps per tile, consumer warps, lane groups per consumer warp
// One producer warp per tile (SPLIT = 1): nothing of a2/a3 or the radial look-up is repeated, and with 12 or 16 warps per CTA the
// compiler has 168 / 128 registers to overlap the polynomial chains of an l-block (a whole tile in ~7300 cycles, against 2 x 5700 for two
// warps sharing it at 96 registers).  The ring holds 8 tiles at 100 columns, so 8 producers; the consumer warps follow from the FMA load:
// four (G = 4: 32 accumulator registers) for up to four vectors, eight for eight.
// Five to eight vectors: the contraction of a tile, coeff[8][ncols] += wts[8][32 points] x vals[ncols][32 points]^T, is a dense 8 x ncols x 32
// product, and with DFMA consumers it was co-limited by shared-memory wavefronts (every lane re-reads its 8 weights per 4 values: ~1000
// wavefronts per tile against 1490 cycles).  MMA = true hands it to the FP64 tensor-core instruction (mma.sync m8n8k4: A = weights of 4
// points, B = values of 8 columns at those points): the same FP64 pipe time (on B200 DMMA runs at the DFMA rate and serialises with it), but
// one A and <= 4 B fragment loads per 4 points and warp instead of 12 loads per point quarter, 2 accumulator doubles per 8 columns, and
// 104 instead of 800 arithmetic issue slots per tile.  What it needs is conflict-free FRAGMENT loads: a fragment is 8 columns x 4
// consecutive points, and 64-bit shared loads are served per half-warp, so the four columns of a half-warp must tile 128 bytes: a column
// pitch of 36 doubles (288 B = 32 B mod 128).  With 32 the eight columns fall on the same 32 bytes of banks (no gain at all), 34 still leaves
// 2-way conflicts (ncu: 3.9 wavefronts per load).  The producers' stores (lane = point) are conflict-free for any pitch.  The wider slots
// leave 7 in the ring at 100 columns, hence 7 producer warps.
template <> struct ProjCfg<4> { static constexpr int NPW = 8, SPLIT = 1, NCW = 4, G = 4, PITCH = 32; static constexpr bool MMA = false; };
// Measured on the 128^3 grid, 100 columns, 8 vectors (DFMA consumers, 8 + 8 warps: 0.354 ms): pitch 32 / 33 (8 slots, conflicting fragment loads)
// 0.361 / 0.360; pitch 34, 7 + 4 warps 0.272; pitch 36, 7 + 4 warps 0.265; pitch 32 with the point index of a column XOR-swizzled by its position
// in its channel (conflict-free at 8 slots and 8 producers, a per-column table for the consumers) 0.267 -- no better, so the plain pitch stays.
template <> struct ProjCfg<8> { static constexpr int NPW = 7, SPLIT = 1, NCW = 4, G = 4, PITCH = 36; static constexpr bool MMA = true; };
static_assert(ProjCfg<4>::SPLIT == ProjCfg<8>::SPLIT, "run_project builds one per-part channel list for both");

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {   // release.cta
    asm volatile("{\n.reg .b64 t;\nmbarrier.arrive.shared::cta.b64 t, [%0];\n}" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {   // acquire.cta
    uint32_t done;
    do {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                     : "=r"(done)
                     : "r"(smem_u32(bar)), "r"(parity)
                     : "memory");
    } while (!done);
}

template <int PITCH>
struct ProjectStage {
    double* sv;   // the tile slot's vals + lane
    const ProjPlan& plan;
    template <int L> __device__ __forceinline__ void block(const double (&blk)[2 * L + 1]) {
#pragma unroll 1   // code size is instruction-fetch traffic (see ProjRowSink)
        for (int s = plan.first[L]; s < plan.first[L + 1]; ++s) {
            double* q = sv + plan.col[s] * PITCH;
            const double f = q[0];   // parked there by the radial pass
            static_for<0, 2 * L + 1>([&](auto mc) { q[decltype(mc)::value * PITCH] = f * blk[decltype(mc)::value]; });
        }
    }
};

// The tensor-core consumer (ProjCfg::MMA): warp cw of NCW owns the 8-column tiles nt = cw + j * NCW, j < R (R = its count, warp-uniform:
// the tile loop is compiled once per R and is branch-free inside).  Per 32-point tile and 4-point step ks: A fragment = wts[v = lane / 4]
// [4 ks + lane % 4], B fragments = vals[8 nt + lane / 4][4 ks + lane % 4], D += A B (m8n8k4, fp64): D[v][8 nt + 2 (lane % 4) + {0, 1}] in this
// lane.  The sums over the points are complete inside the instruction sequence, in a fixed order: no cross-lane reduction at the end.  A
// column tile that reaches past ncols reads weight rows (inside the slot: ncols + 7 < ncols + NV) and its extra columns are not written out.
template <int NV, int NCW, int PITCH, int R>
__device__ __forceinline__ void project_consume_mma(const double* ring, int slot_doubles, int nring, uint64_t* full, uint64_t* empty, int64_t my_tiles,
                                                    int ncols, int nvec, int cw, int lane, double* __restrict__ partial) {
    static_assert(NV == 8, "m8n8k4: eight weight vectors are the M dimension");
    const int grp = lane >> 2, tig = lane & 3;
    double acc[R > 0 ? R : 1][2];
    static_for<0, R>([&](auto jc) { acc[decltype(jc)::value][0] = 0.0; acc[decltype(jc)::value][1] = 0.0; });
    int slot = 0, use = 0;
    for (int64_t seq = 0; seq < my_tiles; ++seq) {
        mbar_wait(full + slot, use & 1);
        if constexpr (R > 0) {
            const double* sv = ring + (size_t)slot * slot_doubles;
            const double* arow = sv + (ncols + grp) * PITCH + tig;
            const double* brow = sv + (8 * cw + grp) * PITCH + tig;
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) {
                const double a = arow[4 * ks];
                double b[R];
                static_for<0, R>([&](auto jc) { b[decltype(jc)::value] = brow[decltype(jc)::value * 8 * NCW * PITCH + 4 * ks]; });
                static_for<0, R>([&](auto jc) {
                    constexpr int J = decltype(jc)::value;
                    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                                 : "+d"(acc[J][0]), "+d"(acc[J][1])
                                 : "d"(a), "d"(b[J]));
                });
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty + slot);
        if (++slot == nring) { slot = 0; ++use; }
    }
    static_for<0, R>([&](auto jc) {
        constexpr int J = decltype(jc)::value;
        const int c = 8 * (cw + J * NCW) + 2 * tig;
        if (grp < nvec) {
            double* row = partial + ((int64_t)blockIdx.x * nvec + grp) * ncols;
            if (c < ncols) row[c] = acc[J][0];
            if (c + 1 < ncols) row[c + 1] = acc[J][1];
        }
    });
}

// The consumer side of sh_project_kernel for a warp whose lanes own R columns each (column owner + j * OWNERS, j < R).
template <int NV, int G, int OWNERS, int R>
__device__ __forceinline__ void project_consume(const double* ring, int slot_doubles, int nring, uint64_t* full, uint64_t* empty, int64_t my_tiles,
                                                int ncols, int nvec, int cw, int lane, double* __restrict__ partial) {
    constexpr int PTS = 32 / G;
    const int g = lane / PTS, pl = lane % PTS;
    const int owner = cw * G + g;
    double acc[NV][R > 0 ? R : 1];
    static_for<0, NV>([&](auto vc) { static_for<0, R>([&](auto jc) { acc[decltype(vc)::value][decltype(jc)::value] = 0.0; }); });
    int slot = 0, use = 0;
    for (int64_t seq = 0; seq < my_tiles; ++seq) {
        mbar_wait(full + slot, use & 1);
        if constexpr (R > 0) {
            const double* sv = ring + (size_t)slot * slot_doubles;
#pragma unroll
            for (int k = 0; k < G; ++k) {
                const int pt = pl + PTS * ((k + g) % G);   // rotated: the G groups read different banks
                const double* wrow = sv + ncols * 32 + pt;
                const double* col = sv + owner * 32 + pt;   // a lane whose owner has one column fewer reads a weights row in its last round: never written out
                double wt[NV], val[R];
                static_for<0, NV>([&](auto vc) { wt[decltype(vc)::value] = wrow[decltype(vc)::value * 32]; });
                static_for<0, R>([&](auto jc) { val[decltype(jc)::value] = col[decltype(jc)::value * OWNERS * 32]; });
                static_for<0, R>([&](auto jc) {
                    static_for<0, NV>([&](auto vc) {
                        acc[decltype(vc)::value][decltype(jc)::value] = fma(wt[decltype(vc)::value], val[decltype(jc)::value], acc[decltype(vc)::value][decltype(jc)::value]);
                    });
                });
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty + slot);
        if (++slot == nring) { slot = 0; ++use; }
    }
    // sum over the group's lanes (butterfly: every lane ends with the same value), one row of `partial` per CTA
    static_for<0, NV>([&](auto vc) {
        constexpr int V = decltype(vc)::value;
        static_for<0, R>([&](auto jc) {
            constexpr int J = decltype(jc)::value;
            double s = acc[V][J];
#pragma unroll
            for (int off = PTS / 2; off >= 1; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
            const int c = owner + J * OWNERS;
            if (pl == 0 && c < ncols && V < nvec) partial[((int64_t)blockIdx.x * nvec + V) * ncols + c] = s;
        });
    });
}

template <int LMAX, int NV, bool FAST>
__global__ void __launch_bounds__(32 * (ProjCfg<NV>::NPW + ProjCfg<NV>::NCW), 1)
    sh_project_kernel(const double* __restrict__ xyz, int64_t n, const double* __restrict__ radial, const __grid_constant__ ProjPlan plan,
                      const double* __restrict__ w, int nvec, double* __restrict__ partial, int nring) {
    using Cfg = ProjCfg<NV>;
    constexpr int NPW = Cfg::NPW, SPLIT = Cfg::SPLIT, NCW = Cfg::NCW, G = Cfg::G, PITCH = Cfg::PITCH;
    static_assert(NPW % SPLIT == 0 && 32 % G == 0 && NV >= G - 1 && PITCH >= 32, "shape");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int ncols = plan.ncols;
    const int slot_doubles = (ncols + NV) * PITCH;
    double* ring = reinterpret_cast<double*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(ring + (size_t)nring * slot_doubles);
    uint64_t* empty = full + PROJ_RING_MAX;
    if (threadIdx.x == 0) {
        for (int s = 0; s < nring; ++s) {
            mbar_init(full + s, SPLIT);   // one arrival per producer warp of the tile
            mbar_init(empty + s, NCW);    // one per consumer warp
        }
    }
    __syncthreads();
    const int64_t ntiles = (n + 31) >> 5;
    const int64_t my_tiles = (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x;   // tiles blockIdx.x + seq * gridDim.x

    if (warp < NPW) {
        // ---------------- producer ----------------
        // Tile streams: at most as many as the ring has slots.  With more streams than slots a producer could be TWO uses ahead of a slot,
        // and a parity wait cannot tell "the use before last is still being read" from "the last use has been released" (DESIGN.md
        // section 6: it hangs, after racing); with streams <= slots the stream's own previous tile guarantees the older release.
        constexpr int MAX_STREAMS = NPW / SPLIT;
        const int STREAMS = MAX_STREAMS < nring ? MAX_STREAMS : nring;
        const int stream = warp / SPLIT, part = warp % SPLIT;
        if (stream >= STREAMS) return;   // a producer warp without a stream (only when the ring is shorter than the warp list)
        const int ps0 = plan.part_first[part], ps1 = plan.part_first[part + 1];   // this warp's channel slots
        // point index of this lane in the stream's current tile; the stream advances by STREAMS * gridDim.x tiles
        int64_t i = (((int64_t)blockIdx.x + (int64_t)stream * gridDim.x) << 5) + lane;
        const int64_t istep = ((int64_t)STREAMS * gridDim.x) << 5;
        // The next tile's point is loaded a whole tile ahead and NOT touched until then: a select on the loaded value right behind the
        // load would make the warp wait for it at once (it did: 14 % of the producers' time).  Idle lanes of a ragged last tile read the
        // last point and are replaced by a harmless one (weights 0) where the values are used.  Streaming loads (evict-first): what
        // should stay in the small L1 next to 213 KB of ring is the radial table.
        auto load_point = [&](int64_t ip, double& x, double& y, double& z) {
            const double* p = xyz + 3 * (ip < n ? ip : n - 1);
            x = __ldcs(p); y = __ldcs(p + 1); z = __ldcs(p + 2);
        };
        double x = 0.0, y = 0.0, z = 1.0, nx = 0.0, ny = 0.0, nz = 1.0;
        int64_t seq = stream;
        if (seq < my_tiles) load_point(i, x, y, z);
        int slot = stream % nring, use = stream / nring;
        for (; seq < my_tiles; seq += STREAMS, i += istep) {
            if (seq + STREAMS < my_tiles) load_point(i + istep, nx, ny, nz);
            // the tile's weights: vector v is fetched by warp part v % SPLIT; masked where they are stored
            constexpr int WPP = (NV + SPLIT - 1) / SPLIT;
            double wv[WPP];
            const bool ok = i < n;
            const int64_t iw = ok ? i : n - 1;
            static_for<0, WPP>([&](auto kc) {
                const int v = part + decltype(kc)::value * SPLIT;
                wv[decltype(kc)::value] = __ldcs(w + (int64_t)(v < nvec ? v : 0) * n + iw);
            });
            if (!ok) { x = 0.0; y = 0.0; z = 1.0; }
            if (use > 0) mbar_wait(empty + slot, (use - 1) & 1);   // the consumers have released the slot's previous tile
            double* sv = ring + (size_t)slot * slot_doubles + lane;
            const RadialPos pos(x, y, z, plan);
#pragma unroll 8   // eight channels' table loads in flight (4: 0.230 ms, 8: 0.228, 16: 0.279 for four vectors on the 128^3 grid)
            for (int k = ps0; k < ps1; ++k) {
                const int s = plan.part_slots[k];
                sv[plan.col[s] * PITCH] = pos.f_row(radial + plan.row[s]);
            }
            const UnitVec u = normalize(x, y, z);
            ProjectStage<PITCH> sink{sv, plan};
            static_for<0, SPLIT>([&](auto pc) {
                constexpr int PART = decltype(pc)::value;
                if (part == PART) eval_projector_blocks<LMAX, FAST, SPLIT, PART>(u, plan, sink);
            });
            static_for<0, WPP>([&](auto kc) {
                const int v = part + decltype(kc)::value * SPLIT;
                if (v < NV) sv[(ncols + v) * PITCH] = (ok && v < nvec) ? wv[decltype(kc)::value] : 0.0;
            });
            __syncwarp();
            if (lane == 0) mbar_arrive(full + slot);
            x = nx; y = ny; z = nz;
            slot += STREAMS;
            while (slot >= nring) { slot -= nring; ++use; }
        }
    } else {
        // ---------------- consumer ----------------
        const int cw = warp - NPW;
        if constexpr (Cfg::MMA) {
            constexpr int RMAX = ((PROJ_MAX_COLS + 7) / 8 + NCW - 1) / NCW;   // 8-column tiles per warp
            const int ntiles8 = (ncols + 7) >> 3;
            const int mine = ntiles8 > cw ? (ntiles8 - cw + NCW - 1) / NCW : 0;   // warp-uniform
            static_for<0, RMAX + 1>([&](auto rc) {
                constexpr int R = decltype(rc)::value;
                if (mine == R) project_consume_mma<NV, NCW, PITCH, R>(ring, slot_doubles, nring, full, empty, my_tiles, ncols, nvec, cw, lane, partial);
            });
        } else {
            static_assert(PITCH == 32, "project_consume reads rows of 32 doubles");
            constexpr int OWNERS = NCW * G, CPW = (PROJ_MAX_COLS + OWNERS - 1) / OWNERS;
            // column rounds of the warp's first owner (warp-uniform): the tile loop is compiled once per count, branch-free inside
            const int rounds = (ncols - cw * G + OWNERS - 1) / OWNERS;
            static_for<0, CPW + 1>([&](auto rc) {
                constexpr int R = decltype(rc)::value;
                if ((rounds < 0 ? 0 : rounds) == R)
                    project_consume<NV, G, OWNERS, R>(ring, slot_doubles, nring, full, empty, my_tiles, ncols, nvec, cw, lane, partial);
            });
        }
    }
}

// coeff[v*coeff_stride + col] = sum over CTAs of partial[cta][v][col], the rows added in a fixed order (reproducible):
// 32 lanes = 32 consecutive (v, column) elements; the block's 32 warps each add every 32nd row of `partial` (coalesced, four
// loads in flight), then the 32 sums are added in order.
__global__ void __launch_bounds__(1024) sh_project_reduce_kernel(const double* __restrict__ partial, int nrows, int nvec, int ncols,
                                                                  double* __restrict__ coeff, int coeff_stride) {
    __shared__ double s[32][33];
    const int ne = nvec * ncols;
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
        const int v = e / ncols, c = e - v * ncols;
        coeff[v * coeff_stride + c] = t;
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
                plan.row[slot] = p * nr;
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


// warps per tile (block_part): the default comes from the 128^3-grid measurements in DESIGN.md section 6
constexpr int PROJ_AOS_SPLIT = 2;

template <int LMAX, int SPLIT>
int launch_proj_aos_split(const double* xyz, int64_t n, const double* radial, const ProjPlan& plan, double* out, int pitch, int mode, size_t smem,
                          cudaStream_t st) {
    const int64_t ntiles = (n + 31) / 32;
    if (ntiles > 0x7fffffffLL) return SH_ERR_COUNT;
    auto launch = [&](auto kern, SmemOptIn& opted_in) -> int {
        if (const int rc = ensure_dynamic_smem(kern, smem, opted_in); rc != SH_OK) return rc;
        kern<<<(unsigned)ntiles, 32 * SPLIT, smem, st>>>(xyz, n, radial, plan, out, pitch, mode, prefetch_plan(n, 32));
        return launch_status();
    };
    static SmemOptIn opted_in[2];   // the opt-in limit only ever grows
    // 16-byte staging stores where every row keeps 16-byte alignment (even pitch; the staging tile itself is 16-byte aligned)
    if (pitch % 2 == 0 && tuned(SH_TUNE_PROJ_AOS_PAIRS, 0) != 1) return launch(sh_proj_aos_kernel<LMAX, SPLIT, true>, opted_in[1]);
    return launch(sh_proj_aos_kernel<LMAX, SPLIT, false>, opted_in[0]);
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

// channel slots of each warp part of sh_project_kernel's producers (block_part<SPLIT>)
template <int SPLIT>
void fill_parts(const int* proj_l, ProjPlan& plan) {
    const int nslots = plan.first[shgen::LMAX_CAP + 1];
    int k = 0;
    for (int part = 0; part < SPLIT; ++part) {
        plan.part_first[part] = (unsigned char)k;
        for (int s = 0; s < nslots; ++s)
            if (block_part<SPLIT>(proj_l[plan.chan[s]]) == part) plan.part_slots[k++] = (unsigned char)s;
    }
    for (int part = SPLIT; part < 5; ++part) plan.part_first[part] = (unsigned char)k;
}

int64_t project_workspace_bytes(int ncols, int nvec) {
    if (ncols < 0 || nvec < 0) return -1;
    const int64_t cols = ncols < PROJ_MAX_COLS ? ncols : PROJ_MAX_COLS, vecs = nvec < PROJ_NV ? nvec : PROJ_NV;
    return (int64_t)sm_count() * PROJ_SEG_CTAS * vecs * cols * (int64_t)sizeof(double);   // one row per CTA of the largest grid
}

// one weight vector: the transposed-segment kernel; rows of `partial` = its CTAs
template <int LMAX>
int launch_project_seg(const double* xyz, int64_t n, const double* radial, const int* proj_l, const ProjPlan& plan, const double* w, double* partial,
                       int64_t* rows, cudaStream_t st) {
    ProjSegments seg;
    make_segments(proj_l, plan, seg);
    const bool fast = tuned(SH_TUNE_PROJECT_FORM, 1) != 2;   // Horner / recurrence forms (default) or the factorized ones (knob value 2)
    const int nslots = plan.first[shgen::LMAX_CAP + 1];
    const size_t smem = (size_t)4 * (project_seg_doubles_per_warp() + 32 * nslots) * sizeof(double);   // 38 KB + 1 KB per slot
    constexpr size_t smem_max = (size_t)4 * (project_seg_doubles_per_warp() + 32 * SH_MAX_PROJ) * sizeof(double);
    auto launch = [&](auto kern, SmemOptIn& opted_in) -> int {
        if (const int rc = ensure_dynamic_smem(kern, smem_max, opted_in); rc != SH_OK) return rc;
        // the grid fills the machine once: resident CTAs per SM for THIS shared-memory size (228 KB per SM, 1 KB reserved per CTA;
        // registers allow PROJ_SEG_CTAS): many channel slots leave fewer, and tiles are dealt statically, so a CTA that is not
        // resident from the start would run as a second wave
        int occ = (int)((size_t)228 * 1024 / (smem + 1024));
        if (occ < 1) occ = 1;
        if (occ > PROJ_SEG_CTAS) occ = PROJ_SEG_CTAS;
        const int64_t ntiles = (n + 31) / 32, cap = (int64_t)sm_count() * occ;
        int64_t blocks = (ntiles + 3) / 4;
        if (blocks > cap) blocks = cap;
        *rows = blocks;
        kern<<<(unsigned)blocks, 128, smem, st>>>(xyz, n, radial, plan, seg, w, partial);
        return launch_status();
    };
    static SmemOptIn opted_in[2];
    return fast ? launch(sh_project_seg_kernel<LMAX, true>, opted_in[1]) : launch(sh_project_seg_kernel<LMAX, false>, opted_in[0]);
}

// 2 to 8 weight vectors: the ring kernel, one persistent CTA per SM; rows of `partial` = its CTAs
template <int LMAX, int NV>
int launch_project_ring(const double* xyz, int64_t n, const double* radial, const ProjPlan& plan, const double* w, int nvec, double* partial,
                        int64_t* rows, cudaStream_t st) {
    using Cfg = ProjCfg<NV>;
    // ring of tile slots: as many as fit (at most PROJ_RING_MAX), then the 2 x PROJ_RING_MAX mbarriers
    const size_t slot_bytes = (size_t)(plan.ncols + NV) * Cfg::PITCH * sizeof(double);
    int nring = (int)(((size_t)227 * 1024 - 2 * PROJ_RING_MAX * sizeof(uint64_t)) / slot_bytes);
    if (nring > PROJ_RING_MAX) nring = PROJ_RING_MAX;
    if (nring < 1) return SH_ERR_PROJECTOR;
    const size_t smem = (size_t)nring * slot_bytes + 2 * PROJ_RING_MAX * sizeof(uint64_t);
    const bool fast = tuned(SH_TUNE_PROJECT_FORM, 1) != 2;
    const int64_t ntiles = (n + 31) / 32;
    const int64_t blocks = ntiles < sm_count() ? ntiles : sm_count();
    *rows = blocks;
    auto launch = [&](auto kern, SmemOptIn& opted_in) -> int {
        if (const int rc = ensure_dynamic_smem(kern, (size_t)227 * 1024, opted_in); rc != SH_OK) return rc;
        kern<<<(unsigned)blocks, 32 * (Cfg::NPW + Cfg::NCW), smem, st>>>(xyz, n, radial, plan, w, nvec, partial, nring);
        return launch_status();
    };
    static SmemOptIn opted_in[2];
    return fast ? launch(sh_project_kernel<LMAX, NV, true>, opted_in[1]) : launch(sh_project_kernel<LMAX, NV, false>, opted_in[0]);
}

template <int LMAX>
int launch_project(const double* xyz, int64_t n, const double* radial, const int* proj_l, const ProjPlan& plan, const double* w, int nvec,
                   double* partial, double* coeff, int coeff_stride, cudaStream_t st) {
    int64_t rows = 0;
    int rc;
    if (nvec == 1) rc = launch_project_seg<LMAX>(xyz, n, radial, proj_l, plan, w, partial, &rows, st);
    else if (nvec <= 4) rc = launch_project_ring<LMAX, 4>(xyz, n, radial, plan, w, nvec, partial, &rows, st);
    else rc = launch_project_ring<LMAX, 8>(xyz, n, radial, plan, w, nvec, partial, &rows, st);
    if (rc != SH_OK) return rc;
    const int elems = nvec * plan.ncols;
    sh_project_reduce_kernel<<<(elems + 31) / 32, 1024, 0, st>>>(partial, (int)rows, nvec, plan.ncols, coeff, coeff_stride);
    return launch_status();
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
        const int lmax = make_plan(proj_l, p0, p1, nr, dr, plan);
        fill_parts<ProjCfg<4>::SPLIT>(proj_l, plan);
        for (int v0 = 0; v0 < nvec; v0 += PROJ_NV) {
            const int nv = nvec - v0 < PROJ_NV ? nvec - v0 : PROJ_NV;
            switch (lmax) {
#define SH_CASE(L) case L: rc = launch_project<L>(xyz, n, radial, proj_l, plan, w + (int64_t)v0 * n, nv, partial, coeff + (int64_t)v0 * ncols + c0, ncols, st); break;
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

// ------------------------------------------------------------------------------------------------
// sh_project_static: sh_project for callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc).  The per-CTA partial sums that sh_project keeps in the caller's `workspace` live in this file-scope device array
// instead: PROJ_STATIC_BYTES = 2 MiB, held by every GPU that loads the library until the process exits.  A request whose
// sh_project_workspace_bytes(ncols, nvec) exceeds it is refused with SH_ERR_SCRATCH (on a 148-SM B200: min(nvec, 8) x min(ncols, 104)
// <= 442, i.e. any width with up to 4 weight vectors, up to 55 columns with 5 to 8; more vectors or columns per call run as several
// passes over the same array, so only these two capped factors count).
// In HOST code the array's name is a host-side stand-in, not a device address (a kernel handed `g_project_scratch` itself would fault,
// or, where the GPU can reach host memory, silently use the wrong memory): the device address comes from cudaGetSymbolAddress, asked
// once per device with that device current, and is what the kernels get.
// Nothing has to start at zero: every row of partial sums the ordered reduction reads was written by a kernel of the SAME call before
// it (each CTA stores, not accumulates, its full row), so the contents a previous call left behind are never read.  All calls on a
// device share the one array: calls that overlap on the GPU (different streams, or graphs replayed concurrently) race.
constexpr size_t PROJ_STATIC_BYTES = (size_t)2 << 20;
static __device__ __align__(256) double g_project_scratch[PROJ_STATIC_BYTES / sizeof(double)];

// device address of g_project_scratch on the CURRENT device (cached per device; racing threads resolve the same value)
int project_scratch_address(double** out) {
    static std::atomic<double*> cache[64];   // static storage: null-initialised
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e);
    double* ptr = dev < 64 ? cache[dev].load(std::memory_order_acquire) : nullptr;
    if (!ptr) {
        e = cudaGetSymbolAddress(reinterpret_cast<void**>(&ptr), g_project_scratch);
        if (e != cudaSuccess) return cuda_fail(e);
        if (!ptr) return SH_ERR_CUDA;
        if (dev < 64) cache[dev].store(ptr, std::memory_order_release);
    }
    *out = ptr;
    return SH_OK;
}

int run_project_static(const double* xyz, int64_t n, int nproj, const int* proj_l, const double* radial, int nr, double dr, const double* w,
                       int nvec, double* coeff, void* stream) {
    // the argument checks of sh_project that need no workspace come first, so that a bad call is reported as what it is
    const int rc = check_projector_args(xyz, n, nproj, proj_l, radial, nr, dr);
    if (rc != SH_OK) return rc;
    if (nvec < 0) return SH_ERR_PROJECTOR;
    const int ncols = projector_count(nproj, proj_l);
    if (nvec == 0 || ncols == 0) return SH_OK;
    const int64_t need = project_workspace_bytes(ncols, nvec);
    if (need < 0 || need > (int64_t)PROJ_STATIC_BYTES) return SH_ERR_SCRATCH;
    double* scratch = nullptr;
    if (n > 0) {   // the empty sum launches nothing that reads the scratch
        const int rs = project_scratch_address(&scratch);
        if (rs != SH_OK) return rs;
    }
    // the same code path as sh_project from here on, with the static array as its workspace: no cudaMalloc, cudaFree or allocating
    // library routine anywhere below (plans live on the host stack, kernels take them by value)
    return run_project(xyz, n, nproj, proj_l, radial, nr, dr, w, nvec, coeff, scratch, n > 0 ? (int64_t)PROJ_STATIC_BYTES : 0, stream);
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
int sh_project_static(const double* xyz, int64_t n, int nproj, const int* proj_l, const double* radial, int nr, double dr, const double* w,
                      int nvec, double* coeff, void* stream) {
    return run_project_static(xyz, n, nproj, proj_l, radial, nr, dr, w, nvec, coeff, stream);
}
int64_t sh_project_static_bytes(void) { return (int64_t)PROJ_STATIC_BYTES; }

}  // extern "C"
