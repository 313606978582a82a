/*
 * shb200.h -- C ABI of libshb200: batched real, complex and spin-1/2 spinor spherical harmonics for
 * all l <= lmax <= 9 at Cartesian points, on one NVIDIA B200 (sm_100a).
 *
 * The operation is the one stated in arxiv 2510.05282 ("SHarmonic"); citations are to
 * /root/reference/PAPER.md lines (P:n) and to this repository's DESIGN.md:
 *   - Y_l^m, Condon-Shortley phase included:        Eq. 5
 *   - real harmonics R_l^m:                          Eq. 6
 *   - spinor harmonics, spin 1/2, j = l +- 1/2:      Eq. 7
 *   - Cartesian front end, the value does not depend on |r|;
 *     at r = 0 every harmonic is 0 except l = 0:
 *   - evaluated as explicit factorized polynomials in x/r, y/r, z/r: Eq. 8, Eq. 16, App. B/C
 *
 * Conventions (the paper's API is per point and per (l, m) and fixes no batch layout):
 *   K = (lmax+1)^2.  Point i, harmonic index k = l(l+1)+m, m = -l..l.
 *   real     element = 1 double           count per point = K
 *   complex  element = (re, im)           count per point = K      (2K doubles)
 *   spinor   element = (up.re, up.im, down.re, down.im)            count per point = 2K (8K doubles)
 *            s = 2 l^2 + (j = l-1/2 ? m_j + j : 2l + m_j + j): l ascending; the j = l-1/2 block (2l entries,
 *            absent for l = 0) then the j = l+1/2 block (2l+2 entries); m_j ascending.
 *   SH_LAYOUT_AOS: out[i * count + e]   ([N][count] elements)
 *   SH_LAYOUT_SOA: out[e * n + i]       ([count][N] elements; an element stays contiguous)
 *
 * Pointers: every `xyz` / `out` of the sh_real / sh_complex / sh_spinor / sh_real_f32 calls is a DEVICE
 * pointer (global memory of the current CUDA device); `xyz` is AoS [n][3].  The *_host calls take HOST
 * pointers.  The caller owns all buffers; the device calls allocate nothing and may be issued concurrently from several
 * threads and on several devices.  What the library does keep, process-wide: the sh_set_tuning() knobs (benchmarking only;
 * they select among kernels with identical results, so a concurrent caller can see another kernel but never another value),
 * per-device caches of pure device properties (SM count, granted shared-memory opt-ins), a launch counter, the last CUDA
 * error text (per thread), and the staging pool of the *_host calls (created on first use, serialised by a mutex, freed by
 * sh_host_release()).  Device calls are asynchronous: they enqueue kernels on
 * `stream` (a cudaStream_t passed as void*; NULL = the legacy default stream) and return without
 * synchronizing.  `out` must be aligned to its element type (8 B for sh_real, 4 B for sh_real_f32); 16-byte
 * aligned `out` (and, for SoA, even n) enables the vectorised / bulk-copy store paths, anything else falls
 * back to a scalar store path with identical results.  `xyz` and `out` must not overlap.
 *
 * Domain: any finite coordinates, including subnormal and huge ones (inputs are pre-scaled by a power
 * of two before r^2 is formed); r = 0 exactly (no epsilon) selects the P:60 convention.  NaN or Inf
 * coordinates give NaN in every l >= 1 output of that point (not an error; the l = 0 harmonic is a constant).
 *
 * Errors: every call returns SH_OK (0) or a negative SH_ERR_* code; nothing is thrown and nothing is
 * written on error.  n == 0 is a successful no-op (pointers may then be NULL).
 */
#ifndef SHB200_H
#define SHB200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    SH_LAYOUT_AOS = 0, /* out[i*count + e] */
    SH_LAYOUT_SOA = 1  /* out[e*n + i]     */
};

/* Optional store-path request, OR-ed into `layout` (bits 8-15).  SH_STORE_AUTO picks the fastest path the
 * alignment allows.  A request the alignment does not allow returns SH_ERR_ALIGNMENT.  Results are identical
 * on every path (same arithmetic, different store mechanism). */
enum {
    SH_STORE_AUTO   = 0 << 8, /* SoA with a 16-byte aligned out: sh_real (even n >= 128), sh_real_f32 (n a multiple of 4, >= 256) and sh_complex
                                 (n >= 64) stage tiles of 128 / 256 / 64 points in shared memory and write each with one TMA tensor store
                                 (cp.async.bulk.tensor.2d through a tensor map of out as [K][n]: rows of 1 KB);
                                 AoS with a 16-byte aligned out: SH_STORE_BULK; everything else: SH_STORE_DIRECT */
    SH_STORE_DIRECT = 1 << 8, /* per-thread st.global.cs; SoA: coalesced planes; AoS: smem transpose + coalesced stores */
    SH_STORE_BULK   = 2 << 8  /* AoS only, needs a 16-byte aligned out: rows staged in shared memory, written by TMA bulk copies
                                 (cp.async.bulk): one copy per 32-point tile where the layout allows, else one per row */
};

/* Input front end, OR-ed into `layout` (bits 16-17).  Default: Cartesian.
 *   SH_COORDS_CARTESIAN   xyz is [n][3] points of any norm; the library divides by r.
 *   SH_COORDS_NORMALIZED  xyz is [n][3] UNIT vectors (Eq. 8, the paper's fastest interface): the normalization step is
 *                         skipped; values are unspecified polynomials if the input is not normalized; a zero
 *                         vector selects the r = 0 convention.
 *   SH_COORDS_ANGULAR     xyz is [n][2] = (theta, phi), polar angle first (Eq. 3-4); x = sin(theta)cos(phi),
 *                         y = sin(theta)sin(phi), z = cos(theta). */
enum {
    SH_COORDS_CARTESIAN  = 0 << 16,
    SH_COORDS_NORMALIZED = 1 << 16,
    SH_COORDS_ANGULAR    = 2 << 16
};

enum {
    SH_OK = 0,
    SH_ERR_NULL = -1,      /* xyz or out is NULL with n > 0 */
    SH_ERR_COUNT = -2,     /* n < 0 */
    SH_ERR_LMAX = -3,      /* lmax outside [0, 9] */
    SH_ERR_LAYOUT = -4,    /* unknown layout, store-path or front-end bits */
    SH_ERR_ALIGNMENT = -5, /* out not aligned to its element type, or requested store path not possible */
    SH_ERR_CUDA = -6,      /* CUDA launch / copy error; text via sh_last_cuda_error() */
    SH_ERR_PROJECTOR = -7, /* sh_projectors / sh_project: nproj, proj_l, nr, dr, nvec or the workspace size is invalid */
    SH_ERR_SCRATCH = -8    /* sh_project_static: the request needs more scratch than the library's static device array holds */
};

/* Real harmonics R_l^m (Eq. 6), fp64.  out: K doubles per point. */
int sh_real(const double* xyz, int64_t n, int lmax, double* out, int layout, void* stream);
/* Complex harmonics Y_l^m (Eq. 5), fp64.  out: K (re, im) pairs per point. */
int sh_complex(const double* xyz, int64_t n, int lmax, double* out, int layout, void* stream);
/* Spinor harmonics (Eq. 7), fp64.  out: 2K elements of 4 doubles per point. */
int sh_spinor(const double* xyz, int64_t n, int lmax, double* out, int layout, void* stream);
/* fp32 variant of sh_real: fp32 in, fp32 out; the normalization runs in fp64, the polynomials in fp32. */
int sh_real_f32(const float* xyz, int64_t n, int lmax, float* out, int layout, void* stream);

/* The paper's own measurement protocol (Table I: "the results are accumulated and never stored"):
 * out[i] = sum over all l <= lmax, m of R_l^m(xyz_i), one double per point, every harmonic evaluated exactly as in sh_real.
 * With 32 bytes of traffic per point instead of 824 this call is bound by the FP64 pipe: it measures the arithmetic side of
 * the roofline of the factorized formulas, and its rate is the one comparable with the paper's CPU / V100 figures.
 * `coords` is one of SH_COORDS_* (no layout bits: there is one value per point); DEVICE pointers; asynchronous on `stream`. */
int sh_real_sum(const double* xyz, int64_t n, int lmax, double* out, int coords, void* stream);

/* Extension beyond the paper's explicit range (its conclusion: "could be easily extended using recurrence
 * relationships for higher values of l"): real / complex harmonics for all l <= lmax <= 32 (sh_lmax_ext()).
 * lmax <= 9 behaves exactly like sh_real / sh_complex.  For 10 <= lmax <= 32 the explicit l <= 9 formulas seed the
 * upward recurrence in l at fixed m of the normalized associated Legendre factors (Eq. 5 with the standard three-term
 * recurrence), and (x + i y)^m continues by complex multiplication; same index convention k = l(l+1)+m, same r = 0
 * convention.  SH_LAYOUT_SOA only for lmax > 9 (SH_ERR_LAYOUT otherwise); all three front ends; DEVICE pointers. */
int sh_real_ext(const double* xyz, int64_t n, int lmax, double* out, int layout, void* stream);
int sh_complex_ext(const double* xyz, int64_t n, int lmax, double* out, int layout, void* stream);
/* Largest lmax the *_ext calls accept (32). */
int sh_lmax_ext(void);

/* Fused projector consumer (the use case the paper names: "the atomic problem is solved in a radial
 * grid ... This produces a series of angular-momentum dependent projectors.  To represent these projectors in a
 * 3-dimensional grid we need to calculate the spherical harmonics for each point").
 * The harmonics are consumed where they are produced instead of being written out in full:
 *   channel p = 0..nproj-1 has angular momentum proj_l[p] in [0, 9] and a radial function tabulated on the uniform
 *   radial grid r_j = j dr:  radial[p*nr + j] = f_p(r_j), j = 0..nr-1 (nr >= 2, dr > 0).  The paper fixes no
 *   interpolation; this library's reading is piecewise linear,
 *     f_p(r) = radial[p][j] + (r/dr - j)(radial[p][j+1] - radial[p][j]),  j = floor(r/dr),   for r <  (nr-1) dr
 *     f_p(r) = 0                                                                             for r >= (nr-1) dr
 *   (a table should end with 0, as projectors vanish at their cutoff radius, to be continuous there).
 *   beta_{p,m}(r_vec) = f_p(|r_vec|) R_{l_p}^m(r_vec/|r_vec|), m = -l_p..l_p  (Eq. 6; at r = 0 only l = 0 survives)
 *   column of (p, m) = sum_{p' < p} (2 proj_l[p'] + 1) + (m + proj_l[p]);  ncols = sh_projector_count(nproj, proj_l).
 *   NaN or Inf coordinates: every l >= 1 column of that point is NaN, the l = 0 columns are 0 (|r| is not inside the table).
 * `proj_l` is a HOST array (read during the call); xyz [n][3] Cartesian points relative to the atom, `radial`, `out`,
 * `w`, `coeff`, `workspace` are DEVICE pointers.  nproj <= SH_MAX_PROJ.  Asynchronous on `stream`; nothing is allocated.
 *
 * sh_projectors: out[i*ncols + col] (SH_LAYOUT_AOS) or out[col*n + i] (SH_LAYOUT_SOA) = beta_col(xyz_i); only the
 *   requested channels are evaluated and written (8 ncols bytes per point instead of 800).
 * sh_project: coeff[v*ncols + col] = sum_i w[v*n + i] beta_col(xyz_i), v < nvec: the projection <beta|psi> with
 *   w = psi dV; NOTHING per point is written.  The sum is taken in a fixed order (per-CTA partial sums in `workspace`,
 *   then one ordered pass), so results are reproducible run to run on one device; they differ from the sum in point
 *   order by rounding only (<= 1e-12 sum_i |w_i beta_i| is the tested bound).  `workspace` must hold at least
 *   sh_project_workspace_bytes(ncols, nvec) bytes, 8-byte aligned; its contents are scratch.  One pass over the points
 *   serves up to 8 weight vectors and 104 columns (whole channels); more vectors or columns run as several passes. */
enum { SH_MAX_PROJ = 32 };
int sh_projector_count(int nproj, const int* proj_l);            /* ncols, or -1 if a proj_l is outside [0, 9] or nproj outside [0, 32] */
int64_t sh_project_workspace_bytes(int ncols, int nvec);        /* -1 on bad arguments */
int sh_projectors(const double* xyz, int64_t n, int nproj, const int* proj_l, const double* radial, int nr, double dr,
                  double* out, int layout, void* stream);
int sh_project(const double* xyz, int64_t n, int nproj, const int* proj_l, const double* radial, int nr, double dr,
               const double* w, int nvec, double* coeff, void* workspace, int64_t workspace_bytes, void* stream);

/* sh_project without any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it): the same computation and the same kernels as sh_project, bit-identical results, but the per-CTA
 * partial sums live in a static device array inside the library instead of a caller-provided workspace.  The caller still passes
 * every input and the output `coeff` (DEVICE pointers; `proj_l` HOST).  The call allocates nothing and frees nothing.
 *   Limit: the array holds sh_project_static_bytes() = 2 MiB on every GPU that loads the library (until the process exits).  A request
 *   with sh_project_workspace_bytes(ncols, nvec) above that returns SH_ERR_SCRATCH and launches nothing; on a 148-SM B200 this means
 *   min(nvec, 8) x min(ncols, 104) <= 442: any number of columns with up to 4 weight vectors, up to 55 columns with 5 to 8 (split a
 *   wider request into calls of 4 vectors, or use sh_project with your own workspace).
 *   Sharing: every call on a device uses the SAME array.  Calls ordered on one stream are safe (nothing in the array has to start at
 *   zero or survives a call); calls that OVERLAP on the GPU -- different streams, concurrently replayed graphs -- race and give
 *   wrong coefficients.  Use sh_project with separate workspaces for those. */
int sh_project_static(const double* xyz, int64_t n, int nproj, const int* proj_l, const double* radial, int nr, double dr,
                      const double* w, int nvec, double* coeff, void* stream);
int64_t sh_project_static_bytes(void);   /* size of the static scratch array: 2097152 */

/* Host-buffer entry points: same results, `xyz` and `out` are HOST pointers (pinned memory gives full
 * PCIe speed; pageable memory works).  The call copies chunks host->device, runs the kernels and copies
 * device->host on two internal streams with double buffering, and returns after `out` is complete.  The
 * staging buffers (640 MiB of device memory) and streams are created on the first host call and kept for
 * later ones; sh_host_release() frees them.  Host calls are serialized among themselves (internal mutex). */
int sh_real_host(const double* xyz, int64_t n, int lmax, double* out, int layout);
int sh_complex_host(const double* xyz, int64_t n, int lmax, double* out, int layout);
int sh_spinor_host(const double* xyz, int64_t n, int lmax, double* out, int layout);
int sh_real_f32_host(const float* xyz, int64_t n, int lmax, float* out, int layout);
/* Frees the staging buffers and streams of the host entry points (no-op if there are none). */
void sh_host_release(void);

/* Scalars (doubles for the fp64 calls, floats for sh_real_f32) written per point; -1 if lmax is out of range
 * (real, complex: [0, 32], the range of the *_ext calls; spinor: [0, 9]). */
int64_t sh_real_count(int lmax);    /* K   */
int64_t sh_complex_count(int lmax); /* 2K  */
int64_t sh_spinor_count(int lmax);  /* 8K  */

/* Element index of (l, m) in the real / complex outputs: l(l+1)+m; -1 if out of range (l <= 32). */
int sh_index_real(int l, int m);
/* Element index of (l, j, m_j) in the spinor output; half-integers are passed doubled (twoj = 2j, twomj = 2m_j);
 * -1 if the triple is not a valid spin-1/2 state with l <= 9. */
int sh_index_spinor(int l, int twoj, int twomj);

/* Launch-heuristic overrides, for benchmarking and A/B measurements only: process-global, do not change results (every
 * value selects among kernels that compute the same arithmetic).  value 0 restores the built-in default; returns
 * SH_ERR_LAYOUT for an unknown knob or a negative value. */
enum {
    SH_TUNE_PREFETCH_WINDOW_POINTS = 0, /* points per burst of the L2 input prefetch (default 262144); 1 = prefetch off */
    SH_TUNE_PROJ_AOS_MODE = 1,      /* sh_projectors AoS copy-out: 1 = warp copy, 2 = one bulk copy per row, 3 = one per tile (when possible) */
    SH_TUNE_SOA_TMA = 2,            /* SoA through TMA tensor stores (sh_real, sh_real_f32, sh_complex; tiles staged in shared memory): 0 = when possible (default), 1 = never (per-thread streaming stores) */
    SH_TUNE_PROJECT_FORM = 3,       /* sh_project polynomials: 0 or 1 = Horner in z^2 for the polar factors and (x + iy)^m by recurrence (the
                                       default of this one FP64-bound call); 2 = the factorized root-pair forms of every other call */
    SH_TUNE_PROJ_AOS_SPLIT = 4,     /* sh_projectors AoS, lmax >= 4: warps that share one 32-point tile, each evaluating part of the l-blocks: 1, 2 (default) or 4 */
    SH_TUNE_SOA_SPLIT = 5,          /* sh_real / sh_real_f32 SoA tensor-store path, lmax >= 4: warps that share a 32-point group of the tile, each evaluating part of the l-blocks: 1 or 2 (default) */
    SH_TUNE_PROJ_AOS_PAIRS = 6,     /* sh_projectors AoS staging: 0 = 16-byte stores where the rows allow (default), 1 = 8-byte stores always */
    SH_TUNE_COUNT = 7
};
int sh_set_tuning(int knob, int value);

/* Static text for an SH_ERR_* code. */
const char* sh_strerror(int code);
/* Text of the last CUDA error seen by this thread's calls ("" if none). */
const char* sh_last_cuda_error(void);
/* Number of kernels this library has launched in this process (for launch accounting in benchmarks). */
int64_t sh_kernel_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* SHB200_H */
