/* wpgrid.h — C ABI of the B200-native w-projection convolutional gridder.
 *
 * Hot path of arxiv 1905.03213 (Lao, An et al. 2019).  Citations are lines of
 * the paper text and the readings in DESIGN.md §2 (R1-R20), which
 * define what the paper leaves unstated.
 *
 * Conventions
 *   - d_* arguments are DEVICE pointers owned by the caller; h_* are HOST
 *     pointers.  The library never frees or keeps them.  Inputs are not modified.
 *   - All work is enqueued on the context's CUDA stream.  Calls return without
 *     synchronising unless a host output (wpg_stats, a host grid) is requested.
 *   - Return value: WPG_OK (0) or a negative error code; text of the last error
 *     via wpg_last_error().  Nothing throws or aborts across this boundary.
 *   - There is no CPU fallback: without a CUDA device every compute call fails
 *     with WPG_ECUDA.
 *   - Complex numbers are interleaved (re, im): "c64" = 2 x float, "c128" = 2 x double.
 *   - Grid layout: grid[jv][ju], row-major, v the slow axis, N x N complex;
 *     cell (N/2, N/2) is u = v = 0.
 *   - Kernel stack layout: K[p][ov][ou][iv][iu], innermost iu; plane p starts at
 *     element plane_offset[p] and holds Q*Q*S_p*S_p complex coefficients.
 *   - Limits: grid_N <= 8192, S_p <= 32, at most 32 distinct S_p, Nw <= 256, S_p * Q even.
 */
#ifndef WPGRID_H
#define WPGRID_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct wpg_ctx wpg_ctx;              /* opaque: device id, stream, cuFFT plan cache, host scratch */

typedef enum { WPG_F32 = 0, WPG_F64 = 1 } wpg_prec;   /* grid + coefficients c64 / c128 */

enum { WPG_OK = 0, WPG_EINVAL = -1, WPG_ENOMEM = -2, WPG_ECUDA = -3 };

/* Description of a kernel stack (the "imaging parameters" of PAPER.md:108). */
typedef struct {
    int Nw;                        /* number of w-planes */
    int oversample;                /* Q */
    int grid_N;                    /* N */
    double w_max;                  /* wavelengths; planes are bin-centred on [-w_max, w_max] (R6) */
    double cell;                   /* radians per image pixel; FoV = N*cell, du = 1/FoV */
    int support_max;               /* S for uniform stacks, max S_p for ragged ones */
    const int *support;            /* HOST [Nw] per-plane S_p, or NULL = uniform support_max */
    const int64_t *plane_offset;   /* HOST [Nw+1] element offsets, or NULL = uniform p*Q*Q*S*S */
} wpg_kdesc;

typedef struct {
    int64_t n_gridded;             /* visibilities gridded */
    int64_t n_skipped_oob;         /* window not fully inside the grid (R8) */
    int64_t n_skipped_zero_weight; /* weight == 0 (flagged, R9) */
    int64_t n_clamped_w;           /* gridded with |w| > w_max, clamped to the edge plane (R6, R19) */
    int64_t n_updates;             /* sum of S_p^2 over gridded visibilities (the metric's unit) */
} wpg_stats;

/* ---- context ---------------------------------------------------------------------------- */
/* device: CUDA ordinal.  cuda_stream: a cudaStream_t (NULL = legacy default stream). */
int  wpg_create(wpg_ctx **out, int device, void *cuda_stream);
void wpg_destroy(wpg_ctx *ctx);
const char *wpg_last_error(const wpg_ctx *ctx);   /* ctx may be NULL: last error of a failed wpg_create */
int  wpg_version(void);

/* Tuning knobs (all have defaults, 0 = default): "segment" = records per gridder work item;
 * "ctas_per_sm" = gridder CTAs per SM; "key_bits" = log2 cap of the binning sort-key space.  Uniform stacks
 * (default 24: a 64 MB offset table that stays in L2): the key is (support class, j0u, j0v) at full resolution
 * unless that exceeds the cap,
 * then low bits of j0v are dropped.  Ragged stacks: the cap is a budget (default: about one key per visibility,
 * 2^24 .. 2^27) split among the support classes on the device after a census of the classes.  "timing" 0/1 (see wpg_phase_ms); "no_pairs" 0/1 (1: fp32 even
 * supports go through the generic run gridder instead of the pair gridder, and wpg_degrid / wpg_grid_pol take their
 * general kernels — for A/B comparison);
 * "row_block" = rows per time step when the rows come time-major, baseline-minor (the row order of a
 * Measurement Set; 0 = unknown, the default): a binning thread then handles the same
 * baseline at consecutive time steps, whose samples mostly hit the same grid point, and
 * updates the bucket counter once per run instead of once per visibility.  A hint only: any value gives
 * the same result.
 * "bin_tile" (with "row_block"; default 16, rounded down to a power of two): consecutive blocks of the binning passes
 * take this many successive groups of time steps of the same 256 baselines / channels, so that the blocks resident
 * together hit the same bucket counters and record stretches while those are still in L2.
 * "chunk_sort" 0/1 (default 1): where the sort key drops low bits of j0v (grids above 4096^2, the sparse support classes
 * of a ragged stack) a fourth pass sorts chunks of 32 consecutive records by the full window start, so that the gridder's
 * window sweeps each bucket monotonically; with it on, the default key cap of a uniform stack whose full-resolution key
 * space exceeds 2^24 follows the data (about 16 records per key, 2^20 .. 2^24).
 * "compress" 0/1 (default 1): record compression — a binning thread's consecutive
 * visibilities with the same plane, window start and sub-cell offsets share one sorted record carrying the sum of their
 * weight * vis; the grid is unchanged (gridding is linear), the counters still count visibilities.  Effective with
 * "row_block" (consecutive samples of one baseline and channel).
 * Unknown name -> WPG_EINVAL. */
int  wpg_set_option(wpg_ctx *ctx, const char *name, int64_t value);

/* Instrumentation (bench.py's roofline and gpu_launches figures).
 * wpg_launch_count: number of this library's own CUDA kernels the context has launched so far
 * (memsets, copies and cuFFT's internal kernels are not counted).
 * Option "timing" = 1 makes wpg_grid record CUDA events on the context's stream before the
 * binning pass, between binning and gridder, and after the gridder; wpg_phase_ms then waits for
 * the last event and returns {binning ms, gridder ms} averaged over the wpg_grid calls made
 * since the previous wpg_phase_ms (WPG_EINVAL if there were none; at most 4096 are kept). */
int64_t wpg_launch_count(const wpg_ctx *ctx);
int  wpg_phase_ms(wpg_ctx *ctx, double *h_out2);

/* ---- a0: W-kernel stack (setup, untimed) — PAPER.md:30 "new convolution kernel function";
 *      DESIGN.md R1-R3, R5-R7, steps K1-K6 -------------------------------------------------- */
/* Taper psi(nu) (R2) at n host points; independent Legendre-series implementation. */
int  wpg_taper(const double *h_nu, int64_t n, double *h_out);
/* Per-plane support by rule K6 (R20) and the matching plane offsets.  Host outputs. */
int  wpg_ragged_support(int Nw, double w_max, int grid_N, double cell, int oversample,
                        int S_min, int S_max, int *h_support_out /*[Nw]*/,
                        int64_t *h_plane_offset_out /*[Nw+1]*/);
int64_t wpg_wkernel_elems(int Nw, int support, int oversample);          /* Nw*Q*Q*S*S */
/* Build the stack described by *desc (uniform if desc->support == NULL) into d_kernels_out
 * (caller-allocated, c64 for WPG_F32 — rounded from fp64 — or c128 for WPG_F64).
 * All arithmetic is fp64 on the device, including the taper and the normalisation scalar (K5): the call allocates
 * nothing, copies nothing from the host and does not synchronise; temporaries live in the caller's workspace
 * (wpg_wkernel_workspace_bytes: the image-plane samples, twiddles and tables of the largest support group). */
size_t wpg_wkernel_workspace_bytes(const wpg_kdesc *desc);
int  wpg_wkernel_build(wpg_ctx *ctx, const wpg_kdesc *desc, wpg_prec prec, void *d_kernels_out,
                       void *d_workspace, size_t workspace_bytes);

/* ---- a1 + a2: binning and gridding — PAPER.md:30, 62-84 ------------------------------------ */
/* Bytes of device scratch wpg_grid needs for this problem size. */
size_t wpg_grid_workspace_bytes(const wpg_ctx *ctx, int64_t nrow, int nchan, const wpg_kdesc *desc,
                                wpg_prec prec);
/* grid += gridding of all (row, chan) visibilities (O4 G1-G7).
 *   d_vis    c64   [nrow][nchan]
 *   d_uvw    f64   [nrow][3], metres (R10)
 *   d_weight f32   [nrow][nchan], 0 = flagged
 *   d_freq   f64   [nchan], Hz      (wavelength inputs: nchan = 1, freq = {299792458})
 *   d_kernels      c64 | c128 stack matching desc and prec
 *   d_grid   c64 | c128 [N][N], ACCUMULATED INTO (caller zeroes)
 *   h_stats_or_null: if non-NULL the call synchronises the stream and fills the counters. */
int  wpg_grid(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
              const double *d_freq, int64_t nrow, int nchan, const void *d_kernels,
              const wpg_kdesc *desc, wpg_prec prec, void *d_grid,
              void *d_workspace, size_t workspace_bytes, wpg_stats *h_stats_or_null);
/* wpg_grid without a workspace argument and without any device allocation (csrc/wpg_static.cu), for callers that
 * cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it.  The scratch
 * (counters, bucket table, sorted records) is a file-scope device array of WPG_STATIC_SCRATCH_BYTES that every GPU
 * holding this library's module keeps until the process exits; its device address is looked up once per device
 * (cudaGetSymbolAddress, with the context's device current) on the first call.
 *   Arguments, layouts, result and h_stats_or_null exactly as wpg_grid; d_grid is ACCUMULATED INTO.
 *   Limit: wpg_grid_workspace_bytes(ctx, nrow, nchan, desc, prec) <= wpg_static_scratch_bytes() = 64 MiB — fp32:
 *   3.1e6 visibilities per call at N = 2048, 3.9e6 at N = 1024 or 8192 (fp64: two thirds of that); N = 4096 and
 *   ragged stacks need option "key_bits" <= 23 (their default 2^24-entry bucket table alone is 64 MiB).  Larger problems return
 *   WPG_ENOMEM with the two sizes in wpg_last_error and launch nothing (split the rows over several calls —
 *   gridding is additive — or use wpg_grid with a workspace of your own).
 *   Calls no cudaMalloc / cudaFree / allocating library routine (a ragged stack's first call on a context creates
 *   its three side streams, which hold no device memory).  Does not synchronise unless h_stats is given.
 *   The array is shared by every call on the device and keeps the last call's contents; the call clears what must
 *   start at zero on the context's stream.  Calls that overlap on the GPU (several contexts or streams) race. */
#define WPG_STATIC_SCRATCH_BYTES ((size_t)64 << 20)
size_t wpg_static_scratch_bytes(void);
int  wpg_grid_static(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                     const double *d_freq, int64_t nrow, int nchan, const void *d_kernels,
                     const wpg_kdesc *desc, wpg_prec prec, void *d_grid, wpg_stats *h_stats_or_null);
/* Same result by the naive design: one global atomic per update, no sorting (the measured
 * "atomic roofline" the tiled gridder must beat; "write access ... in an atomic manner"). */
int  wpg_grid_naive(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                    const double *d_freq, int64_t nrow, int nchan, const void *d_kernels,
                    const wpg_kdesc *desc, wpg_prec prec, void *d_grid, wpg_stats *h_stats_or_null);
/* End-to-end variant with HOST buffers: copies the inputs to device scratch owned by the
 * context (grown on demand; from 2^20 rows on in four row chunks on a copy stream, chunk k being binned and
 * gridded while chunk k + 1 crosses PCIe — gridding is additive), zero-fills a device grid, runs wpg_grid, copies the grid to
 * h_grid_out (overwritten, [N][N] c64|c128) and synchronises.  d_kernels stays on the device.
 * If h_image_out_or_null is non-NULL the dirty image (wpg_dirty_image with weight_sum) is formed
 * on the device as well and copied to it ([N][N] fp32|fp64). */
int  wpg_grid_host(wpg_ctx *ctx, const void *h_vis, const double *h_uvw, const float *h_weight,
                   const double *h_freq, int64_t nrow, int nchan, const void *d_kernels,
                   const wpg_kdesc *desc, wpg_prec prec, void *h_grid_out, wpg_stats *h_stats_or_null,
                   void *h_image_out_or_null, double weight_sum);

/* Binning alone (step a1), for tests and profiling: fills the workspace exactly as wpg_grid
 * does and reports where things are.  Offsets are in bytes from d_workspace. */
typedef struct {
    int64_t n_records;       /* valid visibilities = sorted records */
    int64_t n_keys;          /* number of sort keys = n_classes * keys_per_class */
    int32_t n_classes;       /* distinct supports; key = (class * N + j0u) * ceil(N / 2^key_shift) + (j0v >> key_shift) */
    int32_t key_shift;       /* -1 for ragged stacks: each class gets its own shift, chosen on the device from a
                                census of the classes so that the key budget (n_keys) goes where the visibilities are */
    int32_t record_bytes;    /* 16 (fp32) or 24 (fp64) */
    int32_t keys_per_class;
    int64_t off_records;     /* records sorted by key: {re, im, pos = j0u | j0v << 16, koff} */
    int64_t off_bucket_start;/* uint32 [n_keys + 1] */
} wpg_bin_info;
int  wpg_bin(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
             const double *d_freq, int64_t nrow, int nchan, const wpg_kdesc *desc, wpg_prec prec,
             void *d_workspace, size_t workspace_bytes, wpg_bin_info *h_info_out,
             wpg_stats *h_stats_or_null);

/* ---- the paper's own data order: Eqs. (1)-(2), PAPER.md:62-84 -------------------------
 * Baseline index I_B = (-S^2 + 2 S N_ant + S)/2 + |ant1 - ant2|, S = min(ant1, ant2)  (Eq. 1; autocorrelation
 * slots included: N_ant (N_ant + 1) / 2 values), count array C, B_start_index = exclusive prefix sum of C (Eq. 2),
 * rows re-ordered "grouped by baseline and then ordered by time" (time = input row order: a stable re-order).
 *   d_ant1, d_ant2  int32 [nrow] antenna IDs in 0 .. n_ant - 1 (n_ant <= 4096); at most 8192 rows per baseline
 *                   and call (WPG_EINVAL otherwise — chunk the input in time).
 * wpg_baseline_reorder: the re-order alone (tests): d_bstart_out u32 [N_ant (N_ant + 1) / 2 + 1] = Eq. (2) with the
 *   row count appended, d_perm_out u32 [nrow], perm[slot] = input row.  Synchronises.
 * wpg_grid_baseline_order: grid += gridding of all visibilities as wpg_grid does (same arguments, uniform stacks
 *   only), but with the records in baseline-then-time order and no position sort: the register accumulator
 *   walks each baseline's time series and writes out when the grid point changes.  Same result
 *   as wpg_grid up to summation order.  Synchronises once (after the re-order, to check the antenna IDs). */
size_t wpg_baseline_workspace_bytes(int64_t nrow, int nchan, int n_ant, wpg_prec prec);
int  wpg_baseline_reorder(wpg_ctx *ctx, const int *d_ant1, const int *d_ant2, int n_ant, int64_t nrow,
                          unsigned *d_bstart_out, unsigned *d_perm_out, void *d_workspace, size_t workspace_bytes);
int  wpg_grid_baseline_order(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight,
                             const double *d_freq, const int *d_ant1, const int *d_ant2, int n_ant,
                             int64_t nrow, int nchan, const void *d_kernels, const wpg_kdesc *desc,
                             wpg_prec prec, void *d_grid, void *d_workspace, size_t workspace_bytes,
                             wpg_stats *h_stats_or_null);

/* ---- polarisation axis (data are row x channel x polarisation) ----------
 * The npol correlations of a (row, channel) share position, weight and coefficient slice:
 *   grid[pol][j0v+iv][j0u+iu] += (weight[r][c] * vis[r][c][pol]) * K[p][ov][ou][iv][iu]   for every pol,
 * i.e. npol independent griddings of wpg_grid with one coefficient fetch for all of them.  npol = 2 or 4
 * (WPG_EINVAL otherwise); fp32 and fp64; any stack wpg_grid takes (uniform or ragged, even or odd supports).
 * Uniform fp32 stacks of support 8 or 16 (16-byte aligned) take the pair gridder (one 16-byte load feeds 2 npol
 * updates), everything else the general cell gridder, one launch per support class.
 *   d_vis c64 [nrow][nchan][npol]    d_weight f32 [nrow][nchan]    d_grid c64 | c128 [npol][N][N], ACCUMULATED INTO.
 * wpg_stats counts (row, channel) samples; n_updates = sum of S^2 over them (x npol grid-point updates). */
size_t wpg_grid_pol_workspace_bytes(const wpg_ctx *ctx, int64_t nrow, int nchan, int npol, const wpg_kdesc *desc,
                                    wpg_prec prec);
int  wpg_grid_pol(wpg_ctx *ctx, const void *d_vis, const double *d_uvw, const float *d_weight, const double *d_freq,
                  int64_t nrow, int nchan, int npol, const void *d_kernels, const wpg_kdesc *desc, wpg_prec prec,
                  void *d_grid, void *d_workspace, size_t workspace_bytes, wpg_stats *h_stats_or_null);

/* ---- degridding: the adjoint of wpg_grid with unit weights ---------------
 *   vis_out[r][c] = sum over the S x S window of grid[j0v+iv][j0u+iu] * conj(K[p][ov][ou][iv][iu]),
 * plane, window and sub-cell offsets exactly as in wpg_grid (G1-G4); a visibility whose window is not fully inside
 * the grid is predicted as 0.  With grid = centred FFT of (model image / taper) this predicts the visibilities of
 * the model (measurement model O1).
 *   d_grid  c64 | c128 [N][N] (not modified)      d_vis_out  c64 | c128 [nrow][nchan] (overwritten)
 *   h_counts2_or_null: {predicted, outside}; if non-NULL the call synchronises. */
size_t wpg_degrid_workspace_bytes(int nchan);
int  wpg_degrid(wpg_ctx *ctx, const void *d_grid, const double *d_uvw, const double *d_freq, int64_t nrow, int nchan,
                const void *d_kernels, const wpg_kdesc *desc, wpg_prec prec, void *d_vis_out,
                void *d_workspace, size_t workspace_bytes, int64_t *h_counts2_or_null);

/* ---- multi-GPU: shard the rows, one reduce of the grid -------------------------
 * The paper's decomposition: the visibility rows are split among the ranks, every rank
 * grids its rows into a private full-size grid, and the grids are summed on the master.  The library side of it is
 * this host function; the sum is ONE collective of the N x N complex grid, issued by the binding through
 * torch.distributed (NCCL reduce over NVLink on GPUs; paper_1905_03213_b200/sharded.py).
 * Rows [*row0, *row1) of rank `rank` of `world`: contiguous, disjoint, covering [0, nrow) exactly, sizes equal to
 * within one unit; the unit is one row, or `row_block` rows (a time step of time-major data) if row_block > 0, so that
 * a shard keeps whole time steps and the binning's rows-per-time-step hint stays valid inside it.
 * Host only; returns WPG_EINVAL for world < 1, rank outside [0, world), nrow < 0 or row_block < 0. */
int  wpg_shard_rows(int64_t nrow, int64_t row_block, int world, int rank, int64_t *row0, int64_t *row1);

/* Machine-limit microbenchmarks (instrumentation; SURVEY.md §8(d) wants fractions of MEASURED peaks).
 * which: 0 = red.global.add.v2.f32, a warp per 256-byte row segment at a pseudo-random place of the buffer (the
 *            naive gridder's pattern; "write access ... in an atomic manner");
 *        1 = the same, every lane its own pseudo-random cell;   2 = L1-resident 16-byte loads;
 *        3 = fma.rn.f32x2;   4 = fma.rn.f64;
 *        5 / 6 = the pattern of 0 issued as one cp.reduce.async.bulk (copy engine) per 256-byte / 64-byte segment staged
 *            in shared memory;
 *        7 / 8 = the inner loop of a shared-memory subgrid accumulator (64 x 64-cell tile + halo per CTA, S = 8, one
 *            L1-resident coefficient slice per record): 7 with red.shared.add.f32, 8 with plain load / add / store
 *            (the ceiling of a warp-owned tile); h_out[0] = grid updates/s;
 *        9 = 16-byte loads of whole 512-byte slices at pseudo-random places of an L2-resident, L1-missing 32 MiB
 *            region (the coefficient feed when the slices do not stay in L1).  2, 7, 8, 9 need buf_bytes >= 16 MiB.
 * d_buf: device scratch, buf_bytes >= 1 MiB (the reductions use the largest power-of-two number of 8-byte cells
 * that fits; its contents are overwritten).  h_out[0] = operations/s, h_out[1] = kernel ms.  Synchronises. */
int  wpg_microbench(wpg_ctx *ctx, int which, int iters, void *d_buf, size_t buf_bytes, double *h_out /*[2]*/);

/* ---- a3: dirty image — PAPER.md:52, 88 (IFFT of the grid), R11 (grid correction) ---------- */
size_t wpg_dirty_image_workspace_bytes(int grid_N, wpg_prec prec);
/* image[jm][jl] = Re(centred inverse FFT of grid) * N^2-normalised / weight_sum / taper;
 * d_image real fp32|fp64 [N][N]; d_grid is not modified.  Workspace (caller's): the transform's output and the taper
 * table, evaluated on the device at every call; the context keeps only the cuFFT plan.  Does not synchronise. */
int  wpg_dirty_image(wpg_ctx *ctx, const void *d_grid, const wpg_kdesc *desc, double weight_sum,
                     wpg_prec prec, void *d_image, void *d_workspace, size_t workspace_bytes);

#ifdef __cplusplus
}
#endif
#endif /* WPGRID_H */
