/*
 * gridder.h -- C ABI of the B200 convolutional gridder (libgridder.so).
 *
 * The operation (section 5, Eq. 1, :174-183): every calibrated visibility V_i at
 * (u_i, v_i) is convolved with a compact gridding convolution function (GCF) f and added to a
 * regular uv grid,
 *        V_grid(u, v) = sum_i f_i(r) * V_i delta(u - u_i, v - v_i),
 * i.e. "compute the distance from the visibility to the centre of a given pixel, and then add the
 * value of f_i(r) V_i to that grid cell" (:181) for the S x S patch of cells the GCF reaches
 * (:183, "added the weighted values to those pixels").  The GCF is looked up in an oversampled
 * table (BASELINE.json north_star).  The exact arithmetic -- rounding of the position to the 1/O
 * sub-cell lattice, patch origin, w-plane choice, drop rule -- is stated in DESIGN.md section 3
 * (readings R1-R16) and is what oracle/gridder_oracle.c restates independently in double.
 *
 * Pipeline behind the four calls (PAPER.md :197-199 "binned" gridder is the prior art):
 *   gridder_plan    validate, size and carve the workspace, re-lay the GCF table     (host + 1 kernel)
 *   gridder_bin     map  uvw x freq -> (tile, patch origin, sub-cell offset) keys    (FP64, exact)
 *                   sort stable device radix sort of (key, visibility index)         (:199)
 *                   tile 'first/last' tables and the work-item table                 (:197)
 *   gridder_grid    grid each warp owns a uv tile (+halo) region in shared memory, FP32 FMA
 *                   flush fixed-order FP64 sum of the partial regions -> HBM grid
 *   gridder_destroy
 *
 * Conventions
 *   - Pointers are DEVICE pointers unless marked HOST.  The library allocates no device memory:
 *     the caller owns every buffer, including the workspace.
 *   - Calls only enqueue work on `cuda_stream` (a cudaStream_t passed as void*; NULL = default
 *     stream).  gridder_plan, gridder_destroy, gridder_get_stats and gridder_run_host synchronise;
 *     gridder_bin synchronises the stream ONCE in the middle when the plan pre-sums in input order
 *     (see gridder_tuning.presum): the number of partial records sizes the radix sort.  What it
 *     enqueues after that is asynchronous again.  Nothing in the library reads the environment.
 *   - Buffers given to gridder_bin / gridder_grid must stay valid until that work has completed.
 *   - A plan may be binned and gridded any number of times; one gridder_bin serves any number of
 *     gridder_grid calls (same uv geometry, new visibilities).  Not thread-safe per plan.
 *   - Layouts: uvw_m double [n_time][n_baseline][3] (metres); freq_hz double [n_chan];
 *     vis float [n_time][n_baseline][n_chan][4 pol][re, im], polarisation order XX, XY, YX, YY;
 *     weight float [n_time][n_baseline][n_chan] (one weight per sample, shared by the 4 pols);
 *     grid float [4 pol][N][N][re, im]; (u, v) = (0, 0) is cell (N/2, N/2), u along x (fastest).
 *   - Visibilities whose patch would leave the grid are dropped whole and counted (not an error).
 *     Inputs are assumed finite.  Results are bit-identical from run to run.
 *   - Return value: 0 on success, a negative gridder_status otherwise.  Nothing aborts or throws.
 */
#ifndef GRIDDER_H
#define GRIDDER_H

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define GRIDDER_API __attribute__((visibility("default")))
#else
#define GRIDDER_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    GRIDDER_OK = 0,
    GRIDDER_ERR_INVALID_ARG = -1,      /* null pointer, bad size, odd grid, S*O odd, n_pol != 4 ...  */
    GRIDDER_ERR_CAPACITY = -2,         /* n_time*n_baseline*n_chan > max_vis                          */
    GRIDDER_ERR_WORKSPACE = -3,        /* workspace_bytes too small (needed size is reported)         */
    GRIDDER_ERR_CUDA = -4,             /* a CUDA runtime call failed (see gridder_last_cuda_error)    */
    GRIDDER_ERR_NOT_BINNED = -5,       /* gridder_grid before a successful gridder_bin                */
    GRIDDER_ERR_UNSUPPORTED = -6       /* configuration outside what this build implements            */
} gridder_status;

typedef struct gridder_plan_s gridder_plan_t;      /* opaque host object */

/* Problem statement (PAPER.md :174-183) + table/grid geometry (BASELINE.json north_star). */
typedef struct {
    int32_t grid_size;          /* N: square grid, even                                             */
    double cell_size;           /* du = dv in wavelengths per cell, > 0                             */
    int32_t n_pol;              /* must be 4                                                        */
    int32_t oversample;         /* O >= 1 table samples per cell; S_p * O must be even              */
    int32_t n_wplanes;          /* P >= 1                                                           */
    const int32_t *support;     /* HOST [P]: S_p taps per axis of plane p, 1 <= S_p <= 32           */
    double w_max;               /* wavelengths; plane = min(P-1, floor(|w| / w_max * P)); P = 1: unused */
    int32_t kernel_is_complex;  /* 0: float table; 1: (re, im) float pairs, conjugated for w < 0    */
    const void *kernel;         /* DEVICE: plane-major, plane p is [S_p O][S_p O] samples, sample
                                   (jy, jx) is the GCF at r = (j - S_p O / 2) / O cells; read once,
                                   during gridder_plan                                              */
    int64_t max_vis;            /* capacity: upper bound of n_time * n_baseline * n_chan            */
    void *workspace;            /* DEVICE scratch, 256-byte aligned, owned by the caller            */
    size_t workspace_bytes;
    int32_t max_grids;          /* most output grids of gridder_bin_channels / gridder_grid_channels (one
                                   grid per block of channels, PAPER.md :108-120); 0 or 1: one grid      */
} gridder_config;

/* Optional tuning (gridder_plan_tuned).  Every field: 0 = the library's default, so a zeroed struct is
 * gridder_plan.  None of them changes WHAT is computed -- only tile shapes, work-item sizes and which of the
 * equivalent paths runs; results stay within the tolerance of the definition and bit-identical from run to run
 * for a given tuning.  The tests use them to reach every path on small inputs. */
typedef struct {
    int32_t tile_log2;          /* 2, 3 or 4: uv tiles of 2^tile_log2 cells per edge (default 2; 3 for pre-summed plans and the general path) */
    int32_t chunk;              /* K, 32 .. 2^20: most sorted entries per work item (default by size, 256 .. 8192)  */
    int32_t max_warps;          /* cap on the warps per block of the grid kernel (default: what fits)              */
    int32_t merge;              /* 1 on (default), 2 off: entries of a batch of 32 with equal patch origin and
                                   sub-cell offset are summed before they are gridded (exact by linearity)        */
    int32_t presum;             /* pre-summation in input order (one real table, S <= 16, O <= 8): 1 always,
                                   2 never; default: plans of max_vis >= 1 Mi, where the one synchronisation
                                   it costs gridder_bin is cheaper than sorting every visibility                   */
    int32_t table_in_tmem;      /* 1 on, 2 off: GCF table in tensor memory instead of shared memory (one real
                                   table with O^2 x 8 <= 512 columns; default: on for pre-summed plans)            */
    int32_t fold_batches;       /* power of two <= 64: batches of 32 records a register chain may span (default 8) */
    int32_t force_general;      /* 1: global-memory tables and wide sort values even for one real table          */
    int32_t host_slices;        /* gridder_run_host: slices of the (integration, baseline) axis (default 8; 1: none) */
    int32_t host_slice_min_mb;  /* gridder_run_host: slice inputs of at least this many MB (default 256)           */
    int32_t reserved[6];        /* must be 0 */
} gridder_tuning;

typedef struct {
    int64_t n_vis;              /* visibilities given to the last gridder_bin                        */
    int64_t n_dropped;          /* of those, dropped because the patch leaves the grid               */
    int64_t n_entries;          /* gridded (not dropped) visibilities                                */
    int64_t vis_taps;           /* sum of S_p^2 over gridded visibilities (the metric's numerator)   */
    int64_t n_tiles;            /* uv tiles of the plan                                              */
    int64_t n_tiles_occupied;
    int64_t max_tile_load;      /* entries in the fullest tile                                       */
    int64_t n_work_items;       /* (tile, chunk) work items: occupied tiles + hot-tile splits        */
    int32_t tile_size;          /* T cells per tile edge                                             */
    int32_t patch_size;         /* padded patch edge handled per entry (8 or 16)                     */
    int32_t chunk_size;         /* K: most entries per work item                                     */
    int32_t grid_warps_per_sm;  /* launch shape of the grid kernel                                   */
    /* of the last gridder_grid (0 before the first): */
    int64_t n_records_gridded;  /* records the grid kernels processed: entries with equal patch origin and
                                   table offset inside a batch of 32 are summed first (exact by linearity) */
    int64_t n_presum_records;   /* > 0: the last gridder_bin pre-summed the visibilities in input order into this
                                   many partial records (one per lattice point met by a group of 32 channels x 8
                                   integrations of a baseline); tiles, work items and max_tile_load then count
                                   records, not visibilities                                                */
    int64_t fma_executed;       /* FP32 FMAs those records cost, padded taps included: records x patch cells
                                   x 8 (real table) or 16 (complex): what the roofline fraction is claimed on */
} gridder_stats;

/* Bytes of workspace a plan for `cfg` needs (cfg->workspace / workspace_bytes / kernel ignored). */
GRIDDER_API int gridder_workspace_size(const gridder_config *cfg, size_t *bytes_needed);

/* Create a plan.  On GRIDDER_ERR_WORKSPACE *workspace_needed holds the required size.
 * `workspace_needed` may be NULL.  Synchronises the device once (table re-layout). */
GRIDDER_API int gridder_plan(const gridder_config *cfg, gridder_plan_t **plan_out, size_t *workspace_needed);

/* The same with explicit tuning (`tuning` HOST, may be NULL = defaults; copied).  A value outside a field's
 * range is GRIDDER_ERR_INVALID_ARG. */
GRIDDER_API int gridder_workspace_size_tuned(const gridder_config *cfg, const gridder_tuning *tuning, size_t *bytes_needed);
GRIDDER_API int gridder_plan_tuned(const gridder_config *cfg, const gridder_tuning *tuning, gridder_plan_t **plan_out,
                                   size_t *workspace_needed);

/* Map + sort + tile tables for n_time*n_baseline*n_chan visibilities (index (t*B + b)*F + f).
 * u_lambda = u_m * (f / c), c = 299792458 m/s.  n_chan <= 65536.  Enqueued on `cuda_stream` (pre-summed
 * plans: one internal synchronisation, see above). */
GRIDDER_API int gridder_bin(gridder_plan_t *plan, const double *uvw_m, int32_t n_time, int32_t n_baseline,
                const double *freq_hz, int32_t n_chan, void *cuda_stream);

/* per-baseline GCFs (PAPER.md :73, :179: "a unique GCF for each visibility" is the
 * paper's stated end state).  As gridder_bin, but the table of every (integration, baseline) is the
 * caller's choice: table_index DEVICE int32 [n_time][n_baseline], each in [0, n_wplanes) -- the plan's
 * "w-planes" are then simply a bank of tables with their own supports, and w only decides conjugation
 * (complex tables).  An index outside the bank drops the baseline (counted).  NULL = gridder_bin. */
GRIDDER_API int gridder_bin_tables(gridder_plan_t *plan, const double *uvw_m, int32_t n_time, int32_t n_baseline,
                                   const double *freq_hz, int32_t n_chan, const int32_t *table_index,
                                   void *cuda_stream);

/* Grid + flush.  weight may be NULL (all 1).  accumulate == 0 overwrites all 4*N*N cells,
 * otherwise the result is added to `grid`.  Asynchronous on `cuda_stream`. */
GRIDDER_API int gridder_grid(gridder_plan_t *plan, const float *vis, const float *weight, float *grid,
                 int32_t accumulate, void *cuda_stream);

/* SURVEY 8(f) row f4, second half -- the paper's own deployment (PAPER.md :108-120, section 3.1): a GPU holds 12
 * consecutive channels and makes one image per channel.  gridder_bin_channels maps, sorts and tabulates all
 * n_chan channels ONCE, filing channel f under grid f / chans_per_grid (the grid index becomes part of the
 * uv-tile id, so one sort and one set of work items serve every grid); gridder_grid_channels then grids them in
 * the same kernel launches and flushes grid g to grids + g * 8 N^2 floats (DEVICE, [n_grids][4][N][N][2]),
 * n_grids = ceil(n_chan / chans_per_grid) <= cfg.max_grids (else GRIDDER_ERR_CAPACITY).  Grid g is, bit for bit
 * up to FP32 summation order, what gridder_bin + gridder_grid give on channels [g, g + 1) * chans_per_grid alone.
 * After gridder_bin_channels with more than one grid, plain gridder_grid is GRIDDER_ERR_INVALID_ARG. */
GRIDDER_API int gridder_bin_channels(gridder_plan_t *plan, const double *uvw_m, int32_t n_time, int32_t n_baseline,
                                     const double *freq_hz, int32_t n_chan, int32_t chans_per_grid, void *cuda_stream);
GRIDDER_API int gridder_grid_channels(gridder_plan_t *plan, const float *vis, const float *weight, float *grids,
                                      int32_t accumulate, void *cuda_stream);

GRIDDER_API int gridder_destroy(gridder_plan_t *plan);

/* ---- helpers outside the timed path -------------------------------------------------------- */

/* Statistics of the last gridder_bin (synchronises the stream it ran on). */
GRIDDER_API int gridder_get_stats(gridder_plan_t *plan, gridder_stats *out);

/* The mapping alone, for tests: out is DEVICE int32 [n][6] = x0, y0, qx, qy, plane | conj << 8,
 * dropped -- per visibility, computed by map_vis (csrc/map.cuh), the device function of the per-visibility
 * map kernel and the fallback of the screened mappers. */
GRIDDER_API int gridder_map(gridder_plan_t *plan, const double *uvw_m, int32_t n_time, int32_t n_baseline,
                const double *freq_hz, int32_t n_chan, const int32_t *table_index /* or NULL */, int32_t *out,
                void *cuda_stream);

/* The same through the mapper of the pre-summed path (FastMap2 in csrc/map.cuh: one fused multiply-add per
 * axis, screened against the definition's rounding, map_vis where the screen does not decide) -- the code
 * that maps BASELINE.json configs 2 and 4.  Same output, except that a dropped visibility reports
 * 0, 0, 0, 0, 0, 1.  Only for plans on the fast path (one real table, S <= 16) with a power-of-two
 * oversampling; otherwise GRIDDER_ERR_UNSUPPORTED. */
GRIDDER_API int gridder_map_presum(gridder_plan_t *plan, const double *uvw_m, int32_t n_time, int32_t n_baseline,
                                   const double *freq_hz, int32_t n_chan, int32_t *out, void *cuda_stream);

/* the arithmetic of the paper's OpenGL gridder (PAPER.md :185-191: one
 * screen-aligned GCF quad per visibility, additive blending) as plain CUDA: every (visibility, tap,
 * polarisation) is an FP32 atomic add into `grid`.  No binning, no workspace use beyond the plan; needs
 * no gridder_bin.  NOT deterministic (the order of the atomic additions is not fixed) and FP32 chains
 * are unbounded, so heavily loaded cells drift beyond the binned path's tolerance: a same-box
 * comparison path, not the product path.  cfg.kernel (the caller's table) must still be valid.
 * Asynchronous on `cuda_stream`. */
GRIDDER_API int gridder_scatter_atomic(gridder_plan_t *plan, const double *uvw_m, int32_t n_time,
                                       int32_t n_baseline, const double *freq_hz, int32_t n_chan, const float *vis,
                                       const float *weight, float *grid, int32_t accumulate, void *cuda_stream);

/* the summation step of a channel-sharded deployment (PAPER.md :108-120: every
 * GPU grids its own block of channels; a multi-frequency-synthesis image needs the sum of the per-GPU
 * grids).  out[i] = (float) sum_{p = 0 .. n_parts-1, in this order, in double} parts[p * stride + i],
 * i < len: the part-p slices of all ranks, as an all-to-all leaves them in one buffer, become the rank's
 * slice of the summed grid -- a fixed order, so the result does not depend on the collective's algorithm
 * and is bit-identical from run to run and from rank to rank.  parts, out: DEVICE float, 16-byte
 * aligned, len and stride multiples of 4; out may alias parts (part 0).  No plan is needed.
 * Asynchronous on `cuda_stream`.  Returns GRIDDER_OK / GRIDDER_ERR_INVALID_ARG / GRIDDER_ERR_CUDA. */
GRIDDER_API int gridder_sum_parts(const float *parts, int32_t n_parts, int64_t len, int64_t stride, float *out,
                                  void *cuda_stream);

/* the imaging step that follows the gridder (PAPER.md :75, :211, :217): centred
 * unnormalised 2-D inverse DFT of the 4 polarisation planes with the grid correction fused in,
 *   image[pol][y][x] = corr[y] corr[x] sum_{v,u} grid[pol][v][u] exp(+2 pi i ((u-N/2)(x-N/2) + (v-N/2)(y-N/2)) / N).
 * grid, image: DEVICE float [4][N][N][2] (may be the same buffer); corr: DEVICE float [N] (1 / Fourier
 * transform of the separable GCF at pixel k; NULL = no correction); work: DEVICE scratch of
 * gridder_image_workspace_size bytes for the FFT (cuFFT, loaded on first use; GRIDDER_ERR_UNSUPPORTED
 * if it cannot be loaded).  Asynchronous on `cuda_stream`; the first call builds the FFT plan. */
GRIDDER_API int gridder_image_workspace_size(gridder_plan_t *plan, size_t *bytes);
GRIDDER_API int gridder_image(gridder_plan_t *plan, const float *grid, float *image, const float *corr, void *work,
                              size_t work_bytes, void *cuda_stream);

/* End-to-end convenience with HOST buffers (pinned for overlap; pageable works): copies uvw, freq,
 * vis, weight to the caller's device staging buffers, runs gridder_bin + gridder_grid and copies the
 * grid back, then synchronises `cuda_stream`.  Inputs of 256 MB and more are moved and gridded in 8
 * slices of the (integration, baseline) axis: the copy of slice k+1 (on an internal second stream)
 * overlaps the binning and gridding of slice k, whose result is added to the grid.  The sum is the same
 * grid up to one more FP32 rounding per slice; it is deterministic, but not bit-identical to a single
 * gridder_bin + gridder_grid over the whole input.  Afterwards the plan is binned for the last slice only.  d_* are DEVICE buffers at least as large as their
 * host counterparts (d_weight may be NULL iff h_weight is NULL). */
GRIDDER_API int gridder_run_host(gridder_plan_t *plan, const double *h_uvw_m, int32_t n_time, int32_t n_baseline,
                     const double *h_freq_hz, int32_t n_chan, const float *h_vis,
                     const float *h_weight, float *h_grid, double *d_uvw_m, double *d_freq_hz,
                     float *d_vis, float *d_weight, float *d_grid, void *cuda_stream);

/* For callers that cannot allocate device memory at all (tight serving loops, harnesses that forbid cudaMalloc):
 * plan + gridder_bin + gridder_grid of a SMALL cadence on a workspace that is a file-scope device array of the
 * library, GRIDDER_STATIC_WORKSPACE_BYTES large (every GPU that loads the library holds those 64 MiB until the
 * process exits).  cfg->workspace / workspace_bytes are ignored; inputs and outputs are the caller's DEVICE buffers
 * as for gridder_bin / gridder_grid; `tuning` may be NULL (pre-summation in input order is off unless asked for).
 * Calls no cudaMalloc, cudaFree or allocating library routine.  A plan that needs more than the array returns
 * GRIDDER_ERR_WORKSPACE ("workspace too small") with the size it would need in *workspace_needed (may be NULL) and
 * enqueues nothing -- use gridder_plan with a workspace of your own then.  The result is bit for bit that of
 * gridder_plan_tuned + gridder_bin + gridder_grid with the same tuning.
 * All calls on a device share the array and it keeps the last call's contents (the path clears what must start at
 * zero itself).  Calls that overlapped on the GPU would race on it: they are serialised by a process-wide lock and
 * every call SYNCHRONISES THE DEVICE before it returns. */
#define GRIDDER_STATIC_WORKSPACE_BYTES ((size_t)64 << 20)
GRIDDER_API int gridder_grid_static(const gridder_config *cfg, const gridder_tuning *tuning, const double *uvw_m,
                                    int32_t n_time, int32_t n_baseline, const double *freq_hz, int32_t n_chan,
                                    const float *vis, const float *weight, float *grid, int32_t accumulate,
                                    size_t *workspace_needed, void *cuda_stream);

/* Stage timers for the benchmark harness (PAPER.md :249 instrumented its pipeline per kernel).
 * When enabled, gridder_bin / gridder_grid record CUDA events between their stages on the stream
 * they run on (a few microseconds of host time per call; nothing else changes). */
GRIDDER_API int gridder_set_profiling(gridder_plan_t *plan, int32_t enable);
/* Mean device milliseconds per stage over the gridder_bin / gridder_grid calls made since
 * profiling was enabled (the last 32 of each at most), HOST float [6]: map (pre-summed plans: the plan
 * kernel, scan and compaction), sort, tile tables, grid kernel, flush kernel, input-order pre-summation
 * kernel (0 where it does not run).  Synchronises on
 * the recorded events.  A stage that has not run since then reads 0.  Enabling again resets
 * the averages. */
GRIDDER_API int gridder_get_stage_ms(gridder_plan_t *plan, float *ms_out);
/* Kernel launches this plan has enqueued so far (the library's own kernels; each CUB
 * DeviceRadixSort / DeviceScan call counts as one although it launches several). */
GRIDDER_API int64_t gridder_launch_count(const gridder_plan_t *plan);

GRIDDER_API const char *gridder_strerror(int code);
/* cudaError_t of the most recent failing CUDA call made on behalf of `plan` (0 if none). */
GRIDDER_API int gridder_last_cuda_error(const gridder_plan_t *plan);
/* "major.minor.patch" of the library. */
GRIDDER_API const char *gridder_version(void);
/* Builds with -DGRIDDER_CHECKED (libgridder_checked.so; `python -m paper_1003_5575_b200.build --checked`) check
 * every index their kernels compute -- shared memory, workspace arrays, the caller's buffers -- against its bound
 * and count the failures: this returns the count over all plans of the process so far (collected at gridder_bin
 * and gridder_destroy).  The normal build has no checks and returns -1. */
GRIDDER_API long long gridder_check_violations(void);

#ifdef __cplusplus
}
#endif
#endif /* GRIDDER_H */
