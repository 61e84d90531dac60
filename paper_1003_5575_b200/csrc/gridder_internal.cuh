// Internal declarations of libgridder.so (not part of the C ABI; see include/gridder.h).
//
// Data flow (DESIGN.md sections 5-6):
// (Plans that pre-sum in input order -- presum.cu -- sort and grid partial RECORDS instead of visibilities;
//  everything from the radix sort on is the same code.)
//   map kernel   : visibility i=(t,b,f) -> 32-bit key [class | tile | (plane) | y0l | x0l | aux] + value
//                  fast path (one real table, S <= 16): aux = drop, qy, qx in the key, value = i (u32)
//                  general path (w-planes, complex tables, S <= 32): value = (i, table offset | flags) (u64)
//   radix sort   : stable, on the [class | tile | plane | y0l | x0l] bits only (CUB DeviceRadixSort)
//   tile tables  : per (class, tile) first entry / count -> (tile, chunk) work items, per class:
//                  full chunks first, then the ragged tails
//   grid kernel  : one launch per patch class; one warp per work item, patch accumulators in
//                  registers, region in shared memory
//   flush kernel : per grid cell, FP64 sum of the partial regions that cover it, in a fixed order
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#include "../../include/gridder.h"

// GRIDDER_CHECKED builds (python -m paper_1003_5575_b200.build --checked -> libgridder_checked.so): every index the
// kernels compute for shared memory, the workspace arrays and the caller's buffers is checked against its bound
// and failures are COUNTED (Counters::violations, summed per process by gridder_check_violations) -- the pool's
// compute-sanitizer is closed, so this is the memcheck the tests run (tests/test_gpu_checked_build.py).
#ifdef GRIDDER_CHECKED
#define GR_CHECK(counters, cond) do { if (!(cond)) atomicAdd(&(counters)->violations, 1u); } while (0)
#else
#define GR_CHECK(counters, cond) do { } while (0)
#endif

namespace gridder {

constexpr int kProfRing = 32;                     // calls remembered by the stage timers
constexpr double kSpeedOfLight = 299792458.0;     // m/s (gridder.h: u_lambda = u_m * f / c)
constexpr int kMaxPlanes = 64;
constexpr int kMaxChannels = 1 << 16;              // per gridder_bin call (frequency scale table)
constexpr int kMaxClasses = 3;                    // padded patch 8 (S <= 8), 16 (S <= 16), 32 = 2x2 x 16

// General path, second word of a sorted value ("aux"): bits 0..23 table offset in 256-byte units (tables < 2 GB:
// derive()), 24..29 sub-cell offset q = qy O + qx (names a bin of the carried run, grid.cu stage_write_bins),
// 30 dropped, 31 conjugate table (w < 0).
constexpr int kAuxQShift = 24;
constexpr uint32_t kAuxOffMask = (1u << kAuxQShift) - 1u;

// Bit layout of a sort key (LSB first): [aux: qx, qy (bits_q each), drop flag -- fast path only],
// x0l, y0l (tlog each), plane (plane_bits, may be 0), virtual tile = class slot * n_tiles + tile.
struct KeyLayout {
    int bits_q;        // bits of one sub-cell offset
    int tlog;          // log2 of the tile edge T
    int aux_bits;      // 2*bits_q + 1 (fast path) or 0: not sorted on
    int plane_shift;   // aux_bits + 2*tlog
    int plane_bits;
    int tile_shift;    // plane_shift + plane_bits
    int tile_bits;     // bits of the virtual tile id
    int total_bits;    // tile_shift + tile_bits  (<= 32)
};

// Patch class: how a lane's register patch and the warp's shared region are shaped.
struct ClassGeo {
    int32_t NA, NB;          // register patch = 8 NA x 4 NB cells
    int32_t nsub;            // sub-patches per axis handled per entry (1, or 2 for 16 < S <= 32)
    int32_t SP;              // cells per axis covered per entry = 8 NA nsub
    int32_t RW, RH;          // region = tile + halo
    int32_t sub_bytes;       // one (plane, sub-patch, q) sub-table of the re-laid GCF
    int32_t warps, smem_bytes;
    int32_t region_f4;       // 2 RW RH: float4 per partial region of this class
    int64_t part_off_f4;     // where this class's partial regions start in the workspace array
};

struct MapParams {
    int32_t n_grid;          // N
    int32_t oversample;      // O
    int32_t ntx;             // tiles per grid row
    int32_t n_tiles;         // tile ids per patch class: tiles of one grid x grids of the plan
    int32_t grid_tiles;      // tiles of one grid
    int32_t chans_per_grid;  // channels filed under one grid (gridder_bin_channels); 0: one grid
    int32_t n_planes;
    int32_t general;         // 0: fast path key/value format
    int32_t is_complex;
    int32_t drop_slot;       // class slot dropped visibilities are filed under
    int32_t o_shift;         // log2 O when O is a power of two, else -1
    double cell_size;        // du
    double rcp_cell;         // RN(1 / du): screening value only, never decides a rounding (map.cuh)
    double span;             // N O: scale of the screening margin
    double w_max;
    // FastMap2's constants (map.cuh), made on the host so that no kernel recomputes them
    double fm_chalf, fm_eps, fm_span2;
    int32_t fm_half_so, fm_n_minus_s;
    const int32_t *table_index;   // null, or DEVICE [n_time][n_baseline]: the table of each baseline (row f3)
    KeyLayout key;
    int32_t support[kMaxPlanes];
    int32_t cls_slot[kMaxPlanes];       // class slot of the plane (index into the plan's classes)
    uint32_t tab_off256[kMaxPlanes];    // byte offset / 256 of the plane's re-laid table
    uint32_t q_units[kMaxPlanes];       // sub_bytes / 256 of the plane's class
};

// One (tile, chunk) work item: entries [start, start+len) of the sorted list.
struct WorkItem {
    uint32_t start;
    uint32_t len;
    uint32_t tile;
    uint32_t pad;
};

// Per virtual tile: where its work items are.
struct TileInfo {
    uint32_t count;          // entries in the tile
    uint32_t full_base;      // id of its first full-chunk item
    uint32_t n_full;         // full chunks
    uint32_t tail_item;      // id of its tail item, 0xFFFFFFFF if none
};

// Device-side counters, all integer (order-independent, so deterministic).
struct Counters {
    unsigned long long n_dropped;
    unsigned long long vis_taps;              // sum of S_p^2 over gridded visibilities
    unsigned int n_items;
    unsigned int n_occupied;
    unsigned int max_tile_load;
    unsigned int cls_begin[kMaxClasses];      // work-item range of each class slot
    unsigned int cls_end[kMaxClasses];
    unsigned int queue_head[kMaxClasses];     // work queues of the grid kernel launches
    unsigned int violations;                  // GRIDDER_CHECKED builds: index checks that failed (see GR_CHECK)
    unsigned int pad[1];
    unsigned long long n_exec[kMaxClasses];   // records gridded per class by the last gridder_grid (after merging)
};

struct GridParams {
    const uint32_t *keys;          // sorted keys
    const void *vals;              // sorted values: u32 index (fast path) or u64 (index, aux)
    const WorkItem *items;
    Counters *counters;
    const float4 *vis;             // [n][2] float4
    const float *weight;           // [n] or null
    const float4 *coef;            // re-laid table(s)
    float4 *partials;              // this class's partial regions: [item - first item of the class][region_f4]
    int32_t coef_f4;               // float4 count of the table staged in shared memory (fast path)
    int32_t fold_mask;             // register chains are folded every (fold_mask + 1) batches of 32
    int32_t cls;                   // class slot of this launch
    int32_t sub_stride_bytes;      // table distance between sub-patches (O^2 sub-tables)
    int32_t tmem_cols;             // tensor-memory columns to allocate (MODE 3)
    int32_t n_q;                   // O^2 sub-tables
    int32_t merge;                 // sum entries of a batch with equal origin and table offset before gridding
    int32_t bins;                  // ... and carry the last origin's sums from batch to batch (stage_write_bins)
    uint32_t n_sorted, n_src, max_items_cls;      // bounds (GRIDDER_CHECKED builds): sorted entries, gatherable slots, items
    KeyLayout key;
};

struct FlushParams {
    const TileInfo *tiles;         // this class's table
    const float4 *partials;        // this class's partial regions
    const Counters *counters;
    int32_t cls;
    float2 *grid;                  // [4][N][N]
    int32_t n_grid;
    int32_t ntx, nty;
    int32_t accumulate;
    const unsigned char *cover;    // null, or [n_tiles]: 0 = no region of this class reaches the tile's cells
    uint32_t max_items_cls;        // bound (GRIDDER_CHECKED builds)
};

struct Plan {
    gridder_config cfg;            // copy (support pointer re-targeted to support_copy)
    gridder_tuning tune;           // copy of the caller's tuning (zeros: defaults)
    int32_t support_copy[kMaxPlanes];
    // derived
    int32_t mode;                  // 0 fast real, 1 general real, 2 general complex
    int32_t tmem_cols;             // > 0: fast path with the table in tensor memory (columns to allocate)
    int32_t n_cls;                 // class slots in use
    ClassGeo cls[kMaxClasses];
    int32_t plane_slot[kMaxPlanes];
    uint32_t plane_off256[kMaxPlanes];
    int32_t tlog, T, ntx, nty, n_tiles;
    int32_t max_grids;             // output grids the tile tables have room for (cfg.max_grids, at least 1)
    int32_t n_tiles_cls;           // n_tiles * max_grids: tile ids per patch class
    int32_t n_grids, chans_per_grid;      // of the last bin (1, 0: plain gridder_bin)
    int32_t chunk;                 // K
    int32_t merge;                 // tuning.merge (default on)
    int32_t bins;                  // per-origin bins in the grid kernel: fast path, merging on, O^2 <= 16
    // pre-summation in input order (presum.cu); presum == 0: not used by this plan
    int32_t presum;
    int32_t presum_active;         // the last gridder_bin took it: keys / vals hold the sorted RECORDS
    int64_t ps_group_cap;          // room for this many groups (count / base arrays)
    int64_t ps_cap;                // most partial records an input may have to take this path (3/4 max_vis)
    float4 *ps_sum;                // [max_vis][2] sums of w V of the partial records, in their group's visibility slots
    int32_t ps_n_time, ps_n_bl, ps_n_chan;     // shape of the last bin
    int64_t n_sorted;              // entries of the sorted list of the last bin (records, or visibilities)
    unsigned char *ps_flags;       // [max_vis] one flag byte per visibility
    uint32_t *ps_count, *ps_base;  // [ps_group_cap + 1] records per group and their exclusive scan
    cudaEvent_t count_ev;          // recorded when the record count has reached the host (the one wait of gridder_bin)
    int32_t fold_batches;          // longest FP32 register chain, in batches of 32 entries (power of 2)
    int32_t warps_forced, n_sm;
    int64_t max_items;             // capacity of the work-item table (all classes)
    int64_t max_items_cls;         // capacity of one class's partial-region array
    int64_t partials_f4;           // float4 in all partial-region arrays
    KeyLayout key;
    // workspace carve-up (device pointers into cfg.workspace)
    uint32_t *keys[2];
    void *vals[2];
    void *cub_temp; size_t cub_temp_bytes;
    double *freq_scale;            // [kMaxChannels]: freq / c of the last bin
    uint32_t *tile_start;          // [2][n_vtiles]: first entry | one past the last entry
    unsigned long long *tile_chunks, *tile_chunks_scan;   // packed (n_full << 32 | has_tail), [n_vtiles+1]
    TileInfo *tile_info;           // [n_vtiles]
    unsigned char *tile_cover;     // [n_tiles] scratch of the later classes' flushes
    WorkItem *items;               // [max_items]
    float4 *partials;              // per class: [max_items_cls][region_f4 of the class]
    float4 *coef;                  // re-laid table(s)
    size_t coef_bytes;
    Counters *counters;
    size_t workspace_needed;
    // state
    int sorted_sel;                // which of keys[]/vals[] holds the sorted list
    int64_t n_vis;                 // of the last bin
    bool binned;
    cudaStream_t last_stream;
    int last_cuda_error;
    // harness support: stage timers and a launch counter
    bool profiling;
    cudaEvent_t ev[kProfRing][10]; // per call: bin: 0 map 1 sort 2 tables 3 | grid: 4 (presum 7) (reduce 8) grid 5 flush 6
    int64_t prof_bin_calls, prof_grid_calls;       // since profiling was enabled
    int64_t n_launches;
    cudaStream_t copy_stream;      // gridder_run_host: host-to-device copies of the next slice
    // imager (row f2)
    bool fft_ready;
    int fft_handle;
    size_t fft_work_bytes;
};

// Stage timers: call j of gridder_bin / gridder_grid records into ring slot j % kProfRing.
inline void stage_mark(Plan &p, int i, cudaStream_t s) {
    if (!p.profiling) return;
    const int64_t call = i < 4 ? p.prof_bin_calls : p.prof_grid_calls;
    cudaEventRecord(p.ev[call % kProfRing][i], s);
}

// bin.cu
MapParams make_map_params(const Plan &p);
cudaError_t launch_relayout(const Plan &p, cudaStream_t s);
cudaError_t launch_bin(Plan &p, const double *uvw, int n_time, int n_bl, const double *freq, int n_chan,
                       const int32_t *table_index, cudaStream_t s);
cudaError_t launch_map_debug(const Plan &p, const double *uvw, int n_time, int n_bl, const double *freq,
                             int n_chan, const int32_t *table_index, int32_t *out, cudaStream_t s);
cudaError_t sort_temp_bytes(int64_t n, int begin_bit, int end_bit, bool wide, size_t *bytes);

// scatter.cu (row f4's summation kernel lives beside row f1)
cudaError_t launch_sum_parts(const float *parts, int n_parts, long long len, long long stride, float *out, cudaStream_t s);

cudaError_t scan_temp_bytes(int64_t n, size_t *bytes);

// presum.cu
bool presum_fits(const Plan &p, int n_time, int n_bl, int n_chan);
cudaError_t presum_scan_temp_bytes(int64_t n, size_t *bytes);
cudaError_t launch_presum_plan(Plan &p, const double *uvw, const double *scale, int n_time, int n_bl, int n_chan,
                               cudaStream_t s, long long *n_rec);
cudaError_t launch_presum(Plan &p, const float *vis, const float *weight, cudaStream_t s);
cudaError_t launch_map_presum_debug(const Plan &p, const double *uvw, int n_time, int n_bl, const double *freq, int n_chan,
                                    int32_t *out, cudaStream_t s);

// image.cu
int image_workspace(Plan &p, size_t *bytes);
void image_destroy(Plan &p);
int launch_image(Plan &p, const float *grid, float *image, const float *corr, void *work, size_t work_bytes,
                 cudaStream_t s);

// scatter.cu
cudaError_t launch_scatter_atomic(Plan &p, const double *uvw, int n_time, int n_bl, const double *freq, int n_chan,
                                  const float *vis, const float *weight, float *grid, int accumulate,
                                  cudaStream_t s);

// grid.cu
cudaError_t configure_grid_kernel(Plan &p);          // picks warps/smem per class, sets the smem attribute
cudaError_t launch_grid(Plan &p, const float *vis, const float *weight, float *grid, int accumulate,
                        cudaStream_t s);      // grid: [p.n_grids][4][N][N][2]
size_t grid_smem_bytes(const ClassGeo &g, int tlog, int mode, size_t table_bytes, int warps, bool bins);

}  // namespace gridder
