// Internal declarations of libgridder.so (not part of the C ABI; see include/gridder.h).
//
// Data flow:
//   map kernel   : visibility i=(t,b,f) -> 32-bit key  [tile | y0l | x0l | drop | qy | qx]  + value i
//   radix sort   : stable, on the [tile | y0l | x0l] bits only (CUB DeviceRadixSort)
//   tile tables  : per tile first entry / count -> (tile, chunk) work items, full chunks first
//   grid kernel  : one warp per work item, patch accumulators in registers, region in shared memory
//   flush kernel : per grid cell, FP64 sum of the partial regions that cover it, in a fixed order
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#include "../../include/gridder.h"

namespace gridder {

constexpr int kProfRing = 32;                     // calls remembered by the stage timers
constexpr double kSpeedOfLight = 299792458.0;     // m/s (gridder.h: u_lambda = u_m * f / c)

// Bit layout of a sort key (LSB first): qx, qy (bits_q each), drop flag, x0l, y0l (tlog each), tile.
struct KeyLayout {
    int bits_q;        // bits of one sub-cell offset
    int tlog;          // log2 of the tile edge T
    int aux_bits;      // 2*bits_q + 1: not sorted on
    int tile_shift;    // aux_bits + 2*tlog
    int tile_bits;     // bits of the tile id
    int total_bits;    // tile_shift + tile_bits  (<= 32)
};

struct MapParams {
    int32_t n_grid;          // N
    int32_t oversample;      // O
    int32_t support;         // S (single plane)
    int32_t half_so;         // S*O/2
    int32_t ntx;             // tiles per grid row
    double cell_size;        // du
    KeyLayout key;
};

// One (tile, chunk) work item: entries [start, start+len) of the sorted list.
struct WorkItem {
    uint32_t start;
    uint32_t len;
    uint32_t tile;
    uint32_t pad;
};

// Per tile: where its work items are.  Items [0, n_full_total) are the full chunks (len == K) in
// tile order, items [n_full_total, n_items) the ragged tails in tile order.
struct TileInfo {
    uint32_t count;          // entries in the tile
    uint32_t full_base;      // id of its first full-chunk item
    uint32_t n_full;         // full chunks
    uint32_t tail_item;      // id of its tail item, 0xFFFFFFFF if none
};

// Device-side counters, all integer (order-independent, so deterministic).
struct Counters {
    unsigned long long n_dropped;
    unsigned int n_items;          // full + tail
    unsigned int n_full_total;
    unsigned int n_occupied;
    unsigned int max_tile_load;
    unsigned int queue_head;       // work-item queue of the grid kernel
    unsigned int pad[9];
};

struct GridParams {
    const uint32_t *keys;          // sorted keys
    const uint32_t *vals;          // sorted visibility indices
    const WorkItem *items;
    const Counters *counters_ro;
    Counters *counters;
    const float4 *vis;             // [n][2] float4
    const float *weight;           // [n] or null
    const float4 *coef;            // re-laid table: [O*O][NA][32 lanes][NB] floats
    float4 *partials;              // [item][2][RH*RW] float4
    int32_t coef_f4;               // float4 count of the table
    int32_t fold_mask;             // register chains are folded every (fold_mask + 1) batches of 32
    KeyLayout key;
};

struct FlushParams {
    const TileInfo *tiles;
    const Counters *counters;
    const float4 *partials;
    float2 *grid;                  // [4][N][N]
    int32_t n_grid;
    int32_t ntx, nty;
    int32_t accumulate;
};

struct Plan {
    gridder_config cfg;            // copy (support pointer re-targeted to support_copy)
    int32_t support_copy[64];
    // derived
    int32_t S, NA, NB, tlog, T, ntx, nty, n_tiles;
    int32_t RW, RH, region_f4;     // region_f4 = 2*RH*RW float4 per work item
    int32_t chunk;                 // K
    int32_t fold_batches;          // longest FP32 register chain, in batches of 32 entries (power of 2)
    int32_t warps, n_sm, smem_bytes;
    int64_t max_items;
    KeyLayout key;
    // workspace carve-up (device pointers into cfg.workspace)
    uint32_t *keys[2], *vals[2];
    void *cub_temp; size_t cub_temp_bytes;
    uint32_t *tile_start;          // [2][n_tiles]: first entry | one past the last entry
    unsigned long long *tile_chunks, *tile_chunks_scan;   // packed (n_full << 32 | has_tail), [n_tiles+1]
    TileInfo *tile_info;           // [n_tiles]
    WorkItem *items;               // [max_items]
    float4 *partials;              // [max_items][region_f4]
    float4 *coef;                  // re-laid table
    int32_t coef_f4;
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
    cudaEvent_t ev[kProfRing][7];  // per call: bin: 0 map 1 sort 2 tables 3 | grid: 4 grid 5 flush 6
    int64_t prof_bin_calls, prof_grid_calls;       // since profiling was enabled
    int64_t n_launches;
};

// Stage timers: call j of gridder_bin / gridder_grid records into ring slot j % kProfRing.
inline void stage_mark(Plan &p, int i, cudaStream_t s) {
    if (!p.profiling) return;
    const int64_t call = i < 4 ? p.prof_bin_calls : p.prof_grid_calls;
    cudaEventRecord(p.ev[call % kProfRing][i], s);
}

// bin.cu
cudaError_t launch_relayout(const Plan &p, cudaStream_t s);
cudaError_t launch_bin(Plan &p, const double *uvw, int n_time, int n_bl, const double *freq, int n_chan,
                       cudaStream_t s);
cudaError_t launch_map_debug(const Plan &p, const double *uvw, int n_time, int n_bl, const double *freq,
                             int n_chan, int32_t *out, cudaStream_t s);
cudaError_t sort_temp_bytes(int64_t n, int begin_bit, int end_bit, size_t *bytes);
cudaError_t scan_temp_bytes(int64_t n, size_t *bytes);

// grid.cu
cudaError_t configure_grid_kernel(Plan &p);          // picks warps/smem, sets the smem attribute
cudaError_t launch_grid(Plan &p, const float *vis, const float *weight, float *grid, int accumulate,
                        cudaStream_t s);
size_t grid_smem_bytes(int NA, int NB, int tlog, int oversample, int warps);

}  // namespace gridder
