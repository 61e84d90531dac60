// Binning by CHANNEL RUNS (fast path).  Along a baseline, consecutive channels move the uv point by
// ~3e-4 of its length per channel, so neighbouring channels of one (integration, baseline) mostly share
// their patch origin: config 2/4 average 6.8 visibilities per run of equal [tile | origin].  Sorting
// runs instead of visibilities moves ~4.5x fewer bytes through the radix sort (PAPER.md :199 sorts every
// visibility; SURVEY hard part 7).  Pipeline:
//   map_runs_kernel   exact map of every visibility (same device function as the classic path);
//                     writes its sub-cell offsets / drop flag (1 byte) and, for every run start,
//                     (sort key, first index) into the block's own staging slots, plus the block's count
//   exclusive scan    of the block counts; compact_runs_kernel moves the staged runs to their place as
//                     (key, first index | length << 32)
//   radix sort        (key u32, value u64) over the runs, stable: equal keys stay in index order
//   exclusive scan    entries before each sorted run
//   expand_kernel     sorted runs -> the per-entry sorted (key, index) arrays of the classic path
// The result is the same list, element for element, as sorting the visibilities themselves, so
// everything downstream (tile tables, grid kernel, flush) and every output bit is unchanged.
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>
#include <thrust/iterator/transform_iterator.h>

#include "gridder_internal.cuh"
#include "map.cuh"

namespace gridder {

constexpr int kRunThreads = 256, kRunItems = 4, kRunTile = kRunThreads * kRunItems;     // expansion: entries per block
constexpr int kMapItems = 8, kMapTile = kRunThreads * kMapItems;                       // map: visibilities per block

template <bool FAST>
__global__ void __launch_bounds__(kRunThreads) map_runs_kernel(const double *__restrict__ uvw,
                                                                const double *__restrict__ scale, unsigned int n,
                                                                unsigned int n_chan, const MapParams p,
                                                                unsigned char *__restrict__ qaux,
                                                                uint32_t *__restrict__ stage_key,
                                                                uint32_t *__restrict__ stage_start,
                                                                unsigned int *__restrict__ block_count,
                                                                Counters *counters) {
    __shared__ uint32_t s_last[kRunThreads];
    __shared__ unsigned int s_warp[kRunThreads / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned int bid = blockIdx.x;
    const unsigned int base = bid * (unsigned)kMapTile + (unsigned)tid * kMapItems;    // n <= 2^32 - 4096: no wrap
    const uint32_t aux_mask = (1u << p.key.aux_bits) - 1u;
    FastMap fm;
    if (FAST) fm.init(p);
    auto key_of = [&](const double *L, double s, int &taps) -> uint32_t {
        if (FAST) return fm.key(L[0], L[1], s, p, taps);
        const VisMap m = map_vis(L[0], L[1], 0.0, s, p);
        taps = m.dropped ? 0 : m.S * m.S;
        return fast_key(m, p);
    };

    // thread 0 also maps the visibility just before the block's first one (its key decides whether the
    // block starts inside a run); done before the barrier so that it costs no extra phase
    uint32_t prev = 0xFFFFFFFFu;
    if (tid == 0 && base > 0 && base < n) {
        const unsigned int i = base - 1;
        const unsigned int tb = i / n_chan, f = i - tb * n_chan;
        const double *L = uvw + (size_t)tb * 3;
        int taps;
        prev = key_of(L, scale[f], taps) >> p.key.aux_bits;
    }
    uint32_t sk[kMapItems];
    unsigned int fch[kMapItems];
    unsigned char q[kMapItems];
    unsigned int dropped_here = 0;
    unsigned long long taps_here = 0;
    // (integration, baseline) row and channel of the thread's first visibility; the next ones by increment
    unsigned int tb = 0, f = 0;
    if (base < n) {
        tb = base / n_chan;
        f = base - tb * n_chan;
    }
#pragma unroll
    for (int k = 0; k < kMapItems; ++k) {
        sk[k] = 0xFFFFFFFFu; fch[k] = 1; q[k] = 0;
        if (base + k < n) {
            const double *L = uvw + (size_t)tb * 3;
            int taps;
            const uint32_t key = key_of(L, scale[f], taps);
            if (taps == 0) dropped_here++; else taps_here += (unsigned long long)taps;
            sk[k] = key >> p.key.aux_bits;
            q[k] = (unsigned char)(key & aux_mask);
            fch[k] = f;
            if (++f == n_chan) { f = 0; ++tb; }
        }
    }
    if (base + kMapItems <= n) {
        static_assert(kMapItems == 8, "the offsets of a thread's visibilities are stored as one 8-byte word");
        *reinterpret_cast<uint2 *>(qaux + base) =
            make_uint2((uint32_t)q[0] | ((uint32_t)q[1] << 8) | ((uint32_t)q[2] << 16) | ((uint32_t)q[3] << 24),
                       (uint32_t)q[4] | ((uint32_t)q[5] << 8) | ((uint32_t)q[6] << 16) | ((uint32_t)q[7] << 24));
    } else {
#pragma unroll
        for (int k = 0; k < kMapItems; ++k)
            if (base + k < n) qaux[base + k] = q[k];
    }
    // the sort key of the visibility just before this thread's first one
    s_last[tid] = sk[kMapItems - 1];
    __syncthreads();
    if (tid > 0) prev = s_last[tid - 1];
    // run starts: first channel of a (t, b) row, or a different [tile | origin] than the previous channel
    unsigned int flags = 0, cnt = 0;
#pragma unroll
    for (int k = 0; k < kMapItems; ++k) {
        const bool st = (base + k < n) && (fch[k] == 0 || sk[k] != prev);
        if (st) { flags |= 1u << k; cnt++; }
        prev = sk[k];
    }
    // block-wide exclusive scan of cnt
    unsigned int incl = cnt;
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    unsigned int woff = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kRunThreads / 32; ++w) {
        if (w < warp) woff += s_warp[w];
        total += s_warp[w];
    }
    if (tid == 0) block_count[bid] = total;
    // the block's runs go to its own slots (a block of kMapTile visibilities has at most kMapTile runs)
    unsigned int pos = bid * (unsigned)kMapTile + woff + incl - cnt;
#pragma unroll
    for (int k = 0; k < kMapItems; ++k)
        if (flags & (1u << k)) {
            stage_key[pos] = sk[k] << p.key.aux_bits;
            stage_start[pos] = base + k;
            ++pos;
        }
    for (int o = 16; o > 0; o >>= 1) {
        dropped_here += __shfl_xor_sync(0xffffffffu, dropped_here, o);
        taps_here += __shfl_xor_sync(0xffffffffu, taps_here, o);
    }
    if (lane == 0) {
        if (dropped_here) atomicAdd(&counters->n_dropped, (unsigned long long)dropped_here);
        if (taps_here) atomicAdd(&counters->vis_taps, taps_here);
    }
}

// One warp per map block: its staged runs move to [prefix, prefix + count) of the compact arrays, as
// (key, first index | length << 32); a run ends where the next one starts -- the next staged start of the
// block, or the first start of the next block that has one, or n.
__global__ void __launch_bounds__(256) compact_runs_kernel(const uint32_t *__restrict__ stage_key,
                                                            const uint32_t *__restrict__ stage_start,
                                                            const unsigned int *__restrict__ block_count,
                                                            const unsigned int *__restrict__ block_prefix,
                                                            unsigned int n_blocks, unsigned int n,
                                                            uint32_t *__restrict__ rkey,
                                                            unsigned long long *__restrict__ rval) {
    const unsigned int b = blockIdx.x * 8 + (threadIdx.x >> 5);
    if (b >= n_blocks) return;
    const unsigned int cnt = block_count[b], dst = block_prefix[b], src = b * (unsigned)kMapTile;
    if (cnt == 0) return;
    unsigned int next_first = n;
    if ((threadIdx.x & 31) == 0) {
        for (unsigned int bb = b + 1; bb < n_blocks; ++bb)
            if (block_count[bb] > 0) { next_first = stage_start[bb * (unsigned)kMapTile]; break; }
    }
    next_first = __shfl_sync(0xffffffffu, next_first, 0);
    for (unsigned int j = threadIdx.x & 31; j < cnt; j += 32) {
        const unsigned int st = stage_start[src + j];
        const unsigned int nx = j + 1 < cnt ? stage_start[src + j + 1] : next_first;
        rkey[dst + j] = stage_key[src + j];
        rval[dst + j] = (unsigned long long)st | ((unsigned long long)(nx - st) << 32);
    }
}

struct RunLen {
    __host__ __device__ __forceinline__ unsigned int operator()(const unsigned long long &v) const {
        return (unsigned int)(v >> 32);
    }
};

// Sorted runs -> sorted entries.  A block produces kRunTile consecutive entries: it finds the run holding
// its first entry (binary search in the scanned lengths), stages the following runs in shared memory
// and every thread looks its entries up there.
// For every expand block: the run holding its first entry (one binary search per thread, all in parallel).
__global__ void __launch_bounds__(256) expand_partition_kernel(const uint32_t *__restrict__ rcum, unsigned int n_runs,
                                                                unsigned int n_blocks, unsigned int *__restrict__ part) {
    const unsigned int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n_blocks) return;
    const unsigned int e0 = b * (unsigned)kRunTile;
    unsigned int lo = 0, hi = n_runs;                     // last run with rcum[r] <= e0
    while (hi - lo > 1) {
        const unsigned int mid = (lo + hi) >> 1;
        if (rcum[mid] <= e0) lo = mid; else hi = mid;
    }
    part[b] = lo;
}

// blk_run[g] = last run with rcum <= 64 g: where reduce_runs_kernel (grid.cu) starts looking for the runs of
// the entries 64 g .. 64 g + 63 (dense plans read the sorted runs themselves; nothing is expanded)
__global__ void __launch_bounds__(256) block_run_kernel(const uint32_t *__restrict__ rcum, unsigned int n_runs,
                                                         unsigned int n_blocks64, uint32_t *__restrict__ blk_run) {
    const unsigned int g = blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= n_blocks64) return;
    const unsigned int e0 = g * 64u;
    unsigned int lo = 0, hi = n_runs;
    while (hi - lo > 1) {
        const unsigned int mid = (lo + hi) >> 1;
        if (rcum[mid] <= e0) lo = mid; else hi = mid;
    }
    blk_run[g] = lo;
}

__global__ void __launch_bounds__(kRunThreads) expand_kernel(const uint32_t *__restrict__ rkey,
                                                              const unsigned long long *__restrict__ rval,
                                                              const uint32_t *__restrict__ rcum, unsigned int n_runs,
                                                              unsigned int n, const unsigned int *__restrict__ part,
                                                              const unsigned char *__restrict__ qaux,
                                                              uint32_t *__restrict__ keys, uint32_t *__restrict__ vals,
                                                              int tile_shift, uint32_t *__restrict__ tile_start,
                                                              uint32_t *__restrict__ tile_end) {
    __shared__ uint32_t s_cum[kRunTile + 1], s_key[kRunTile], s_start[kRunTile];
    __shared__ unsigned int s_cnt;
    const unsigned int e0 = blockIdx.x * (unsigned)kRunTile;
    const unsigned int e1 = min(n, e0 + (unsigned)kRunTile);
    const unsigned int r0 = part[blockIdx.x];
    // runs r0 .. r0 + cnt - 1 cover [e0, e1): at most kRunTile of them (every run has >= 1 entry)
    unsigned int mine = 0;
    for (unsigned int j = threadIdx.x; j < (unsigned)kRunTile; j += kRunThreads) {
        const unsigned int r = r0 + j;
        if (r >= n_runs) break;
        {
            const uint32_t c = rcum[r];
            if (c >= e1) break;                            // rcum ascends: no later run starts inside the block
            {
                const unsigned long long v = rval[r];
                const uint32_t key = rkey[r];
                s_cum[j] = c;
                s_key[j] = key;
                s_start[j] = (unsigned int)v;
                mine = j + 1;
                if (c >= e0) {
                    // the run starts in this block: the block notes where its tile starts and ends (the paper's
                    // 'first' / 'last' tables, :197; what tile_bounds_runs_kernel does on its own)
                    const uint32_t t = key >> tile_shift;
                    if (r == 0 || (rkey[r - 1] >> tile_shift) != t) tile_start[t] = c;
                    if (r == n_runs - 1) tile_end[t] = n;
                    else if ((rkey[r + 1] >> tile_shift) != t) tile_end[t] = rcum[r + 1];
                }
            }
        }
    }
    // cnt = 1 + the largest staged j (runs are staged from j = 0 without gaps)
    mine = __reduce_max_sync(0xffffffffu, mine);
    if (threadIdx.x == 0) s_cnt = 0;
    __syncthreads();
    if ((threadIdx.x & 31) == 0) atomicMax(&s_cnt, mine);
    __syncthreads();
    const unsigned int cnt = s_cnt;
    // a thread produces kRunItems consecutive entries: one search, then a walk along the staged runs
    const unsigned int ef = e0 + threadIdx.x * kRunItems;
    if (ef >= e1) return;
    unsigned int lo = 0, hi = cnt;                        // last staged run with s_cum <= ef
    while (hi - lo > 1) {
        const unsigned int mid = (lo + hi) >> 1;
        if (s_cum[mid] <= ef) lo = mid; else hi = mid;
    }
    uint32_t ko[kRunItems], vo[kRunItems];
#pragma unroll
    for (int k = 0; k < kRunItems; ++k) {
        const unsigned int e = ef + k;
        ko[k] = vo[k] = 0;
        if (e < e1) {
            while (lo + 1 < cnt && s_cum[lo + 1] <= e) ++lo;
            const unsigned int idx = s_start[lo] + (e - s_cum[lo]);
            ko[k] = s_key[lo] | (uint32_t)qaux[idx];
            vo[k] = idx;
        }
    }
    if (ef + kRunItems <= e1) {
        *reinterpret_cast<uint4 *>(keys + ef) = make_uint4(ko[0], ko[1], ko[2], ko[3]);
        *reinterpret_cast<uint4 *>(vals + ef) = make_uint4(vo[0], vo[1], vo[2], vo[3]);
    } else {
#pragma unroll
        for (int k = 0; k < kRunItems; ++k)
            if (ef + k < e1) { keys[ef + k] = ko[k]; vals[ef + k] = vo[k]; }
    }
}

// The paper's 'first' / 'last' tables (:197) from the sorted RUNS: a tile starts where a run's tile differs
// from the previous run's.  Same tables as tile_bounds_kernel builds from the entries, 7x less to read.
__global__ void __launch_bounds__(256) tile_bounds_runs_kernel(const uint32_t *__restrict__ rkey,
                                                                const uint32_t *__restrict__ rcum, unsigned int n_runs,
                                                                unsigned int n, int tile_shift,
                                                                uint32_t *__restrict__ tile_start,
                                                                uint32_t *__restrict__ tile_end) {
    for (unsigned int r = blockIdx.x * blockDim.x + threadIdx.x; r < n_runs; r += gridDim.x * blockDim.x) {
        const uint32_t t = rkey[r] >> tile_shift;
        if (r == 0 || (rkey[r - 1] >> tile_shift) != t) tile_start[t] = rcum[r];
        if (r == n_runs - 1) tile_end[t] = n;
        else if ((rkey[r + 1] >> tile_shift) != t) tile_end[t] = rcum[r + 1];
    }
}

#define GR_TRY(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return e_; } while (0)

cudaError_t runs_temp_bytes(int64_t cap, int begin_bit, int end_bit, size_t *bytes) {
    size_t a = 0, b = 0;
    cub::DoubleBuffer<uint32_t> k(nullptr, nullptr);
    cub::DoubleBuffer<unsigned long long> v(nullptr, nullptr);
    cudaError_t e = cub::DeviceRadixSort::SortPairs(nullptr, a, k, v, (long long)cap, begin_bit, end_bit, (cudaStream_t)0);
    if (e != cudaSuccess) return e;
    auto it = thrust::make_transform_iterator((const unsigned long long *)nullptr, RunLen());
    e = cub::DeviceScan::ExclusiveSum(nullptr, b, it, (unsigned int *)nullptr, (long long)cap, (cudaStream_t)0);
    *bytes = a > b ? a : b;
    return e;
}

// Map + bin by channel runs.  *used = false (nothing but the counters and qaux touched) when the
// visibilities form more runs than the plan has room for: the caller then bins them one by one.
// Synchronises the stream once: the number of runs sizes the sort.
cudaError_t launch_bin_runs(Plan &p, const double *uvw, const double *scale, long long n, int n_chan, cudaStream_t s,
                            bool *used) {
    *used = false;
    p.fused_bin = 0;
    const MapParams mp = make_map_params(p);
    const unsigned int n_blocks = (unsigned int)((n + kRunTile - 1) / kRunTile);       // expansion blocks
    const unsigned int n_mblocks = (unsigned int)((n + kMapTile - 1) / kMapTile);      // map blocks
    uint32_t *rkey[2] = {p.run_key[0], p.run_key[1]};
    unsigned long long *rval[2] = {p.run_val[0], p.run_val[1]};
    // staging slots: the second sort buffers of the classic path, which this path does not sort with
    uint32_t *stage_key = p.keys[1], *stage_start = (uint32_t *)p.vals[1];
    unsigned int *block_count = p.run_blk, *block_prefix = p.run_blk + (n_blocks + 1), *part = p.run_blk + 2 * (n_blocks + 1);
    GR_TRY(cudaMemsetAsync(block_count + n_mblocks, 0, sizeof(unsigned int), s));
    if (mp.o_shift >= 0 && mp.drop_slot == 0)
        map_runs_kernel<true><<<n_mblocks, kRunThreads, 0, s>>>(uvw, scale, (unsigned)n, (unsigned)n_chan, mp, p.qaux,
                                                                stage_key, stage_start, block_count, p.counters);
    else
        map_runs_kernel<false><<<n_mblocks, kRunThreads, 0, s>>>(uvw, scale, (unsigned)n, (unsigned)n_chan, mp, p.qaux,
                                                                 stage_key, stage_start, block_count, p.counters);
    GR_TRY(cudaGetLastError());
    size_t tb = p.cub_temp_bytes;
    GR_TRY(cub::DeviceScan::ExclusiveSum(p.cub_temp, tb, (const unsigned int *)block_count, block_prefix,
                                         (long long)n_mblocks + 1, s));
    p.n_launches += 2;
    unsigned int n_runs = 0;
    GR_TRY(cudaMemcpyAsync(&n_runs, block_prefix + n_mblocks, sizeof(unsigned int), cudaMemcpyDeviceToHost, s));
    GR_TRY(cudaStreamSynchronize(s));
    p.n_runs = n_runs;
    if ((long long)n_runs > p.run_cap) return cudaSuccess;          // too fragmented: classic path
    compact_runs_kernel<<<(n_mblocks + 7) / 8, 256, 0, s>>>(stage_key, stage_start, block_count, block_prefix, n_mblocks,
                                                           (unsigned)n, rkey[0], rval[0]);
    GR_TRY(cudaGetLastError());
    stage_mark(p, 1, s);
    cub::DoubleBuffer<uint32_t> k(rkey[0], rkey[1]);
    cub::DoubleBuffer<unsigned long long> v(rval[0], rval[1]);
    tb = p.cub_temp_bytes;
    GR_TRY(cub::DeviceRadixSort::SortPairs(p.cub_temp, tb, k, v, (long long)n_runs, p.key.aux_bits, p.key.total_bits, s));
    auto it = thrust::make_transform_iterator((const unsigned long long *)v.Current(), RunLen());
    tb = p.cub_temp_bytes;
    GR_TRY(cub::DeviceScan::ExclusiveSum(p.cub_temp, tb, it, p.run_cum, (long long)n_runs, s));
    p.srun_key = k.Current();
    p.srun_val = v.Current();
    if (p.fuse) {
        // dense plan: the pre-summation reads the sorted runs; the per-entry list is never written
        const unsigned int nb64 = (unsigned int)((n + 63) / 64);
        block_run_kernel<<<(nb64 + 255) / 256, 256, 0, s>>>(p.run_cum, n_runs, nb64, p.blk_run);
        GR_TRY(cudaGetLastError());
        p.fused_bin = 1;
    } else {
        expand_partition_kernel<<<(n_blocks + 255) / 256, 256, 0, s>>>(p.run_cum, n_runs, n_blocks, part);
        GR_TRY(cudaGetLastError());
        expand_kernel<<<n_blocks, kRunThreads, 0, s>>>(k.Current(), v.Current(), p.run_cum, n_runs, (unsigned)n, part, p.qaux,
                                                       p.keys[0], (uint32_t *)p.vals[0], p.key.tile_shift, p.tile_start,
                                                       p.tile_start + (size_t)p.n_tiles * p.n_cls);
        GR_TRY(cudaGetLastError());
    }
    if (p.fuse) {                    // (expand_kernel builds the tile tables on its way)
        const int tb_blocks = (int)min((long long)(n_runs + 255) / 256, (long long)p.n_sm * 32);
        tile_bounds_runs_kernel<<<tb_blocks, 256, 0, s>>>(k.Current(), p.run_cum, n_runs, (unsigned)n, p.key.tile_shift,
                                                          p.tile_start, p.tile_start + (size_t)p.n_tiles * p.n_cls);
        GR_TRY(cudaGetLastError());
    }
    p.sorted_sel = 0;
    p.n_launches += 5;
    *used = true;
    return cudaSuccess;
}

}  // namespace gridder
