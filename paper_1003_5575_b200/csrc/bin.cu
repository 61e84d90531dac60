// gridder_bin: map (uvw x freq -> key), stable radix sort, tile tables and work items.
// PAPER.md :181 "calculate which patch", :197 "sorted the visibilities according to the bin",
// "look up tables of the 'first' and 'last' visibilities within each bin", :199 sort on the GPU.
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>
#include <cub/util_type.cuh>

#include "gridder_internal.cuh"

namespace gridder {

// ------------------------------------------------------------------------------------------
// GCF table re-layout: user table K[jy][jx] ([S*O]^2) -> coef[q = qy*O + qx][a][lane][b], the order
// the grid kernel's lanes read it in (one vector load per lane per column block a).  Lane
// (rq = lane >> 3, c8 = lane & 7) owns taps ty = rq + 4 b, tx = c8 + 8 a; taps beyond S are zero
// (the patch is padded to 8 NA x 4 NB cells).
// ------------------------------------------------------------------------------------------
__global__ void relayout_kernel(const float *__restrict__ table, float *__restrict__ coef, int S, int O,
                                int NA, int NB) {
    const int total = O * O * NA * 32 * NB;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < total; i += gridDim.x * blockDim.x) {
        int b = i % NB;
        int lane = (i / NB) % 32;
        int a = (i / (NB * 32)) % NA;
        int q = i / (NB * 32 * NA);
        int qy = q / O, qx = q % O;
        int ty = (lane >> 3) + 4 * b, tx = (lane & 7) + 8 * a;
        float v = 0.f;
        if (ty < S && tx < S) v = table[(size_t)(qy + ty * O) * (S * O) + (qx + tx * O)];
        coef[i] = v;
    }
}

cudaError_t launch_relayout(const Plan &p, cudaStream_t s) {
    const int total = p.coef_f4 * 4;
    relayout_kernel<<<(total + 255) / 256, 256, 0, s>>>((const float *)p.cfg.kernel, (float *)p.coef,
                                                         p.S, p.cfg.oversample, p.NA, p.NB);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// The mapping (steps 1-4).  Every FP64 operation is an explicit
// round-to-nearest intrinsic, so no FMA contraction can change a result: this must agree with the
// definition to the last bit, because one visibility in the wrong sub-cell is far outside the
// tolerance.
// ------------------------------------------------------------------------------------------
struct AxisMap {
    long long x0;   // patch origin
    int q;          // sub-cell table offset in [0, O)
    bool far;       // hopelessly off the grid
};

__device__ __forceinline__ long long floor_div_ll(long long a, long long b) {
    long long q = a / b;
    if ((a % b != 0) && (a < 0)) q -= 1;
    return q;
}

__device__ __forceinline__ AxisMap map_axis(double coord_lambda, const MapParams &p) {
    AxisMap m;
    const double a = __ddiv_rn(coord_lambda, p.cell_size);
    const double g = __dadd_rn(a, (double)(p.n_grid / 2));
    const double h = __dmul_rn(g, (double)p.oversample);
    const double r = floor(__dadd_rn(h, 0.5));
    m.far = !(r > -1.0e15 && r < 1.0e15);
    const long long X = m.far ? 0 : (long long)r;
    const long long A = X - (long long)p.half_so;
    const long long O = p.oversample;
    m.x0 = floor_div_ll(A + O - 1, O);
    m.q = (int)(m.x0 * O - A);
    if (m.far) { m.x0 = -(1ll << 61); m.q = 0; }
    return m;
}

struct VisMap {
    long long x0, y0;
    int qx, qy;
    bool dropped;
};

__device__ __forceinline__ VisMap map_vis(double u_m, double v_m, double s, const MapParams &p) {
    const double ul = __dmul_rn(u_m, s), vl = __dmul_rn(v_m, s);
    const AxisMap mx = map_axis(ul, p), my = map_axis(vl, p);
    VisMap m;
    m.x0 = mx.x0; m.y0 = my.x0; m.qx = mx.q; m.qy = my.q;
    const long long N = p.n_grid, S = p.support;
    m.dropped = mx.far || my.far || m.x0 < 0 || m.x0 + S > N || m.y0 < 0 || m.y0 + S > N;
    return m;
}

__global__ void __launch_bounds__(256) map_kernel(const double *__restrict__ uvw,
                                                   const double *__restrict__ freq, long long n_tb,
                                                   int n_chan, MapParams p, uint32_t *__restrict__ keys,
                                                   uint32_t *__restrict__ vals, Counters *counters) {
    const long long n = n_tb * n_chan;
    unsigned int dropped_here = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        const long long tb = i / n_chan;
        const int f = (int)(i - tb * n_chan);
        const double s = __ddiv_rn(freq[f], kSpeedOfLight);
        const VisMap m = map_vis(uvw[tb * 3 + 0], uvw[tb * 3 + 1], s, p);
        uint32_t key;
        if (m.dropped) {
            key = 1u << (2 * p.key.bits_q);          // tile 0, origin (0,0), drop flag
            dropped_here++;
        } else {
            const uint32_t x0 = (uint32_t)m.x0, y0 = (uint32_t)m.y0;
            const uint32_t tmask = (1u << p.key.tlog) - 1u;
            const uint32_t tile = (y0 >> p.key.tlog) * (uint32_t)p.ntx + (x0 >> p.key.tlog);
            key = (tile << p.key.tile_shift) | ((y0 & tmask) << (p.key.aux_bits + p.key.tlog)) |
                  ((x0 & tmask) << p.key.aux_bits) | ((uint32_t)m.qy << p.key.bits_q) | (uint32_t)m.qx;
        }
        keys[i] = key;
        vals[i] = (uint32_t)i;
    }
    // one integer atomic per warp that saw drops (the count does not depend on the order)
    for (int o = 16; o > 0; o >>= 1) dropped_here += __shfl_xor_sync(0xffffffffu, dropped_here, o);
    if ((threadIdx.x & 31) == 0 && dropped_here)
        atomicAdd(&counters->n_dropped, (unsigned long long)dropped_here);
}

__global__ void __launch_bounds__(256) map_debug_kernel(const double *__restrict__ uvw,
                                                         const double *__restrict__ freq, long long n_tb,
                                                         int n_chan, MapParams p, int32_t *__restrict__ out) {
    const long long n = n_tb * n_chan;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        const long long tb = i / n_chan;
        const int f = (int)(i - tb * n_chan);
        const double s = __ddiv_rn(freq[f], kSpeedOfLight);
        const VisMap m = map_vis(uvw[tb * 3 + 0], uvw[tb * 3 + 1], s, p);
        const long long lim = 1ll << 30;
        const long long cx = m.x0 < -lim ? -lim : (m.x0 > lim ? lim : m.x0);
        const long long cy = m.y0 < -lim ? -lim : (m.y0 > lim ? lim : m.y0);
        int32_t *o = out + i * 6;
        o[0] = (int32_t)cx; o[1] = (int32_t)cy; o[2] = m.qx; o[3] = m.qy; o[4] = 0; o[5] = m.dropped ? 1 : 0;
    }
}

static MapParams make_map_params(const Plan &p) {
    MapParams mp;
    mp.n_grid = p.cfg.grid_size;
    mp.oversample = p.cfg.oversample;
    mp.support = p.S;
    mp.half_so = p.S * p.cfg.oversample / 2;
    mp.ntx = p.ntx;
    mp.cell_size = p.cfg.cell_size;
    mp.key = p.key;
    return mp;
}

static int blocks_for(long long n, int threads, int n_sm) {
    long long b = (n + threads - 1) / threads;
    long long cap = (long long)n_sm * 16;
    if (b > cap) b = cap;
    if (b < 1) b = 1;
    return (int)b;
}

cudaError_t launch_map_debug(const Plan &p, const double *uvw, int n_time, int n_bl, const double *freq,
                             int n_chan, int32_t *out, cudaStream_t s) {
    const long long n_tb = (long long)n_time * n_bl;
    map_debug_kernel<<<blocks_for(n_tb * n_chan, 256, p.n_sm), 256, 0, s>>>(uvw, freq, n_tb, n_chan,
                                                                             make_map_params(p), out);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// Tile tables from the sorted keys (the paper's 'first'/'last' look-up tables, :197).
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) tile_bounds_kernel(const uint32_t *__restrict__ keys, long long n,
                                                           int tile_shift, uint32_t *__restrict__ tile_start,
                                                           uint32_t *__restrict__ tile_end) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        const uint32_t t = keys[i] >> tile_shift;
        if (i == 0 || (keys[i - 1] >> tile_shift) != t) tile_start[t] = (uint32_t)i;
        if (i == n - 1 || (keys[i + 1] >> tile_shift) != t) tile_end[t] = (uint32_t)(i + 1);
    }
}

// chunks per tile: (full chunks << 32) | has_tail, one extra zero element at [n_tiles] so that the
// exclusive scan's last element is the pair of totals.
__global__ void __launch_bounds__(256) tile_chunks_kernel(const uint32_t *__restrict__ tile_start,
                                                           const uint32_t *__restrict__ tile_end, int n_tiles,
                                                           int chunk, unsigned long long *__restrict__ packed,
                                                           Counters *counters) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t > n_tiles) return;
    unsigned long long v = 0;
    if (t < n_tiles) {
        const uint32_t cnt = tile_end[t] - tile_start[t];
        if (cnt) {
            v = ((unsigned long long)(cnt / chunk) << 32) | (unsigned long long)((cnt % chunk) ? 1 : 0);
            atomicAdd(&counters->n_occupied, 1u);
            atomicMax(&counters->max_tile_load, cnt);
        }
    }
    packed[t] = v;
}

__global__ void __launch_bounds__(256) item_fill_kernel(const uint32_t *__restrict__ tile_start,
                                                         const uint32_t *__restrict__ tile_end,
                                                         const unsigned long long *__restrict__ scan, int n_tiles,
                                                         int chunk, TileInfo *__restrict__ info,
                                                         WorkItem *__restrict__ items, Counters *counters) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const unsigned long long totals = scan[n_tiles];
    const uint32_t n_full_total = (uint32_t)(totals >> 32), n_tail_total = (uint32_t)totals;
    if (t == 0) {
        counters->n_full_total = n_full_total;
        counters->n_items = n_full_total + n_tail_total;
        counters->queue_head = 0;
    }
    if (t >= n_tiles) return;
    const uint32_t start = tile_start[t], cnt = tile_end[t] - start;
    const uint32_t nf = cnt / chunk, rem = cnt - nf * chunk;
    const uint32_t full_base = (uint32_t)(scan[t] >> 32), tail_base = (uint32_t)scan[t];
    TileInfo ti;
    ti.count = cnt;
    ti.full_base = full_base;
    ti.n_full = nf;
    ti.tail_item = rem ? n_full_total + tail_base : 0xFFFFFFFFu;
    info[t] = ti;
    for (uint32_t c = 0; c < nf; ++c) {
        WorkItem w;
        w.start = start + c * chunk; w.len = chunk; w.tile = t; w.pad = 0;
        items[full_base + c] = w;
    }
    if (rem) {
        WorkItem w;
        w.start = start + nf * chunk; w.len = rem; w.tile = t; w.pad = 0;
        items[n_full_total + tail_base] = w;
    }
}

cudaError_t sort_temp_bytes(int64_t n, int begin_bit, int end_bit, size_t *bytes) {
    *bytes = 0;
    cub::DoubleBuffer<uint32_t> k(nullptr, nullptr), v(nullptr, nullptr);
    return cub::DeviceRadixSort::SortPairs(nullptr, *bytes, k, v, (long long)n, begin_bit, end_bit, (cudaStream_t)0);
}

cudaError_t scan_temp_bytes(int64_t n, size_t *bytes) {
    *bytes = 0;
    return cub::DeviceScan::ExclusiveSum(nullptr, *bytes, (const unsigned long long *)nullptr,
                                         (unsigned long long *)nullptr, (long long)n, (cudaStream_t)0);
}

#define GR_TRY(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return e_; } while (0)

cudaError_t launch_bin(Plan &p, const double *uvw, int n_time, int n_bl, const double *freq, int n_chan,
                       cudaStream_t s) {
    const long long n_tb = (long long)n_time * n_bl;
    const long long n = n_tb * n_chan;
    GR_TRY(cudaMemsetAsync(p.counters, 0, sizeof(Counters), s));
    // tile_start and tile_end are adjacent: [2][n_tiles]
    GR_TRY(cudaMemsetAsync(p.tile_start, 0, sizeof(uint32_t) * 2 * (size_t)p.n_tiles, s));
    uint32_t *tile_end = p.tile_start + p.n_tiles;
    stage_mark(p, 0, s);
    if (n > 0) {
        map_kernel<<<blocks_for(n, 256, p.n_sm), 256, 0, s>>>(uvw, freq, n_tb, n_chan, make_map_params(p),
                                                                p.keys[0], p.vals[0], p.counters);
        GR_TRY(cudaGetLastError());
        stage_mark(p, 1, s);
        cub::DoubleBuffer<uint32_t> k(p.keys[0], p.keys[1]), v(p.vals[0], p.vals[1]);
        size_t tb = p.cub_temp_bytes;
        GR_TRY(cub::DeviceRadixSort::SortPairs(p.cub_temp, tb, k, v, n, p.key.aux_bits, p.key.total_bits, s));
        p.sorted_sel = k.selector;
        stage_mark(p, 2, s);
        p.n_launches += 3;
        tile_bounds_kernel<<<blocks_for(n, 256, p.n_sm), 256, 0, s>>>(p.keys[p.sorted_sel], n,
                                                                        p.key.tile_shift, p.tile_start, tile_end);
        GR_TRY(cudaGetLastError());
    } else {
        p.sorted_sel = 0;
        stage_mark(p, 1, s);
        stage_mark(p, 2, s);
    }
    const int nt1 = p.n_tiles + 1;
    tile_chunks_kernel<<<(nt1 + 255) / 256, 256, 0, s>>>(p.tile_start, tile_end, p.n_tiles, p.chunk,
                                                           p.tile_chunks, p.counters);
    GR_TRY(cudaGetLastError());
    size_t tb = p.cub_temp_bytes;
    GR_TRY(cub::DeviceScan::ExclusiveSum(p.cub_temp, tb, (const unsigned long long *)p.tile_chunks,
                                         p.tile_chunks_scan, (long long)nt1, s));
    item_fill_kernel<<<(nt1 + 255) / 256, 256, 0, s>>>(p.tile_start, tile_end, p.tile_chunks_scan, p.n_tiles,
                                                         p.chunk, p.tile_info, p.items, p.counters);
    GR_TRY(cudaGetLastError());
    p.n_launches += 3;
    stage_mark(p, 3, s);
    if (p.profiling) p.prof_bin_calls++;
    return cudaSuccess;
}

}  // namespace gridder
