// gridder_bin: map (uvw x freq -> key), stable radix sort, tile tables and work items.
// PAPER.md :181 "calculate which patch", :197 "sorted the visibilities according to the bin",
// "look up tables of the 'first' and 'last' visibilities within each bin", :199 sort on the GPU.
#include <cub/device/device_radix_sort.cuh>
#include <cub/device/device_scan.cuh>
#include <cub/util_type.cuh>

#include <cstring>

#include "gridder_internal.cuh"
#include "map.cuh"

namespace gridder {

// ------------------------------------------------------------------------------------------
// GCF table re-layout, one launch per w-plane: user table K[jy][jx] ([S*O]^2 samples, float or
// float pairs) -> coef[sub = sy*nsub + sx][q = qy*O + qx][a][lane][b], the order the grid kernel's
// lanes read it in (one vector load per lane per column block a).  Lane (rq = lane >> 3,
// c8 = lane & 7) owns taps ty = SPY*sy + rq + 4 b, tx = SPX*sx + c8 + 8 a of sub-patch (sy, sx);
// taps beyond S are zero (the patch is padded to 8 NA nsub x 4 NB nsub cells).
// ------------------------------------------------------------------------------------------
__global__ void relayout_kernel(const float *__restrict__ table, float *__restrict__ coef, int S, int O,
                                int NA, int NB, int nsub, int cplx) {
    const int E = cplx ? 2 : 1;
    const int total = nsub * nsub * O * O * NA * 32 * NB;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < total; i += gridDim.x * blockDim.x) {
        int r = i;
        const int b = r % NB; r /= NB;
        const int lane = r % 32; r /= 32;
        const int a = r % NA; r /= NA;
        const int q = r % (O * O); r /= (O * O);
        const int sub = r;
        const int qy = q / O, qx = q % O;
        const int ty = 4 * NB * (sub / nsub) + (lane >> 3) + 4 * b;
        const int tx = 8 * NA * (sub % nsub) + (lane & 7) + 8 * a;
        // a lane's NB * E floats: contiguous, except 8 floats (complex, NB = 4) = two float4 kept 32 lanes apart
        // ([a][j][lane][4]) so that each of the warp's two 128-bit loads is one contiguous 512-byte run
        size_t o = (size_t)i * E;
        if (NB * E == 8) o = ((((size_t)(sub * O * O + q) * NA + a) * 2 + (b >> 1)) * 32 + lane) * 4 + (b & 1) * 2;
        for (int e = 0; e < E; ++e) {
            float v = 0.f;
            if (ty < S && tx < S) v = table[((size_t)(qy + ty * O) * (S * O) + (qx + tx * O)) * E + e];
            coef[o + e] = v;
        }
    }
}

cudaError_t launch_relayout(const Plan &p, cudaStream_t s) {
    const int O = p.cfg.oversample;
    const int E = p.cfg.kernel_is_complex ? 2 : 1;
    size_t in_off = 0;
    for (int pl = 0; pl < p.cfg.n_wplanes; ++pl) {
        const ClassGeo &g = p.cls[p.plane_slot[pl]];
        const int S = p.support_copy[pl];
        const int total = g.nsub * g.nsub * O * O * g.NA * 32 * g.NB;
        float *out = reinterpret_cast<float *>(reinterpret_cast<char *>(p.coef) + (size_t)p.plane_off256[pl] * 256);
        relayout_kernel<<<(total + 255) / 256, 256, 0, s>>>((const float *)p.cfg.kernel + in_off, out, S, O, g.NA,
                                                             g.NB, g.nsub, p.cfg.kernel_is_complex ? 1 : 0);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        in_off += (size_t)S * O * S * O * E;
    }
    return cudaSuccess;
}

// s[f] = freq[f] / c, once per gridder_bin
__global__ void freq_scale_kernel(const double *__restrict__ freq, int n_chan, double *__restrict__ scale) {
    const int f = blockIdx.x * blockDim.x + threadIdx.x;
    if (f < n_chan) scale[f] = __ddiv_rn(freq[f], kSpeedOfLight);
}

template <bool GENERAL>
__global__ void __launch_bounds__(256) map_kernel(const double *__restrict__ uvw, const double *__restrict__ scale,
                                                   unsigned int n, unsigned int n_chan, const MapParams p,
                                                   uint32_t *__restrict__ keys, void *__restrict__ vals,
                                                   Counters *counters) {
    unsigned int dropped_here = 0;
    unsigned long long taps_here = 0;
    const unsigned int stride = gridDim.x * blockDim.x;
    const uint32_t tmask = (1u << p.key.tlog) - 1u;
    for (unsigned long long ii = blockIdx.x * blockDim.x + threadIdx.x; ii < n; ii += stride) {
        const unsigned int i = (unsigned int)ii;
        const unsigned int tb = i / n_chan;
        const unsigned int f = i - tb * n_chan;
        const double *L = uvw + (size_t)tb * 3;
        const VisMap m = map_vis(L[0], L[1], GENERAL ? L[2] : 0.0, scale[f], p, tb);
        uint32_t key;
        if (m.dropped) {
            dropped_here++;
            key = (uint32_t)(p.drop_slot * p.n_tiles) << p.key.tile_shift;       // tile 0, origin (0,0)
            if (!GENERAL) key |= 1u << (2 * p.key.bits_q);
        } else {
            taps_here += (unsigned long long)(m.S * m.S);
            const uint32_t x0 = (uint32_t)m.x0, y0 = (uint32_t)m.y0;
            const uint32_t tile = (y0 >> p.key.tlog) * (uint32_t)p.ntx + (x0 >> p.key.tlog);
            const uint32_t gtile = p.chans_per_grid ? (f / (uint32_t)p.chans_per_grid) * (uint32_t)p.grid_tiles : 0u;
            const uint32_t vtile = (uint32_t)(p.cls_slot[m.plane] * p.n_tiles) + gtile + tile;
            key = (vtile << p.key.tile_shift) | ((y0 & tmask) << (p.key.aux_bits + p.key.tlog)) |
                  ((x0 & tmask) << p.key.aux_bits);
            if (p.key.plane_bits) key |= (uint32_t)m.plane << p.key.plane_shift;
            if (!GENERAL) key |= ((uint32_t)m.qy << p.key.bits_q) | (uint32_t)m.qx;
        }
        keys[i] = key;
        if (GENERAL) {
            const uint32_t q = (uint32_t)(m.qy * p.oversample + m.qx);
            uint32_t aux = m.dropped ? (1u << 30) : (p.tab_off256[m.plane] + q * p.q_units[m.plane]) | ((q & 63u) << kAuxQShift);
            if (m.conj) aux |= 1u << 31;
            reinterpret_cast<uint2 *>(vals)[i] = make_uint2(i, aux);
        } else {
            reinterpret_cast<uint32_t *>(vals)[i] = i;
        }
    }
    // integer atomics, one per warp (the sums do not depend on the order)
    for (int o = 16; o > 0; o >>= 1) {
        dropped_here += __shfl_xor_sync(0xffffffffu, dropped_here, o);
        taps_here += __shfl_xor_sync(0xffffffffu, taps_here, o);
    }
    if ((threadIdx.x & 31) == 0) {
        if (dropped_here) atomicAdd(&counters->n_dropped, (unsigned long long)dropped_here);
        if (taps_here) atomicAdd(&counters->vis_taps, taps_here);
    }
}

__global__ void __launch_bounds__(256) map_debug_kernel(const double *__restrict__ uvw,
                                                         const double *__restrict__ freq, long long n_tb,
                                                         int n_chan, const MapParams p, int32_t *__restrict__ out) {
    const long long n = n_tb * n_chan;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        const long long tb = i / n_chan;
        const int f = (int)(i - tb * n_chan);
        const double s = __ddiv_rn(freq[f], kSpeedOfLight);
        const VisMap m = map_vis(uvw[tb * 3 + 0], uvw[tb * 3 + 1], uvw[tb * 3 + 2], s, p, (unsigned int)tb);
        int32_t *o = out + i * 6;
        o[0] = m.x0; o[1] = m.y0; o[2] = m.qx; o[3] = m.qy;      // origins are clamped to +-2^30 by the map
        o[4] = m.plane | (m.conj << 8); o[5] = m.dropped ? 1 : 0;
    }
}

MapParams make_map_params(const Plan &p) {
    MapParams mp;
    memset(&mp, 0, sizeof(mp));
    mp.n_grid = p.cfg.grid_size;
    mp.oversample = p.cfg.oversample;
    mp.ntx = p.ntx;
    mp.n_tiles = p.n_tiles_cls;
    mp.grid_tiles = p.n_tiles;
    mp.chans_per_grid = p.n_grids > 1 ? p.chans_per_grid : 0;
    mp.n_planes = p.cfg.n_wplanes;
    mp.general = p.mode != 0;
    mp.is_complex = p.cfg.kernel_is_complex ? 1 : 0;
    mp.drop_slot = 0;
    mp.o_shift = -1;
    for (int b = 0; b < 7; ++b)
        if ((1 << b) == p.cfg.oversample) mp.o_shift = b;
    mp.cell_size = p.cfg.cell_size;
    mp.rcp_cell = 1.0 / p.cfg.cell_size;
    mp.span = (double)p.cfg.grid_size * p.cfg.oversample;
    mp.w_max = p.cfg.w_max;
    mp.fm_chalf = (double)(p.cfg.grid_size / 2) * (double)p.cfg.oversample + 0.5;
    mp.fm_eps = mp.span * 7.1054273576010019e-15;             // 2^-47 N O
    mp.fm_span2 = 2.0 * mp.span;
    mp.fm_half_so = (p.support_copy[0] * p.cfg.oversample) >> 1;
    mp.fm_n_minus_s = p.cfg.grid_size - p.support_copy[0];
    mp.key = p.key;
    for (int i = 0; i < p.cfg.n_wplanes; ++i) {
        mp.support[i] = p.support_copy[i];
        mp.cls_slot[i] = p.plane_slot[i];
        mp.tab_off256[i] = p.plane_off256[i];
        mp.q_units[i] = (uint32_t)(p.cls[p.plane_slot[i]].sub_bytes / 256);
    }
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
                             int n_chan, const int32_t *table_index, int32_t *out, cudaStream_t s) {
    const long long n_tb = (long long)n_time * n_bl;
    MapParams mp = make_map_params(p);
    mp.table_index = table_index;
    map_debug_kernel<<<blocks_for(n_tb * n_chan, 256, p.n_sm), 256, 0, s>>>(uvw, freq, n_tb, n_chan, mp, out);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// Tile tables from the sorted keys (the paper's 'first'/'last' look-up tables, :197), per virtual
// tile = class slot * n_tiles + tile.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) tile_bounds_kernel(const uint32_t *__restrict__ keys, long long n,
                                                           int tile_shift, uint32_t *__restrict__ tile_start,
                                                           uint32_t *__restrict__ tile_end) {
    // four keys per thread (one 16-byte load), the neighbours of the quad with two scalar loads
    const long long n4 = (n + 3) / 4;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n4; q += (long long)gridDim.x * blockDim.x) {
        const long long i0 = 4 * q;
        uint32_t t[6];                                        // tiles of entries i0 - 1 .. i0 + 4 (0xFFFFFFFF: none)
        if (i0 + 4 <= n) {
            const uint4 k = *reinterpret_cast<const uint4 *>(keys + i0);
            t[1] = k.x >> tile_shift; t[2] = k.y >> tile_shift; t[3] = k.z >> tile_shift; t[4] = k.w >> tile_shift;
        } else {
            for (int j = 0; j < 4; ++j) t[1 + j] = i0 + j < n ? keys[i0 + j] >> tile_shift : 0xFFFFFFFFu;
        }
        t[0] = i0 > 0 ? keys[i0 - 1] >> tile_shift : 0xFFFFFFFFu;
        t[5] = i0 + 4 < n ? keys[i0 + 4] >> tile_shift : 0xFFFFFFFFu;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            if (i0 + j >= n) break;
            if (t[j] != t[1 + j]) tile_start[t[1 + j]] = (uint32_t)(i0 + j);
            if (t[2 + j] != t[1 + j]) tile_end[t[1 + j]] = (uint32_t)(i0 + j + 1);
        }
    }
}

// chunks per tile: (full chunks << 32) | has_tail, one extra zero element at [n_vtiles] so that the
// exclusive scan's last element is the pair of totals.
__global__ void __launch_bounds__(256) tile_chunks_kernel(const uint32_t *__restrict__ tile_start,
                                                           const uint32_t *__restrict__ tile_end, int n_vtiles,
                                                           int chunk, unsigned long long *__restrict__ packed,
                                                           Counters *counters) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t > n_vtiles) return;
    unsigned long long v = 0;
    if (t < n_vtiles) {
        const uint32_t cnt = tile_end[t] - tile_start[t];
        if (cnt) {
            v = ((unsigned long long)(cnt / chunk) << 32) | (unsigned long long)((cnt % chunk) ? 1 : 0);
            atomicAdd(&counters->n_occupied, 1u);
            atomicMax(&counters->max_tile_load, cnt);
        }
    }
    packed[t] = v;
}

// Work items of class slot c occupy ids [B_c, B_c + F_c + T_c): its F_c full chunks in tile order,
// then its T_c tails in tile order; B_c = sum over earlier classes.  scan[] is the exclusive scan of
// the packed (full << 32 | tail) counts over the virtual tiles.
__global__ void __launch_bounds__(256) item_fill_kernel(const uint32_t *__restrict__ tile_start,
                                                         const uint32_t *__restrict__ tile_end,
                                                         const unsigned long long *__restrict__ scan, int n_tiles,
                                                         int n_cls, int chunk, TileInfo *__restrict__ info,
                                                         WorkItem *__restrict__ items, Counters *counters, unsigned int max_items) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const int n_vtiles = n_tiles * n_cls;
    if (t == 0) {
        uint32_t base = 0;
        for (int c = 0; c < n_cls; ++c) {
            const unsigned long long lo = scan[(size_t)c * n_tiles], hi = scan[(size_t)(c + 1) * n_tiles];
            const uint32_t nf = (uint32_t)(hi >> 32) - (uint32_t)(lo >> 32), nt = (uint32_t)hi - (uint32_t)lo;
            counters->cls_begin[c] = base;
            base += nf + nt;
            counters->cls_end[c] = base;
        }
        counters->n_items = base;
    }
    if (t >= n_vtiles) return;
    const int c = t / n_tiles;
    uint32_t base = 0;
    for (int k = 0; k < c; ++k) {
        const unsigned long long lo = scan[(size_t)k * n_tiles], hi = scan[(size_t)(k + 1) * n_tiles];
        base += ((uint32_t)(hi >> 32) - (uint32_t)(lo >> 32)) + ((uint32_t)hi - (uint32_t)lo);
    }
    const unsigned long long c_lo = scan[(size_t)c * n_tiles], c_hi = scan[(size_t)(c + 1) * n_tiles];
    const uint32_t cls_full = (uint32_t)(c_hi >> 32) - (uint32_t)(c_lo >> 32);
    const uint32_t start = tile_start[t], cnt = tile_end[t] - start;
    const uint32_t nf = cnt / chunk, rem = cnt - nf * chunk;
    const uint32_t full_base = base + ((uint32_t)(scan[t] >> 32) - (uint32_t)(c_lo >> 32));
    const uint32_t tail_id = base + cls_full + ((uint32_t)scan[t] - (uint32_t)c_lo);
    TileInfo ti;
    ti.count = cnt;
    ti.full_base = full_base;
    ti.n_full = nf;
    ti.tail_item = rem ? tail_id : 0xFFFFFFFFu;
    info[t] = ti;
    GR_CHECK(counters, (unsigned long long)full_base + nf <= max_items && (!rem || tail_id < max_items));
    for (uint32_t k = 0; k < nf; ++k) {
        WorkItem w;
        w.start = start + k * chunk; w.len = chunk; w.tile = t; w.pad = 0;
        items[full_base + k] = w;
    }
    if (rem) {
        WorkItem w;
        w.start = start + nf * chunk; w.len = rem; w.tile = t; w.pad = 0;
        items[tail_id] = w;
    }
}

cudaError_t sort_temp_bytes(int64_t n, int begin_bit, int end_bit, bool wide, size_t *bytes) {
    *bytes = 0;
    cub::DoubleBuffer<uint32_t> k(nullptr, nullptr);
    if (wide) {
        cub::DoubleBuffer<unsigned long long> v(nullptr, nullptr);
        return cub::DeviceRadixSort::SortPairs(nullptr, *bytes, k, v, (long long)n, begin_bit, end_bit, (cudaStream_t)0);
    }
    cub::DoubleBuffer<uint32_t> v(nullptr, nullptr);
    return cub::DeviceRadixSort::SortPairs(nullptr, *bytes, k, v, (long long)n, begin_bit, end_bit, (cudaStream_t)0);
}

cudaError_t scan_temp_bytes(int64_t n, size_t *bytes) {
    *bytes = 0;
    return cub::DeviceScan::ExclusiveSum(nullptr, *bytes, (const unsigned long long *)nullptr,
                                         (unsigned long long *)nullptr, (long long)n, (cudaStream_t)0);
}

#define GR_TRY(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return e_; } while (0)

cudaError_t launch_bin(Plan &p, const double *uvw, int n_time, int n_bl, const double *freq, int n_chan,
                       const int32_t *table_index, cudaStream_t s) {
    const long long n_tb = (long long)n_time * n_bl;
    const long long n = n_tb * n_chan;
    const int n_vtiles = p.n_tiles_cls * p.n_cls;
    GR_TRY(cudaMemsetAsync(p.counters, 0, sizeof(Counters), s));
    // tile_start and tile_end are adjacent: [2][n_vtiles]
    GR_TRY(cudaMemsetAsync(p.tile_start, 0, sizeof(uint32_t) * 2 * (size_t)n_vtiles, s));
    uint32_t *tile_end = p.tile_start + n_vtiles;
    stage_mark(p, 0, s);
    if (n > 0) {
        double *scale = p.freq_scale;
        freq_scale_kernel<<<(n_chan + 255) / 256, 256, 0, s>>>(freq, n_chan, scale);
        GR_TRY(cudaGetLastError());
        bool by_runs = false;          // the sorted list is there already (records of a pre-summed plan)
        p.presum_active = 0;
        p.n_sorted = n;
        if (p.presum && !table_index && presum_fits(p, n_time, n_bl, n_chan)) {
            // pre-summation in input order (presum.cu): flags per visibility, keys per partial record; the
            // RECORDS are what is sorted and gridded.  Inputs that merge too little take the per-visibility path.
            long long n_rec = 0;
            GR_TRY(launch_presum_plan(p, uvw, scale, n_time, n_bl, n_chan, s, &n_rec));
            if (n_rec <= p.ps_cap) {
                stage_mark(p, 1, s);
                cub::DoubleBuffer<uint32_t> k(p.keys[0], p.keys[1]);
                cub::DoubleBuffer<uint32_t> v((uint32_t *)p.vals[0], (uint32_t *)p.vals[1]);
                size_t tb = p.cub_temp_bytes;
                GR_TRY(cub::DeviceRadixSort::SortPairs(p.cub_temp, tb, k, v, n_rec, p.key.aux_bits, p.key.total_bits, s));
                p.sorted_sel = k.selector;
                p.n_launches += 1;
                stage_mark(p, 2, s);
                p.presum_active = 1;
                p.n_sorted = n_rec;
                p.ps_n_time = n_time; p.ps_n_bl = n_bl; p.ps_n_chan = n_chan;
                by_runs = true;          // (skips the per-visibility map and sort below)
                if (n_rec > 0) {
                    tile_bounds_kernel<<<blocks_for(n_rec, 256, p.n_sm), 256, 0, s>>>(p.keys[p.sorted_sel], n_rec,
                                                                                      p.key.tile_shift, p.tile_start, tile_end);
                    GR_TRY(cudaGetLastError());
                }
            } else {
                GR_TRY(cudaMemsetAsync(p.counters, 0, 2 * sizeof(unsigned long long), s));   // counted again below
            }
        }
        if (!by_runs) {
            MapParams mp = make_map_params(p);
            mp.table_index = table_index;
            if (p.mode == 0)
                map_kernel<false><<<blocks_for(n, 256, p.n_sm), 256, 0, s>>>(uvw, scale, (unsigned)n, (unsigned)n_chan, mp,
                                                                              p.keys[0], p.vals[0], p.counters);
            else
                map_kernel<true><<<blocks_for(n, 256, p.n_sm), 256, 0, s>>>(uvw, scale, (unsigned)n, (unsigned)n_chan, mp,
                                                                             p.keys[0], p.vals[0], p.counters);
            GR_TRY(cudaGetLastError());
            stage_mark(p, 1, s);
            cub::DoubleBuffer<uint32_t> k(p.keys[0], p.keys[1]);
            size_t tb = p.cub_temp_bytes;
            if (p.mode == 0) {
                cub::DoubleBuffer<uint32_t> v((uint32_t *)p.vals[0], (uint32_t *)p.vals[1]);
                GR_TRY(cub::DeviceRadixSort::SortPairs(p.cub_temp, tb, k, v, n, p.key.aux_bits, p.key.total_bits, s));
            } else {
                cub::DoubleBuffer<unsigned long long> v((unsigned long long *)p.vals[0], (unsigned long long *)p.vals[1]);
                GR_TRY(cub::DeviceRadixSort::SortPairs(p.cub_temp, tb, k, v, n, p.key.aux_bits, p.key.total_bits, s));
            }
            p.sorted_sel = k.selector;
            stage_mark(p, 2, s);
            p.n_launches += 4;
        }
        if (!by_runs) {
            tile_bounds_kernel<<<blocks_for(n, 256, p.n_sm), 256, 0, s>>>(p.keys[p.sorted_sel], n,
                                                                            p.key.tile_shift, p.tile_start, tile_end);
            GR_TRY(cudaGetLastError());
        }
    } else {
        p.sorted_sel = 0;
        stage_mark(p, 1, s);
        stage_mark(p, 2, s);
    }
    const int nt1 = n_vtiles + 1;
    tile_chunks_kernel<<<(nt1 + 255) / 256, 256, 0, s>>>(p.tile_start, tile_end, n_vtiles, p.chunk,
                                                           p.tile_chunks, p.counters);
    GR_TRY(cudaGetLastError());
    size_t tb = p.cub_temp_bytes;
    GR_TRY(cub::DeviceScan::ExclusiveSum(p.cub_temp, tb, (const unsigned long long *)p.tile_chunks,
                                         p.tile_chunks_scan, (long long)nt1, s));
    item_fill_kernel<<<(nt1 + 255) / 256, 256, 0, s>>>(p.tile_start, tile_end, p.tile_chunks_scan, p.n_tiles_cls,
                                                         p.n_cls, p.chunk, p.tile_info, p.items, p.counters, (unsigned int)p.max_items);
    GR_TRY(cudaGetLastError());
    p.n_launches += 3;
    stage_mark(p, 3, s);
    if (p.profiling) p.prof_bin_calls++;
    return cudaSuccess;
}

}  // namespace gridder
