// PRE-SUMMATION IN INPUT ORDER (fast path: one real table, S <= 16).
//
// Visibilities that fall on the same point of the 1/O sub-cell lattice use identical taps, and gridding is
// linear: sum_i C w_i V_i = C sum_i w_i V_i (Eq. 1 :176).  Where do such
// visibilities sit in MEMORY?  Next to each other: along a baseline the uv point moves ~3e-4 of its length
// per 40 kHz channel and ~7e-5 per second of hour angle, so the neighbouring channels and the integrations
// of ONE baseline mostly share their lattice point (BASELINE.json config 4: 9.1 visibilities per point
// inside a group of 32 channels x 8 integrations of one baseline; config 2, one integration: 2.0).
//
// So the visibilities are never sorted.  They are streamed once, in the order they are stored:
//   gridder_bin   presum_plan_kernel   geometry only: per GROUP (one baseline, 32 consecutive channels, up to 8
//                                      consecutive integrations) the exact map of every visibility, then which
//                                      visibilities share a lattice point -> one FLAG BYTE per visibility and
//                                      one key per partial RECORD
//                 scan + compact       record keys to their final places (group order)
//                 radix sort           of the RECORDS (key, record index) by tile and origin
//   gridder_grid  presum_kernel        warp per group: lane = channel, 8 integrations in registers; visibilities,
//                                      weights and flags are read fully coalesced, once; writes sum of w V per record
//                 grid_kernel          on the sorted records (gathered through the index), then the flush
//
// How a group finds its records (both kernels follow the same rules, the plan kernel from the keys, the
// pre-summation kernel from the flag bytes):
//   * lane = channel (column), rows r = 0..7 = integrations.  A T-RUN is a maximal run of equal keys down a
//     column (the uv point moves on a line, so a lattice point is met once: a run).
//   * a t-run of column f LINKS FORWARD to the t-run of column f + 1 with the same key, if there is one.  Only
//     the first t-run of a key in its column takes part in links (a second one -- possible for adversarial
//     inputs only -- becomes a record of its own), so every t-run has at most one predecessor.
//   * a t-run with no predecessor is a CHAIN HEAD = one record; the record is the sum over its chain of
//     t-runs, added in chain order: a fixed order, so results are bit-identical from run to run.
//   * records of a group are numbered in (column, row) order of their heads.
// Flag byte of visibility (t, b, f), meaningful where a t-run starts (0 elsewhere):
//   bit 0 t-run starts here | bit 1 chain head | bit 2 dropped (off the grid) | bit 3 has a forward link |
//   bits 4-6 row where the linked t-run of column f + 1 starts.
#include <cub/device/device_scan.cuh>

#include "gridder_internal.cuh"
#include "map.cuh"

namespace gridder {

constexpr uint32_t kAbsent = 0xFFFFFFFFu;      // no visibility here (ragged group); never a key (see fast_key)

struct PsGeo {
    uint32_t n_time, n_bl, n_chan;
    uint32_t n_fchunk;          // ceil(n_chan / 32)
    uint32_t rows;              // min(8, n_time): integrations per group
    uint32_t n_tblock;          // ceil(n_time / rows)
    uint32_t n_groups;          // n_tblock * n_bl * n_fchunk; group g = (tb * n_bl + b) * n_fchunk + fc
    uint32_t slots;             // rows * 32: staging slots (most records) of a group
};

__device__ __forceinline__ void group_coords(const PsGeo &g, uint32_t grp, uint32_t &tb, uint32_t &b, uint32_t &fc) {
    fc = grp % g.n_fchunk;
    const uint32_t rb = grp / g.n_fchunk;
    b = rb % g.n_bl;
    tb = rb / g.n_bl;
}

// exclusive prefix of x over the lanes of a warp, and the total
__device__ __forceinline__ uint32_t warp_excl(uint32_t x, int lane, uint32_t &total) {
    uint32_t incl = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    total = __shfl_sync(0xffffffffu, incl, 31);
    return incl - x;
}

template <bool FAST>
__global__ void __launch_bounds__(256) presum_plan_kernel(const double *__restrict__ uvw, const double *__restrict__ scale,
                                                           const PsGeo geo, const MapParams p,
                                                           unsigned char *__restrict__ flags, uint32_t *__restrict__ stage,
                                                           uint32_t *__restrict__ count, Counters *counters) {
    const int lane = threadIdx.x & 31;
    const uint32_t gw = blockIdx.x * 8u + (threadIdx.x >> 5), nw = gridDim.x * 8u;
    const uint32_t dropbit = 1u << (2 * p.key.bits_q);
    FastMap fm;
    if (FAST) fm.init(p);
    unsigned int dropped_here = 0;
    unsigned long long taps_here = 0;

    for (uint32_t grp = gw; grp < geo.n_groups; grp += nw) {
        uint32_t tb, b, fc;
        group_coords(geo, grp, tb, b, fc);
        const uint32_t f = fc * 32u + (uint32_t)lane, t0 = tb * geo.rows;
        const bool col = f < geo.n_chan;
        const double s = col ? scale[f] : 0.0;
        uint32_t key[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            key[r] = kAbsent;
            if (col && (uint32_t)r < geo.rows && t0 + r < geo.n_time) {
                const double *L = uvw + ((size_t)(t0 + r) * geo.n_bl + b) * 3;
                int taps;
                if (FAST) {
                    key[r] = fm.key(__ldg(L), __ldg(L + 1), s, p, taps);
                } else {
                    const VisMap m = map_vis(__ldg(L), __ldg(L + 1), 0.0, s, p);
                    taps = m.dropped ? 0 : m.S * m.S;
                    key[r] = fast_key(m, p);
                }
                if (taps == 0) dropped_here++; else taps_here += (unsigned long long)taps;
            }
        }
        // t-runs, and which of them is the first of its key in the column
        uint32_t th = 0, fo = 0, drop = 0;
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            if (key[r] == kAbsent) continue;
            const bool start = r == 0 || key[r] != key[r - 1];
            if (!start) continue;
            th |= 1u << r;
            if (key[r] & dropbit) { drop |= 1u << r; continue; }
            bool first = true;
#pragma unroll
            for (int r2 = 0; r2 < r; ++r2) first = first && key[r2] != key[r];
            if (first) fo |= 1u << r;
        }
        // forward links into column f + 1 (same warp only: chains do not cross a group)
        uint32_t nfo = __shfl_down_sync(0xffffffffu, fo, 1);
        if (lane == 31) nfo = 0u;
        uint32_t nk[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) nk[r] = __shfl_down_sync(0xffffffffu, key[r], 1);
        uint32_t link = 0;          // 4 bits per row: has a link | the linked row << 1
        uint32_t targets = 0;       // rows of column f + 1 this column links to
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            if (!((fo >> r) & 1u)) continue;
#pragma unroll
            for (int r2 = 0; r2 < 8; ++r2)
                if (((nfo >> r2) & 1u) && nk[r2] == key[r]) {
                    link |= (1u | ((uint32_t)r2 << 1)) << (4 * r);
                    targets |= 1u << r2;
                }
        }
        uint32_t pred = __shfl_up_sync(0xffffffffu, targets, 1);
        if (lane == 0) pred = 0;
        const uint32_t head = th & ~drop & ~pred;
        // records of the group in (column, row) order of their heads
        uint32_t total;
        uint32_t idx = warp_excl((uint32_t)__popc(head), lane, total);
        if (lane == 0) count[grp] = total;
        uint32_t *st = stage + (size_t)grp * geo.slots;
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            if (key[r] == kAbsent) continue;
            const uint32_t bit = 1u << r;
            unsigned char fl = 0;
            if (th & bit)
                fl = (unsigned char)(1u | ((head & bit) ? 2u : 0u) | ((drop & bit) ? 4u : 0u) | (((link >> (4 * r)) & 15u) << 3));
            flags[((size_t)(t0 + r) * geo.n_bl + b) * geo.n_chan + f] = fl;
            if (head & bit) st[idx++] = key[r];
        }
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

// Staged record keys -> their final places (group order); the sort's values are the record indices.
__global__ void __launch_bounds__(256) presum_compact_kernel(const uint32_t *__restrict__ stage,
                                                              const uint32_t *__restrict__ count,
                                                              const uint32_t *__restrict__ base, const PsGeo geo,
                                                              uint32_t *__restrict__ rec_key, uint32_t *__restrict__ rec_idx) {
    const int lane = threadIdx.x & 31;
    const uint32_t nw = gridDim.x * 8u;
    for (uint32_t grp = blockIdx.x * 8u + (threadIdx.x >> 5); grp < geo.n_groups; grp += nw) {
        const uint32_t cnt = count[grp], dst = base[grp];
        const uint32_t *st = stage + (size_t)grp * geo.slots;
        for (uint32_t j = lane; j < cnt; j += 32) {
            rec_key[dst + j] = st[j];
            rec_idx[dst + j] = dst + j;
        }
    }
}

__device__ __forceinline__ float4 ld_stream4(const float4 *p) {
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.L2::256B.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

constexpr int kPsWarps = 4;                          // 33 KB of static shared memory per block
constexpr int kPsWarpF4 = 2 * 8 * 32 + 16;          // slot planes A and B [row][lane], then 256 flag bytes

// gridder_grid, first kernel of a pre-summed plan: rec_sum[record] = sum over the record's chain of w V.
template <bool WEIGHTED>
__global__ void __launch_bounds__(kPsWarps * 32) presum_kernel(const float4 *__restrict__ vis, const float *__restrict__ weight,
                                                               const unsigned char *__restrict__ flags,
                                                               const uint32_t *__restrict__ base, const PsGeo geo,
                                                               float4 *__restrict__ rec_sum) {
    __shared__ float4 smem[kPsWarps * kPsWarpF4];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float4 *slotA = smem + warp * kPsWarpF4, *slotB = slotA + 8 * 32;
    unsigned char *sflag = reinterpret_cast<unsigned char *>(slotB + 8 * 32);
    const uint32_t nw = gridDim.x * (uint32_t)kPsWarps;

    for (uint32_t grp = blockIdx.x * (uint32_t)kPsWarps + warp; grp < geo.n_groups; grp += nw) {
        uint32_t tb, b, fc;
        group_coords(geo, grp, tb, b, fc);
        const uint32_t f = fc * 32u + (uint32_t)lane, t0 = tb * geo.rows;
        const bool col = f < geo.n_chan;
        // everything the group needs is requested at once: 8 rows x (32 B + 4 B + 1 B) per lane
        float4 va[8], vb[8];
        float w[8];
        uint32_t fl[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            va[r] = vb[r] = make_float4(0.f, 0.f, 0.f, 0.f);
            w[r] = 0.f;
            fl[r] = 0u;
            if (col && (uint32_t)r < geo.rows && t0 + r < geo.n_time) {
                const size_t i = ((size_t)(t0 + r) * geo.n_bl + b) * geo.n_chan + f;
                va[r] = ld_stream4(vis + 2 * i);
                vb[r] = ld_stream4(vis + 2 * i + 1);
                w[r] = WEIGHTED ? __ldcs(weight + i) : 1.0f;
                fl[r] = flags[i];
            }
        }
        const uint32_t rbase = base[grp];
        // t-runs: a column's visibilities are added down the rows; a finished run goes to the slot of the row
        // it started in
        float4 xa = make_float4(0.f, 0.f, 0.f, 0.f), xb = xa;
        int start = -1;
        uint32_t head = 0;
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            sflag[r * 32 + lane] = (unsigned char)fl[r];
            if (fl[r] & 1u) {
                if (start >= 0) { slotA[start * 32 + lane] = xa; slotB[start * 32 + lane] = xb; }
                start = r;
                xa = make_float4(w[r] * va[r].x, w[r] * va[r].y, w[r] * va[r].z, w[r] * va[r].w);
                xb = make_float4(w[r] * vb[r].x, w[r] * vb[r].y, w[r] * vb[r].z, w[r] * vb[r].w);
                if (fl[r] & 2u) head |= 1u << r;
            } else {
                xa.x = fmaf(w[r], va[r].x, xa.x); xa.y = fmaf(w[r], va[r].y, xa.y);
                xa.z = fmaf(w[r], va[r].z, xa.z); xa.w = fmaf(w[r], va[r].w, xa.w);
                xb.x = fmaf(w[r], vb[r].x, xb.x); xb.y = fmaf(w[r], vb[r].y, xb.y);
                xb.z = fmaf(w[r], vb[r].z, xb.z); xb.w = fmaf(w[r], vb[r].w, xb.w);
            }
        }
        if (start >= 0) { slotA[start * 32 + lane] = xa; slotB[start * 32 + lane] = xb; }
        __syncwarp();
        // chain heads: walk the chain through the columns, adding the t-run sums in chain order
        uint32_t total;
        uint32_t idx = rbase + warp_excl((uint32_t)__popc(head), lane, total);
        while (head) {
            const int r = __ffs(head) - 1;
            head &= head - 1u;
            float4 sa = slotA[r * 32 + lane], sb = slotB[r * 32 + lane];
            uint32_t cf = sflag[r * 32 + lane];
            int c = lane;
            while (cf & 8u) {
                const int rr = (int)((cf >> 4) & 7u);
                ++c;
                const float4 ta = slotA[rr * 32 + c], tb4 = slotB[rr * 32 + c];
                sa.x += ta.x; sa.y += ta.y; sa.z += ta.z; sa.w += ta.w;
                sb.x += tb4.x; sb.y += tb4.y; sb.z += tb4.z; sb.w += tb4.w;
                cf = sflag[rr * 32 + c];
            }
            rec_sum[2 * (size_t)idx] = sa;
            rec_sum[2 * (size_t)idx + 1] = sb;
            ++idx;
        }
        __syncwarp();           // the slots are reused by the next group
    }
}

#define GR_TRY(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return e_; } while (0)

static PsGeo make_geo(int n_time, int n_bl, int n_chan) {
    PsGeo g;
    g.n_time = (uint32_t)n_time; g.n_bl = (uint32_t)n_bl; g.n_chan = (uint32_t)n_chan;
    g.n_fchunk = (uint32_t)((n_chan + 31) / 32);
    g.rows = (uint32_t)(n_time < 8 ? n_time : 8);
    if (g.rows == 0) g.rows = 1;
    g.n_tblock = (uint32_t)((n_time + (int)g.rows - 1) / (int)g.rows);
    g.n_groups = g.n_tblock * g.n_bl * g.n_fchunk;
    g.slots = g.rows * 32u;
    return g;
}

// Can this input be pre-summed by the plan?  (Host-side, shapes only.)
bool presum_fits(const Plan &p, int n_time, int n_bl, int n_chan) {
    if (!p.presum || n_time <= 0 || n_bl <= 0 || n_chan <= 0) return false;
    const PsGeo g = make_geo(n_time, n_bl, n_chan);
    const unsigned long long ng = (unsigned long long)g.n_tblock * g.n_bl * g.n_fchunk;
    if (ng > (unsigned long long)p.ps_group_cap) return false;
    if (ng * g.slots > (unsigned long long)p.ps_stage_cap) return false;        // staging lives in the record sums
    return true;
}

cudaError_t presum_scan_temp_bytes(int64_t n, size_t *bytes) {
    *bytes = 0;
    return cub::DeviceScan::ExclusiveSum(nullptr, *bytes, (const uint32_t *)nullptr, (uint32_t *)nullptr, (long long)n,
                                         (cudaStream_t)0);
}

// gridder_bin of a pre-summed plan, first half: flags, record keys (compacted into keys[0] / vals[0]) and the
// record count (*n_rec, read back: the stream is synchronised once).
cudaError_t launch_presum_plan(Plan &p, const double *uvw, const double *scale, int n_time, int n_bl, int n_chan,
                               cudaStream_t s, long long *n_rec) {
    const PsGeo geo = make_geo(n_time, n_bl, n_chan);
    const MapParams mp = make_map_params(p);
    uint32_t *stage = reinterpret_cast<uint32_t *>(p.rec_sum);
    const int blocks = (int)min((long long)(geo.n_groups + 7) / 8, (long long)p.n_sm * 64);
    GR_TRY(cudaMemsetAsync(p.ps_count + geo.n_groups, 0, sizeof(uint32_t), s));
    if (mp.o_shift >= 0 && mp.drop_slot == 0)
        presum_plan_kernel<true><<<blocks, 256, 0, s>>>(uvw, scale, geo, mp, p.ps_flags, stage, p.ps_count, p.counters);
    else
        presum_plan_kernel<false><<<blocks, 256, 0, s>>>(uvw, scale, geo, mp, p.ps_flags, stage, p.ps_count, p.counters);
    GR_TRY(cudaGetLastError());
    size_t tb = p.cub_temp_bytes;
    GR_TRY(cub::DeviceScan::ExclusiveSum(p.cub_temp, tb, (const uint32_t *)p.ps_count, p.ps_base,
                                         (long long)geo.n_groups + 1, s));
    unsigned int total = 0;
    GR_TRY(cudaMemcpyAsync(&total, p.ps_base + geo.n_groups, sizeof(unsigned int), cudaMemcpyDeviceToHost, s));
    presum_compact_kernel<<<blocks, 256, 0, s>>>(stage, p.ps_count, p.ps_base, geo, p.keys[0], (uint32_t *)p.vals[0]);
    GR_TRY(cudaGetLastError());
    GR_TRY(cudaStreamSynchronize(s));
    p.n_launches += 3;
    *n_rec = (long long)total;
    return cudaSuccess;
}

// gridder_grid of a pre-summed plan, first kernel.
cudaError_t launch_presum(Plan &p, const float *vis, const float *weight, cudaStream_t s) {
    const PsGeo geo = make_geo(p.ps_n_time, p.ps_n_bl, p.ps_n_chan);
    const int blocks = (int)min((long long)(geo.n_groups + kPsWarps - 1) / kPsWarps, (long long)p.n_sm * 32);
    if (weight)
        presum_kernel<true><<<blocks, kPsWarps * 32, 0, s>>>(reinterpret_cast<const float4 *>(vis), weight, p.ps_flags,
                                                              p.ps_base, geo, p.rec_sum);
    else
        presum_kernel<false><<<blocks, kPsWarps * 32, 0, s>>>(reinterpret_cast<const float4 *>(vis), nullptr, p.ps_flags,
                                                               p.ps_base, geo, p.rec_sum);
    p.n_launches += 1;
    return cudaGetLastError();
}

}  // namespace gridder
