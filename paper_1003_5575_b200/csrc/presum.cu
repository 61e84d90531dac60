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
//   gridder_bin   presum_plan_kernel   geometry only: per GROUP (8 rows x 32 consecutive channels; a row is one
//                                      (integration, baseline)) the exact map of every visibility, then which
//                                      visibilities share a lattice point -> one FLAG BYTE per visibility and
//                                      one key per partial RECORD
//                 scan + compact       record keys to their final places (group order)
//                 radix sort           of the RECORDS (key, slot of the record's sum) by tile and origin
//   gridder_grid  presum_kernel        warp per group: lane = channel, 8 rows in registers; visibilities, weights and
//                                      flags are read fully coalesced, once; writes sum of w V per record
//                 grid_kernel          on the sorted records (gathered through the slot index), then the flush
//
// How a group finds its records (both kernels follow the same rules, the plan kernel from the keys, the
// pre-summation kernel from the flag bytes):
//   * lane = channel (column), rows r = 0..7.  A T-RUN is a maximal run of equal keys down a column (the uv point
//     of a baseline moves on a line with the integration, so a lattice point is met once: a run).
//   * a t-run of column f LINKS FORWARD to the t-run of column f + 1 that holds the same key in one of the run's
//     own rows (the first such row decides).  Runs of one lattice point in neighbouring columns overlap in their
//     rows or are strangers to each other -- then they stay two records, which costs a record, never correctness.
//     A t-run of column f + 1 is linked to at most once (the first claimant in row order), so every t-run has at
//     most one predecessor and chains cannot merge or loop.
//   * a t-run with no predecessor is a CHAIN HEAD = one record; the record is the sum over its chain of
//     t-runs, added in chain order: a fixed order, so results are bit-identical from run to run.
//   * records of a group are numbered in (column, row) order of their heads; record j's sum lives in the group's
//     own visibility slots (slot_index), its staged key at a closed-form offset (stage_offset).
// Flag byte of visibility (t, b, f), meaningful where a t-run starts (0 elsewhere):
//   bit 0 has a forward link | bits 1-3 row where the linked t-run of column f + 1 starts |
//   bit 4 t-run starts here | bit 5 chain head | bit 6 dropped (off the grid).
#include <cub/device/device_scan.cuh>

#include "gridder_internal.cuh"
#include "map.cuh"

namespace gridder {

constexpr uint32_t kFlagLink = 1u, kFlagStart = 16u, kFlagHead = 32u, kFlagDrop = 64u;
constexpr uint32_t kAbsent = 0xFFFFFFFFu;      // no visibility here (ragged group); never a lattice code (map.cuh)

// A group is 8 ROWS x 32 channels; a row is one (integration, baseline).  Rows of a group: rt integrations
// (at most 8, in t-blocks of equal size: make_geo) of each of rb = 8 / rt consecutive baselines, the integrations of
// a baseline next to each other -- so 8 integrations of one baseline when there are that many, 8 baselines when
// there is one integration.
// (Summing visibilities with equal keys is valid whatever rows they come from.)
struct PsGeo {
    uint32_t n_time, n_bl, n_chan;
    uint32_t n_fchunk;          // ceil(n_chan / 32)
    uint32_t rt, rb;            // integrations x baselines per group
    uint32_t n_tblock;          // ceil(n_time / rt)
    uint32_t n_bgroup;          // ceil(n_bl / rb)
    uint32_t n_groups;          // n_tblock * n_bgroup * n_fchunk; group g = (tb * n_bgroup + bg) * n_fchunk + fc
    uint32_t n_vis;             // n_time * n_bl * n_chan
    float rcp_fchunk, rcp_bgroup;       // 1 / n_fchunk, 1 / n_bgroup (div_small)
};

// x / d for x < 2^24 (group indices: a plan has fewer than 2^32 / 256 groups... and 2^24 bounds them for every
// accepted shape, see presum_fits): float reciprocal and one correction step instead of a 32-bit division.
__device__ __forceinline__ uint32_t div_small(uint32_t x, uint32_t d, float rcp) {
    uint32_t q = (uint32_t)((float)x * rcp);
    if (q * d > x) --q;
    if ((q + 1u) * d <= x) ++q;
    return q;
}

__device__ __forceinline__ void group_coords(const PsGeo &g, uint32_t grp, uint32_t &t0, uint32_t &b0, uint32_t &f0) {
    const uint32_t rest = div_small(grp, g.n_fchunk, g.rcp_fchunk), fc = grp - rest * g.n_fchunk;
    const uint32_t tb = div_small(rest, g.n_bgroup, g.rcp_bgroup);
    f0 = fc * 32u;
    b0 = (rest - tb * g.n_bgroup) * g.rb;
    t0 = tb * g.rt;
}

// Row r of a group: integration t0 + rt of baseline b0 + rb.  RT > 0: the integrations per group are known at
// compile time (1, 2, 4 or 8: all 8 rows in use), RT == 0: any (geo.rt).
template <int RT>
__device__ __forceinline__ void row_of(const PsGeo &g, int r, uint32_t &rt, uint32_t &rb) {
    if constexpr (RT > 0) {
        rt = (uint32_t)(r % RT);
        rb = (uint32_t)(r / RT);
    } else {
        rb = (uint32_t)r / g.rt;
        rt = (uint32_t)r - rb * g.rt;
    }
}
// (all element indices fit 32 bits: a plan holds fewer than 2^32 visibilities)
template <int RT>
__device__ __forceinline__ bool row_index(const PsGeo &g, int r, uint32_t t0, uint32_t b0, uint32_t &row) {
    uint32_t rt, rb;
    row_of<RT>(g, r, rt, rb);
    row = (t0 + rt) * g.n_bl + (b0 + rb);
    return (RT > 0 || rb < g.rb) && t0 + rt < g.n_time && b0 + rb < g.n_bl;
}
// The same relative to the group's first row: row = row0 + row_step<RT>(g, r), valid iff row_ok<RT>(g, r, nrt, nrb)
// with nrt = n_time - t0, nrb = n_bl - b0 -- a multiply-add and a compare or two of uniform values per row.
template <int RT>
__device__ __forceinline__ uint32_t row_step(const PsGeo &g, int r) {
    uint32_t rt, rb;
    row_of<RT>(g, r, rt, rb);
    return rt * g.n_bl + rb;
}
template <int RT>
__device__ __forceinline__ bool row_ok(const PsGeo &g, int r, uint32_t nrt, uint32_t nrb) {
    uint32_t rt, rb;
    row_of<RT>(g, r, rt, rb);
    return (RT > 0 || rb < g.rb) && rt < nrt && rb < nrb;
}

// Where the sum of record j of a group lives in ps_sum (an array as large as the visibility array): in the group's
// own visibility slots, filled row segment by row segment -- so a group's records are contiguous runs of up to 32,
// their places need no scan over the groups, and no two groups share a slot.  (A group has at most as many records
// as visibilities.)
__device__ __forceinline__ uint32_t slot_index(const PsGeo &g, uint32_t t0, uint32_t b0, uint32_t f0, uint32_t j) {
    const uint32_t ncols = min(32u, g.n_chan - f0), nrt = min(g.rt, g.n_time - t0);
    // j < 256, ncols <= 32, k < 8, nrt <= 8: multiply-shift divisions are exact (j * 32 < 2^16)
    const uint32_t k = (j * ((65536u + ncols - 1u) / ncols)) >> 16, c = j - k * ncols;          // k-th valid row of the group
    const uint32_t kb = (k * ((65536u + nrt - 1u) / nrt)) >> 16, kt = k - kb * nrt;
    return ((t0 + kt) * g.n_bl + (b0 + kb)) * g.n_chan + f0 + c;
}

// Where a group's staged record keys start: the number of visibilities of the groups before it (group order: t-block,
// baseline group, channel chunk) -- a closed form, so the staging area is exactly as large as the visibility count
// however ragged the groups are.  (A group has at most as many records as visibilities.)
__device__ __forceinline__ uint32_t stage_offset(const PsGeo &g, uint32_t t0, uint32_t b0, uint32_t f0) {
    const uint32_t nrt = min(g.rt, g.n_time - t0), nrb = min(g.rb, g.n_bl - b0);
    return (t0 * g.n_bl + nrt * b0) * g.n_chan + nrt * nrb * f0;
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

template <bool FAST, int RT>
__global__ void __launch_bounds__(256, 5) presum_plan_kernel(const double *__restrict__ uvw, const double *__restrict__ scale,
                                                           const PsGeo geo, const MapParams p,
                                                           unsigned char *__restrict__ flags, uint32_t *__restrict__ stage,
                                                           uint32_t *__restrict__ count, Counters *counters) {
    const int lane = threadIdx.x & 31;
    const uint32_t gw = blockIdx.x * 8u + (threadIdx.x >> 5), nw = gridDim.x * 8u;
    FastMap2 fm;
    if (FAST) fm.init(p);
    unsigned int dropped_here = 0, mapped_here = 0;

    const uint32_t g_end_all = geo.n_groups;
    for (uint32_t grp = gw; grp < geo.n_groups; grp += nw) {
        uint32_t t0, b0, f0;
        group_coords(geo, grp, t0, b0, f0);
        const uint32_t f = f0 + (uint32_t)lane;
        const bool col = f < geo.n_chan;
        const double s = col ? scale[f] : 0.0;
        const double ks = FAST ? fm.chan_scale(s) : 0.0;
        // (gridder_bin_channels: the channel's grid is part of the tile id, so nothing merges across grids)
        const uint32_t gtile = p.chans_per_grid ? (f / (uint32_t)p.chans_per_grid) * (uint32_t)p.grid_tiles : 0u;
        uint32_t key[8];                 // lattice codes (FastMap2::lat): equal exactly when the sort keys are
        uint32_t valid = 0, slow = 0;
        const uint32_t row0 = t0 * geo.n_bl + b0, nrt = geo.n_time - t0, nrb = geo.n_bl - b0;
        const double *L0 = uvw + (size_t)row0 * 3;
        if (grp + nw < g_end_all && lane < 8) {         // the uvw rows of the group this warp takes next: into L1 now
            uint32_t nt0, nb0, nf0, nrow;
            group_coords(geo, grp + nw, nt0, nb0, nf0);
            if (row_index<RT>(geo, lane, nt0, nb0, nrow)) asm volatile("prefetch.global.L1 [%0];" :: "l"(uvw + (size_t)nrow * 3));
        }
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            key[r] = kAbsent;
            if (row_ok<RT>(geo, r, nrt, nrb) && col) {
                const double *L = L0 + (size_t)row_step<RT>(geo, r) * 3;
                key[r] = FAST ? fm.lat(__ldg(L), __ldg(L + 1), ks) : FastMap2::kUndecided;
                if (key[r] == FastMap2::kUndecided) slow |= 1u << r;
                valid |= 1u << r;
            }
        }
        while (slow) {              // the screen did not decide (about one visibility in 10^8), or no fast mapper
            const int r = __ffs(slow) - 1;
            slow &= slow - 1u;
            uint32_t row;
            row_index<RT>(geo, r, t0, b0, row);
            const double *L = uvw + (size_t)row * 3;
            const uint32_t k = FastMap2::slow_lat(__ldg(L), __ldg(L + 1), s, p);
#pragma unroll
            for (int rr = 0; rr < 8; ++rr)
                if (rr == r) key[rr] = k;
        }
        // t-runs (bit r of th: a run starts in row r), dropped visibilities, rows whose key equals the next column's
        uint32_t th = 0, dropv = 0, eq = 0;
        // (a chain stays inside one output grid: gridder_bin_channels)
        const uint32_t next_gtile = __shfl_down_sync(0xffffffffu, gtile, 1);       // (every lane takes part)
        const bool same_grid = lane < 31 && next_gtile == gtile;
#pragma unroll
        for (int r = 0; r < 8; ++r) {          // (branch-free: the masks are cut to the valid rows afterwards)
            const uint32_t nk = __shfl_down_sync(0xffffffffu, key[r], 1);
            th |= (uint32_t)(r == 0 || key[r] != key[r - 1]) << r;
            dropv |= (uint32_t)(key[r] == FastMap2::kDropped) << r;
            eq |= (uint32_t)(nk == key[r]) << r;
        }
        th &= valid;
        eq &= same_grid ? valid : 0u;
        const uint32_t drop = th & dropv;                   // dropped runs
        mapped_here += (unsigned)__popc(valid);
        dropped_here += (unsigned)__popc(dropv);
        // forward links: a run links to the run of the next column that holds the same key in one of the run's
        // own rows (runs of a lattice point in neighbouring columns overlap in their rows, or they are strangers:
        // then they stay two records, which is only a record more).  A target is taken once.
        // The flag bytes of the 8 rows are assembled in two words, byte r % 4 of word r / 4.
        const uint32_t nth = __shfl_down_sync(0xffffffffu, th, 1);
        uint32_t w_lo = 0, w_hi = 0;
        uint32_t targets = 0;       // rows of column f + 1 this column links to
        for (uint32_t m = th & ~drop; m; m &= m - 1u) {
            const int r = __ffs(m) - 1;
            const uint32_t later = th & ~((2u << r) - 1u);                    // starts of the later runs
            const uint32_t rows = ((later ? (later & (0u - later)) : 256u) - 1u) & ~((1u << r) - 1u);
            const uint32_t hit = eq & rows;
            if (!hit) continue;
            const int rs = __ffs(hit) - 1;
            const int h = 31 - __clz(nth & ((2u << rs) - 1u));                // start of the neighbour's run through row rs
            if ((targets >> h) & 1u) continue;
            targets |= 1u << h;
            const uint32_t nib = (kFlagLink | ((uint32_t)h << 1)) << (8 * (r & 3));
            if (r < 4) w_lo |= nib; else w_hi |= nib;
        }
        uint32_t pred = __shfl_up_sync(0xffffffffu, targets, 1);
        if (lane == 0) pred = 0;
        const uint32_t head = th & ~drop & ~pred;
        // bit k of a 4-bit mask to bit 8 k: the shifted copies of x in x * 0x204081 do not overlap
        w_lo |= (((th & 15u) * 0x204081u) & 0x01010101u) * kFlagStart | (((head & 15u) * 0x204081u) & 0x01010101u) * kFlagHead |
                (((drop & 15u) * 0x204081u) & 0x01010101u) * kFlagDrop;
        w_hi |= (((th >> 4) * 0x204081u) & 0x01010101u) * kFlagStart | (((head >> 4) * 0x204081u) & 0x01010101u) * kFlagHead |
                (((drop >> 4) * 0x204081u) & 0x01010101u) * kFlagDrop;
        // records of the group in (column, row) order of their heads
        uint32_t total;
        uint32_t idx = warp_excl((uint32_t)__popc(head), lane, total);
        if (lane == 0) count[grp] = total;
        uint32_t *st = stage + stage_offset(geo, t0, b0, f0);
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const uint32_t bit = 1u << r;
            if (valid & bit) {
                const uint32_t i = (row0 + row_step<RT>(geo, r)) * geo.n_chan + f;
                GR_CHECK(counters, i < geo.n_vis);
                flags[i] = (unsigned char)((r < 4 ? w_lo : w_hi) >> (8 * (r & 3)));
            }
        }
        // the sort keys of the records: only the heads need one (a ninth of the visibilities in config 4)
        for (uint32_t m = head; m; m &= m - 1u) {
            const int r = __ffs(m) - 1;
            uint32_t c = key[0];
#pragma unroll
            for (int rr = 1; rr < 8; ++rr)
                if (rr == r) c = key[rr];
            GR_CHECK(counters, (size_t)(st - stage) + idx < geo.n_vis);
            st[idx++] = FastMap2::key_of(c, p, gtile);
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        dropped_here += __shfl_xor_sync(0xffffffffu, dropped_here, o);
        mapped_here += __shfl_xor_sync(0xffffffffu, mapped_here, o);
    }
    if (lane == 0) {      // (fast path: one table, every gridded visibility has S^2 taps)
        if (dropped_here) atomicAdd(&counters->n_dropped, (unsigned long long)dropped_here);
        const unsigned long long taps = (unsigned long long)(mapped_here - dropped_here) * (unsigned)(p.support[0] * p.support[0]);
        if (taps) atomicAdd(&counters->vis_taps, taps);
    }
}

// Staged record keys -> their final places (group order).  The sort's values name the record's sum (slot_index).
__global__ void __launch_bounds__(256) presum_compact_kernel(const uint32_t *__restrict__ stage,
                                                              const uint32_t *__restrict__ count,
                                                              const uint32_t *__restrict__ base, const PsGeo geo,
                                                              uint32_t *__restrict__ rec_key, uint32_t *__restrict__ rec_idx,
                                                              Counters *counters) {
    const int lane = threadIdx.x & 31;
    const uint32_t nw = gridDim.x * 8u;
    for (uint32_t grp = blockIdx.x * 8u + (threadIdx.x >> 5); grp < geo.n_groups; grp += nw) {
        const uint32_t cnt = count[grp], dst = base[grp];
        uint32_t t0, b0, f0;
        group_coords(geo, grp, t0, b0, f0);
        const uint32_t *st = stage + stage_offset(geo, t0, b0, f0);
        for (uint32_t j = lane; j < cnt; j += 32) {
            GR_CHECK(counters, dst + j < geo.n_vis && slot_index(geo, t0, b0, f0, j) < geo.n_vis && (size_t)(st - stage) + j < geo.n_vis);
            rec_key[dst + j] = st[j];
            rec_idx[dst + j] = slot_index(geo, t0, b0, f0, j);
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

__device__ __forceinline__ void prefetch_l2(const void *p) { asm volatile("prefetch.global.L2 [%0];" :: "l"(p)); }

// gridder_grid, first kernel of a pre-summed plan: ps_sum[slot_index(group, j)] = sum over the chain of record j
// of the group of w V.
template <bool WEIGHTED, int RT>
__global__ void __launch_bounds__(kPsWarps * 32) presum_kernel(const float4 *__restrict__ vis, const float *__restrict__ weight,
                                                               const unsigned char *__restrict__ flags, const PsGeo geo,
                                                               float4 *__restrict__ rec_sum, Counters *counters) {
    __shared__ float4 smem[kPsWarps * kPsWarpF4];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float4 *slotA = smem + warp * kPsWarpF4, *slotB = slotA + 8 * 32;
    unsigned char *sflag = reinterpret_cast<unsigned char *>(slotB + 8 * 32);
    const uint32_t nw = gridDim.x * (uint32_t)kPsWarps;
    // this lane's share of the prefetch of the warp's NEXT group: row pr, 128-byte lines pl and pl + 4 of the
    // row's 1 KB of visibilities; lanes 0-7 also the row's weights, lanes 8-15 its flags
    const int pr = lane & 7;
    const uint32_t pl = (uint32_t)lane >> 3;

    for (uint32_t grp = blockIdx.x * (uint32_t)kPsWarps + warp; grp < geo.n_groups; grp += nw) {
        uint32_t t0, b0, f0;
        group_coords(geo, grp, t0, b0, f0);
        if (grp + nw < geo.n_groups) {
            // The group this warp takes next is asked into L2 now: a warp has one group's loads in flight at a
            // time, which alone does not keep HBM busy
            uint32_t nt0, nb0, nf0;
            group_coords(geo, grp + nw, nt0, nb0, nf0);
            uint32_t row;
            if (row_index<RT>(geo, pr, nt0, nb0, row)) {
                const size_t i0 = (size_t)(row * geo.n_chan + nf0);
                const uint32_t nf = min(32u, geo.n_chan - nf0);
                if (pl * 4u < nf) prefetch_l2(vis + 2 * (i0 + pl * 4u));
                if ((pl + 4u) * 4u < nf) prefetch_l2(vis + 2 * (i0 + (pl + 4u) * 4u));
                if (pl == 0 && WEIGHTED) prefetch_l2(weight + i0);
                if (pl == 1) prefetch_l2(flags + i0);
            }
        }
        const uint32_t f = f0 + (uint32_t)lane;
        const bool col = f < geo.n_chan;
        // everything the group needs is requested at once: 8 rows x (32 B + 4 B + 1 B) per lane
        const uint32_t row0 = t0 * geo.n_bl + b0, nrt = geo.n_time - t0, nrb = geo.n_bl - b0;
        float4 va[8], vb[8];
        float w[8];
        uint32_t fl[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            va[r] = vb[r] = make_float4(0.f, 0.f, 0.f, 0.f);
            w[r] = 0.f;
            fl[r] = 0u;
            if (row_ok<RT>(geo, r, nrt, nrb) && col) {
                const size_t i = (size_t)((row0 + row_step<RT>(geo, r)) * geo.n_chan + f);
                GR_CHECK(counters, i < geo.n_vis);
                va[r] = ld_stream4(vis + 2 * i);
                vb[r] = ld_stream4(vis + 2 * i + 1);
                w[r] = WEIGHTED ? __ldcs(weight + i) : 1.0f;
                fl[r] = flags[i];
            }
        }
        // t-runs: a column's visibilities are added down the rows; a finished run goes to the slot of the row
        // it started in
        float4 xa = make_float4(0.f, 0.f, 0.f, 0.f), xb = xa;
        int start = -1;
        uint32_t head = 0;
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            sflag[r * 32 + lane] = (unsigned char)fl[r];
            if (fl[r] & kFlagStart) {
                if (start >= 0) { slotA[start * 32 + lane] = xa; slotB[start * 32 + lane] = xb; }
                start = r;
                xa = make_float4(w[r] * va[r].x, w[r] * va[r].y, w[r] * va[r].z, w[r] * va[r].w);
                xb = make_float4(w[r] * vb[r].x, w[r] * vb[r].y, w[r] * vb[r].z, w[r] * vb[r].w);
                if (fl[r] & kFlagHead) head |= 1u << r;
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
        uint32_t j = warp_excl((uint32_t)__popc(head), lane, total);       // records in (column, row) order of their heads
        while (head) {
            const int r = __ffs(head) - 1;
            head &= head - 1u;
            float4 sa = slotA[r * 32 + lane], sb = slotB[r * 32 + lane];
            uint32_t cf = sflag[r * 32 + lane];
            int c = lane;
            while (cf & kFlagLink) {
                const int rr = (int)((cf >> 1) & 7u);
                ++c;
                GR_CHECK(counters, c < 32);
                const float4 ta = slotA[rr * 32 + c], tb4 = slotB[rr * 32 + c];
                sa.x += ta.x; sa.y += ta.y; sa.z += ta.z; sa.w += ta.w;
                sb.x += tb4.x; sb.y += tb4.y; sb.z += tb4.z; sb.w += tb4.w;
                cf = sflag[rr * 32 + c];
            }
            const size_t idx = (size_t)slot_index(geo, t0, b0, f0, j++);
            GR_CHECK(counters, idx < geo.n_vis && j <= total);
            rec_sum[2 * idx] = sa;
            rec_sum[2 * idx + 1] = sb;
        }
        __syncwarp();           // the slots are reused by the next group
    }
}

// gridder_map_presum: the keys of FastMap2, decoded (test interface)
__global__ void __launch_bounds__(256) map_presum_debug_kernel(const double *__restrict__ uvw, const double *__restrict__ freq,
                                                                long long n_tb, int n_chan, const MapParams p,
                                                                int32_t *__restrict__ out) {
    FastMap2 fm;
    fm.init(p);
    const long long n = n_tb * n_chan;
    const uint32_t tmask = (1u << p.key.tlog) - 1u, qmask = (1u << p.key.bits_q) - 1u;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const long long tb = i / n_chan;
        const double s = __ddiv_rn(freq[(int)(i - tb * n_chan)], kSpeedOfLight);
        uint32_t c = fm.lat(uvw[tb * 3], uvw[tb * 3 + 1], fm.chan_scale(s));
        if (c == FastMap2::kUndecided) c = FastMap2::slow_lat(uvw[tb * 3], uvw[tb * 3 + 1], s, p);
        const uint32_t key = c == FastMap2::kDropped ? 0u : FastMap2::key_of(c, p);
        int32_t *o = out + i * 6;
        if (c == FastMap2::kDropped) {
            o[0] = o[1] = o[2] = o[3] = o[4] = 0; o[5] = 1;
        } else {
            const uint32_t tile = key >> p.key.tile_shift;
            o[0] = (int32_t)(((tile % (uint32_t)p.ntx) << p.key.tlog) | ((key >> p.key.aux_bits) & tmask));
            o[1] = (int32_t)(((tile / (uint32_t)p.ntx) << p.key.tlog) | ((key >> (p.key.aux_bits + p.key.tlog)) & tmask));
            o[2] = (int32_t)(key & qmask);
            o[3] = (int32_t)((key >> p.key.bits_q) & qmask);
            o[4] = 0; o[5] = 0;
        }
    }
}

cudaError_t launch_map_presum_debug(const Plan &p, const double *uvw, int n_time, int n_bl, const double *freq, int n_chan,
                                    int32_t *out, cudaStream_t s) {
    const MapParams mp = make_map_params(p);
    if (p.mode != 0 || mp.o_shift < 0) return cudaErrorNotSupported;
    const long long n_tb = (long long)n_time * n_bl, n = n_tb * n_chan;
    long long blocks = (n + 255) / 256;
    if (blocks > (long long)p.n_sm * 16) blocks = (long long)p.n_sm * 16;
    map_presum_debug_kernel<<<(int)(blocks < 1 ? 1 : blocks), 256, 0, s>>>(uvw, freq, n_tb, n_chan, mp, out);
    return cudaGetLastError();
}

#define GR_TRY(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) return e_; } while (0)

static PsGeo make_geo(int n_time, int n_bl, int n_chan) {
    PsGeo g;
    g.n_time = (uint32_t)n_time; g.n_bl = (uint32_t)n_bl; g.n_chan = (uint32_t)n_chan;
    g.n_fchunk = (uint32_t)((n_chan + 31) / 32);
    // integrations per group: at most 8, in t-blocks of equal size (9 integrations: 5 + 4, not 8 + 1)
    const uint32_t blocks = ((uint32_t)(n_time > 0 ? n_time : 1) + 7u) / 8u;
    g.rt = ((uint32_t)(n_time > 0 ? n_time : 1) + blocks - 1) / blocks;
    g.rb = 8u / g.rt;
    g.n_tblock = ((uint32_t)n_time + g.rt - 1) / g.rt;
    g.n_bgroup = ((uint32_t)n_bl + g.rb - 1) / g.rb;
    g.n_groups = g.n_tblock * g.n_bgroup * g.n_fchunk;
    g.n_vis = g.n_time * g.n_bl * g.n_chan;
    g.rcp_fchunk = 1.0f / (float)g.n_fchunk;
    g.rcp_bgroup = 1.0f / (float)g.n_bgroup;
    return g;
}

// Can this input be pre-summed by the plan?  (Host-side, shapes only: the plan has room for max_vis / 8 + 1024
// groups, i.e. for groups of 8 visibilities and more on average.)
bool presum_fits(const Plan &p, int n_time, int n_bl, int n_chan) {
    if (!p.presum || n_time <= 0 || n_bl <= 0 || n_chan <= 0) return false;
    const PsGeo g = make_geo(n_time, n_bl, n_chan);
    const unsigned long long ng = (unsigned long long)g.n_tblock * g.n_bgroup * g.n_fchunk;
    if (ng > (unsigned long long)p.ps_group_cap || ng >= (1ull << 24)) return false;      // (2^24: div_small)
    return true;
}

cudaError_t presum_scan_temp_bytes(int64_t n, size_t *bytes) {
    *bytes = 0;
    return cub::DeviceScan::ExclusiveSum(nullptr, *bytes, (const uint32_t *)nullptr, (uint32_t *)nullptr, (long long)n,
                                         (cudaStream_t)0);
}

// gridder_bin of a pre-summed plan, first half: flags, record keys (compacted into keys[0] / vals[0]) and the
// record count (*n_rec, read back: the host waits once, for the count; the compaction is still running then).
cudaError_t launch_presum_plan(Plan &p, const double *uvw, const double *scale, int n_time, int n_bl, int n_chan,
                               cudaStream_t s, long long *n_rec) {
    const PsGeo geo = make_geo(n_time, n_bl, n_chan);
    const MapParams mp = make_map_params(p);
    // staging: the sort's second key buffer, which nothing uses before the sort
    uint32_t *stage = p.keys[1];
    const int blocks = (int)min((long long)(geo.n_groups + 7) / 8, (long long)p.n_sm * 64);
    GR_TRY(cudaMemsetAsync(p.ps_count + geo.n_groups, 0, sizeof(uint32_t), s));
    const bool fast = mp.o_shift >= 0 && mp.drop_slot == 0;
#define PS_PLAN(F, R) presum_plan_kernel<F, R><<<blocks, 256, 0, s>>>(uvw, scale, geo, mp, p.ps_flags, stage, p.ps_count, p.counters)
    switch (fast ? (int)geo.rt : -1) {
        case 8: PS_PLAN(true, 8); break;
        case 4: PS_PLAN(true, 4); break;
        case 2: PS_PLAN(true, 2); break;
        case 1: PS_PLAN(true, 1); break;
        case -1: PS_PLAN(false, 0); break;
        default: PS_PLAN(true, 0); break;
    }
#undef PS_PLAN
    GR_TRY(cudaGetLastError());
    size_t tb = p.cub_temp_bytes;
    GR_TRY(cub::DeviceScan::ExclusiveSum(p.cub_temp, tb, (const uint32_t *)p.ps_count, p.ps_base,
                                         (long long)geo.n_groups + 1, s));
    // the record count goes to the host as soon as the scan is done; the host waits for THAT (an event), not for the
    // compaction enqueued behind it, so the sort is enqueued while the compaction still runs and the GPU never idles
    unsigned int total = 0;
    if (!p.count_ev) GR_TRY(cudaEventCreateWithFlags(&p.count_ev, cudaEventDisableTiming));
    GR_TRY(cudaMemcpyAsync(&total, p.ps_base + geo.n_groups, sizeof(unsigned int), cudaMemcpyDeviceToHost, s));
    GR_TRY(cudaEventRecord(p.count_ev, s));
    presum_compact_kernel<<<blocks, 256, 0, s>>>(stage, p.ps_count, p.ps_base, geo, p.keys[0], (uint32_t *)p.vals[0], p.counters);
    GR_TRY(cudaGetLastError());
    GR_TRY(cudaEventSynchronize(p.count_ev));
    p.n_launches += 3;
    *n_rec = (long long)total;
    return cudaSuccess;
}

// gridder_grid of a pre-summed plan, first kernel.
cudaError_t launch_presum(Plan &p, const float *vis, const float *weight, cudaStream_t s) {
    const PsGeo geo = make_geo(p.ps_n_time, p.ps_n_bl, p.ps_n_chan);
    const int blocks = (int)min((long long)(geo.n_groups + kPsWarps - 1) / kPsWarps, (long long)p.n_sm * 32);
    const float4 *v4 = reinterpret_cast<const float4 *>(vis);
#define PS_SUM(W, R) presum_kernel<W, R><<<blocks, kPsWarps * 32, 0, s>>>(v4, weight, p.ps_flags, geo, p.ps_sum, p.counters)
    if (weight) {
        switch (geo.rt) {
            case 8: PS_SUM(true, 8); break;
            case 1: PS_SUM(true, 1); break;
            default: PS_SUM(true, 0); break;
        }
    } else {
        switch (geo.rt) {
            case 8: PS_SUM(false, 8); break;
            case 1: PS_SUM(false, 1); break;
            default: PS_SUM(false, 0); break;
        }
    }
#undef PS_SUM
    p.n_launches += 1;
    return cudaGetLastError();
}

}  // namespace gridder
