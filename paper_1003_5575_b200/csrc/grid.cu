// gridder_grid: the gridding kernel (FP32 FMA, registers + shared memory) and the deterministic flush.
//
// Grid kernel.  PAPER.md :197-199 gathers per pixel from 9 bins; here the work
// is turned round so that every lane does useful FMAs on every visibility:
//   * a work item is <= K consecutive entries of one uv tile's sorted list; ONE WARP owns it;
//   * the warp keeps the item's (T + SP - 1)^2-cell region (tile + halo) in shared memory;
//   * for the current patch origin the SP x SP patch lives in REGISTERS, NA*NB cells (x 4 pol
//     complex = 8 floats) per lane; entries are sorted by origin, so the patch is exchanged with
//     the shared region only when the origin changes ("fold");
//   * per entry a lane does two broadcast LDS.128 of the staged visibility, NA vector loads of its
//     taps of the GCF sub-table and 4*NA*NB packed FFMA2 (fma.rn.f32x2; 8*NA*NB for a complex table);
//   * a warp runs ONE software pipeline over the whole stream of its work items: keys three
//     batches ahead, visibilities (cp.async, 128-bit) two ahead, weighting and record staging one
//     ahead, so the start of an item costs no exposed memory latency;
//   * no atomics on data anywhere: every region cell has one owner lane, every work item its own
//     partial region in HBM (the only atomic is the integer work-queue counter).
// Flush kernel: each grid cell sums, in FP64 and in a fixed (class, tile row, tile column, chunk)
// order, the partial regions that cover it, and writes the complex64 grid once.
#include <climits>

#include "gridder_internal.cuh"

namespace gridder {

// MODE 0: one real table with S <= 16, resident in shared memory, 32-bit (key, index) entries.
// MODE 1: real tables read from global memory (any number of planes, sub-patches), wide entries.
// MODE 2: complex tables (w-planes), conjugated for w < 0, read from global memory, wide entries.
// MODE 3: as MODE 0, but the table lives in TENSOR MEMORY: lane l of every warp reads its NA*NB taps of
//         sub-table q with one tcgen05.ld (32 lanes x 32 bit x NA*NB columns at column q*NA*NB), which
//         takes the taps off the shared-memory return path -- the path this kernel is bound by.
// NSUB == 2: an entry covers 2 x 2 register patches (supports 17..32).  Sub-patch (sy, sx) of a work item is
//         gridded as a VIRTUAL work item of its own (same entries, its quarter of the table, its own
//         tile + halo region, anchored 16 (sx, sy) cells up the grid), so the region stays 19 x 19.
constexpr int kSentinel = -(1 << 20);   // origin of the record that ends a work item
constexpr int kForce = INT_MIN;         // never an origin: forces a fold at the next record

template <int NA, int NB, int NSUB, int TLOG, int MODE>
struct Geo {
    static constexpr bool CPLX = MODE == 2;
    static constexpr bool GEN = MODE == 1 || MODE == 2;
    static constexpr bool TMEM = MODE == 3;
    static constexpr int SPX = 8 * NA, SPY = 4 * NB;           // register patch
    static constexpr int T = 1 << TLOG;
    static constexpr int RW = T + SPX - 1, RH = T + SPY - 1;   // region = tile + halo of ONE register patch
    static constexpr int VSHIFT = NSUB > 1 ? 2 : 0;            // log2 of the virtual items per work item
    static constexpr int CELLS = RW * RH;                      // a work item's partial region in HBM
    // Fast path (entries of an item come in (y0, x0) order): the warp keeps only SPY rows of the region in shared
    // memory, as a ring -- a patch covers SPY rows, and a row below the current origin's can get nothing more, so
    // it is written to the item's partial and its slot reused as the origin moves up.  11.8 instead of 16.9 KB per
    // warp at T = 8: 12 warps per SM instead of 10.  (The general path sorts by w-plane first: whole region.)
    static constexpr bool CIRC = !GEN;
    static constexpr int RHB = CIRC ? SPY : RH;                // region rows held in shared memory
    static constexpr int CELLS_B = RW * RHB;
    static constexpr int VF4 = 2;                              // float4 per staged visibility
    static constexpr int SLOT_F4 = VF4 + 1;                    // + (table offset of the NEXT record, origin)
    static constexpr int PIPE = GEN ? 3 : 2;                   // records in flight in the consumer (taps fetched PIPE - 1 ahead)
    static constexpr int SLOTS = GEN ? 40 : 36;                // 32 records + sentinel / pads (PIPE) + look-ahead (PIPE)
    static constexpr int NBINS = GEN ? 32 : 16;                // bins of a carried run: sub-cell offsets (x conjugate)
    static constexpr int SLOTS_BINS = SLOTS + NBINS;           // ... + the records a carried run's bins may add
    static constexpr int RAW_F4 = 32 * 2 + 8;                  // cp.async landing: 32 x {a, b}, 32 weights
    static constexpr int BINS_F4 = 2 * NBINS + (GEN ? NBINS / 4 : 0);   // per-run bins (kernels with p.bins): [bin][2] float4
                                                               // (+ general path: the table offset of each bin)
    __host__ __device__ static constexpr int warp_f4(bool bins) {
        return 2 * CELLS_B + 2 * (bins ? SLOTS_BINS : SLOTS) * SLOT_F4 + RAW_F4 + (bins ? BINS_F4 : 0);
    }
    static constexpr int SUB_BYTES = NA * NB * 32 * (CPLX ? 8 : 4);   // one (plane, sub-patch, q) sub-table
};

__device__ __forceinline__ void stg_stream(float4 *p, const float4 &v) {
    asm volatile("st.global.L1::no_allocate.v4.f32 [%0], {%1,%2,%3,%4};"
                 :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

__device__ __forceinline__ void cp_async_16(void *dst_smem, const void *src, bool pred) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(dst_smem);
    const int n = pred ? 16 : 0;                      // 0 source bytes: the destination is zero-filled
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(d), "l"(src), "r"(n) : "memory");
}

__device__ __forceinline__ void cp_async_4(void *dst_smem, const void *src, bool pred) {
    const uint32_t d = (uint32_t)__cvta_generic_to_shared(dst_smem);
    const int n = pred ? 4 : 0;
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4, %2;" :: "r"(d), "l"(src), "r"(n) : "memory");
}

__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// ---- the per-warp stream of batches ---------------------------------------------------------------
// A batch is <= 32 consecutive entries of one work item.  bits: count (0..32) | last batch of its
// item << 6 | end of stream << 7 | batch index inside the item << 8.
struct Desc {
    int bits;
    unsigned item;
    __device__ __forceinline__ int cnt() const { return bits & 63; }
    __device__ __forceinline__ bool last() const { return bits & 64; }
    __device__ __forceinline__ bool end() const { return bits & 128; }
    __device__ __forceinline__ int bidx() const { return bits >> 8; }
};

constexpr int kClaim = 1;       // work items claimed per queue access (one: the end of the kernel is balanced to an item;
                                // 4 at a time left up to four items of imbalance: config 4 grid kernel 6.59 -> 6.42 ms)

struct Producer {
    WorkItem grp, nxt;                   // lane l: descriptor l of the current / the next claimed group
    unsigned grp_base, nxt_base;
    int grp_cnt, nxt_cnt, grp_pos;
    unsigned it_start, it_len, it_off, it_id;
    unsigned item_begin, item_end;       // this launch's (patch class's) range of the work-item table
    unsigned v_end;                      // virtual items of the launch (work items << vshift)
    int vshift;
    bool ended;

    __device__ __forceinline__ void claim(const GridParams &p, int lane) {
        unsigned b = 0;
        if (lane == 0) b = atomicAdd(&p.counters->queue_head[p.cls], (unsigned)kClaim);
        b = __shfl_sync(0xffffffffu, b, 0);
        nxt_base = b;                    // virtual item ids, relative to the class
        nxt_cnt = nxt_base < v_end ? (int)min((unsigned)kClaim, v_end - nxt_base) : 0;
        WorkItem w;
        w.start = w.len = w.tile = w.pad = 0;
        if (lane < nxt_cnt) w = p.items[item_begin + ((nxt_base + lane) >> vshift)];
        nxt = w;
    }

    __device__ __forceinline__ void init(const GridParams &p, int lane, int vshift_) {
        ended = false;
        it_len = it_off = it_start = it_id = 0;
        item_begin = p.counters->cls_begin[p.cls];
        item_end = p.counters->cls_end[p.cls];
        vshift = vshift_;
        v_end = (item_end - item_begin) << vshift;
        claim(p, lane);
        grp = nxt; grp_base = nxt_base; grp_cnt = nxt_cnt; grp_pos = 0;
        if (grp_cnt > 0) claim(p, lane); else ended = true;
    }

    // Descriptor of the next batch of this warp's stream and the position of its first entry.
    __device__ __forceinline__ Desc next(const GridParams &p, int lane, unsigned &start) {
        Desc d;
        d.bits = 128; d.item = 0; start = 0;
        if (ended) return d;
        if (it_off >= it_len) {
            if (grp_pos >= grp_cnt) {
                grp = nxt; grp_base = nxt_base; grp_cnt = nxt_cnt; grp_pos = 0;
                if (grp_cnt == 0) { ended = true; return d; }
                claim(p, lane);
            }
            it_start = __shfl_sync(0xffffffffu, grp.start, grp_pos);
            it_len = __shfl_sync(0xffffffffu, grp.len, grp_pos);
            it_id = grp_base + grp_pos;
            ++grp_pos;
            it_off = 0;
        }
        const unsigned left = it_len - it_off;
        d.bits = (int)min(32u, left) | (left <= 32u ? 64 : 0) | (int)((it_off >> 5) << 8);
        d.item = it_id;
        start = it_start + it_off;
        it_off += 32;
        return d;
    }
};

// One sorted entry as the grid kernel sees it.
struct Entry {
    uint32_t key, idx, aux;
};

template <bool GEN>
__device__ __forceinline__ Entry load_entry(const GridParams &p, unsigned e, bool valid) {
    Entry k;
    k.key = k.idx = k.aux = 0u;
    if (valid) {
        GR_CHECK(p.counters, e < p.n_sorted);
        k.key = __ldg(p.keys + e);
        if (GEN) {
            const uint2 v = __ldg(reinterpret_cast<const uint2 *>(p.vals) + e);
            k.idx = v.x;
            k.aux = v.y;
        } else {
            k.idx = p.vals ? __ldg(reinterpret_cast<const uint32_t *>(p.vals) + e) : e;     // null: records, in place
        }
    }
    return k;
}

// Starts the copies of one batch: lane's visibility goes to raw[lane] and raw[32 + lane], its weight to
// the float array behind.  A lane past the end of the batch, or a dropped visibility, gets zeros.
template <bool GEN>
__device__ __forceinline__ void issue_vis(const GridParams &p, float4 *raw, int lane, const Entry k, bool valid) {
    const bool dropped = GEN ? ((k.aux >> 30) & 1u) : ((k.key >> (2 * p.key.bits_q)) & 1u);
    const bool live = valid && !dropped;
    GR_CHECK(p.counters, !live || k.idx < p.n_src);
    const float4 *src = p.vis + 2 * (size_t)(live ? k.idx : 0u);
    cp_async_16(raw + lane, src, live);                // two planes of 32 float4: conflict-free to read back
    cp_async_16(raw + 32 + lane, src + 1, live);
    if (p.weight) cp_async_4(reinterpret_cast<float *>(raw + 64) + lane, p.weight + (live ? k.idx : 0u), live);
    cp_async_commit();
}

// Moves a landed batch from the raw buffer into one half of the record ring in the consumer's format:
// the weighted visibility (VF4 float4) and (table byte offset, region offset of the patch origin).
//
// MERGING.  Entries of a batch with the same patch origin AND the same table offset use identical taps,
// and gridding is linear: sum_i C w_i V_i = C sum_i w_i V_i.  Such entries are therefore summed here
// (8 additions each) and gridded once (256 FMAs each saved): the group's first lane adds the others in
// ascending lane order -- a fixed order, so results stay bit-identical from run to run -- and the
// surviving records are compacted to the front of the ring.  Exact up to FP32 rounding order, valid
// because the table is a function of (plane, sub-cell offset) only.  Neighbouring channels of a
// baseline and the many baselines through one dense cell make this 2.5x (config 2) to 3.4x (config 4)
// fewer records.  p.merge == 0 keeps every entry.
//
// Returns the number of records written.  The last batch of an item is followed by a sentinel record
// with a negative origin, which makes the consumer fold the last patch into the region; an odd count
// is padded with a record that adds nothing.
template <int NA, int NB, int NSUB, int TLOG, int MODE>
__device__ __forceinline__ int stage_write(const GridParams &p, const float4 *raw, float4 *half, int lane,
                                           const Desc d, const Entry k) {
    using G = Geo<NA, NB, NSUB, TLOG, MODE>;
    const int cnt = d.cnt();
    const uint32_t tmask = (1u << TLOG) - 1u;
    uint32_t x0l, y0l;
    int coff;
    if (G::GEN) {
        x0l = k.key & tmask;
        y0l = (k.key >> TLOG) & tmask;
        coff = (int)((k.aux & kAuxOffMask) << 8);          // table offset in 256-byte units
        if (G::CPLX) coff |= (int)(k.aux >> 31);           // bit 0: use the conjugate table (w < 0)
    } else {
        const uint32_t qmask = (1u << (2 * p.key.bits_q)) - 1u;
        x0l = (k.key >> p.key.aux_bits) & tmask;
        y0l = (k.key >> (p.key.aux_bits + TLOG)) & tmask;
        coff = (int)((k.key & qmask) * (uint32_t)(G::TMEM ? NA * NB : G::SUB_BYTES));   // bytes, or TMEM columns
    }
    // origin inside the tile: offset into the region, or (ring of rows) row << 8 | column
    const int poff = G::CIRC ? (int)((y0l << 8) | x0l) : (int)(y0l * G::RW + x0l);
    const bool valid = lane < cnt;
    const float4 ra = raw[lane], rb = raw[32 + lane];
    const float w = p.weight ? reinterpret_cast<const float *>(raw + 64)[lane] : 1.0f;
    const float o[8] = {ra.x * w, ra.y * w, ra.z * w, ra.w * w, rb.x * w, rb.y * w, rb.z * w, rb.w * w};
    float sum[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) sum[i] = o[i];

    // groups of equal (origin, table offset); lanes past the end are groups of their own
    bool keep = valid;
    if (p.merge) {
        const unsigned long long gkey =
            valid ? (((unsigned long long)(uint32_t)poff << 32) | (uint32_t)coff) : (0xFFFFFFFF00000000ull | (uint32_t)lane);
        const unsigned grp = __match_any_sync(0xffffffffu, gkey);
        keep = valid && (__ffs(grp) - 1 == lane);
        unsigned rest = keep ? (grp & ~(1u << lane)) : 0u;
        while (__any_sync(0xffffffffu, rest != 0u)) {
            const int src = rest ? __ffs(rest) - 1 : lane;
            const bool add = rest != 0u;
            rest &= rest - 1u;
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                const float t = __shfl_sync(0xffffffffu, o[i], src);
                if (add) sum[i] += t;
            }
        }
    }
    // compaction: record r of the ring is the r-th kept lane
    const unsigned kept = __ballot_sync(0xffffffffu, keep);
    const int n_rec = __popc(kept);
    const int slot_id = __popc(kept & ((1u << lane) - 1u));
    const unsigned above = kept & ~((2u << lane) - 1u);             // kept lanes after this one
    int next_coff = __shfl_sync(0xffffffffu, coff, above ? __ffs(above) - 1 : lane);
    if (!above) next_coff = 0;
    const int last_poff = __shfl_sync(0xffffffffu, poff, 31 - __clz(kept | 1u));
    GR_CHECK(p.counters, n_rec + G::PIPE <= G::SLOTS);
    if (keep) {
        // slot r carries the table offset of record r + 1 (the consumer loads taps one record ahead)
        // and the origin of record r; every slot also carries its own table offset (slot 0's is used)
        float4 *slot = half + slot_id * G::SLOT_F4;
        slot[0] = make_float4(sum[0], sum[1], sum[2], sum[3]);
        slot[1] = make_float4(sum[4], sum[5], sum[6], sum[7]);
        slot[G::VF4] = make_float4(__int_as_float(next_coff), __int_as_float(poff), __int_as_float(coff), 0.f);
    }
    if (lane < G::PIPE) {    // sentinel + pads (last batch of an item) or pads (count not a multiple of PIPE)
        float4 *s2 = half + (n_rec + lane) * G::SLOT_F4;
#pragma unroll
        for (int i = 0; i < G::VF4; ++i) s2[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        s2[G::VF4] = make_float4(__int_as_float(0), __int_as_float(d.last() ? kSentinel : last_poff), __int_as_float(0), 0.f);
    }
    return n_rec;
}

// stage_write with PER-ORIGIN BINS carried from batch to batch (O^2 <= 16, merging on).  A hot origin
// has hundreds of entries but only O^2 different sets of taps (x 2 with conjugated w-planes); merging inside a
// batch of 32 still leaves up to that many records per batch.  Here the records of the batch's LAST run -- entries
// of one origin (general path: one origin of one plane; the sort puts them next to each other) -- are not handed to
// the consumer: they go to bins in shared memory (lane-distinct after the batch merge: no two lanes touch a bin),
// the next batches add to them while the run lasts, and when it ends the non-empty bins become its records, in bin
// order, ahead of the batch's own records -- the sorted order, so results stay bit-identical from run to run.
// Every (item, plane, origin, offset) is then gridded exactly once.  The last batch of an item carries nothing over.
template <int NA, int NB, int NSUB, int TLOG, int MODE>
__device__ __forceinline__ int stage_write_bins(const GridParams &p, const float4 *raw, float4 *half, int lane,
                                                const Desc d, const Entry k, float4 *bins, int &bin_org, int &bin_poff,
                                                unsigned &bin_occ) {
    using G = Geo<NA, NB, NSUB, TLOG, MODE>;
    const int cnt = d.cnt();
    const uint32_t tmask = (1u << TLOG) - 1u;
    int poff, org, bin, coff;           // region offset of the origin | identity of the run | bin of the run | table offset
    if (G::GEN) {
        const uint32_t x0l = k.key & tmask, y0l = (k.key >> TLOG) & tmask;
        poff = (int)(y0l * G::RW + x0l);
        org = (int)(k.key & ((1u << p.key.tile_shift) - 1u));                  // plane | y0l | x0l
        bin = (int)(((k.aux >> kAuxQShift) & 15u) | ((k.aux >> 31) << 4));      // offset, conjugate
        coff = (int)((k.aux & kAuxOffMask) << 8) | (int)(k.aux >> 31);
    } else {
        const uint32_t qmask = (1u << (2 * p.key.bits_q)) - 1u;
        const uint32_t x0l = (k.key >> p.key.aux_bits) & tmask, y0l = (k.key >> (p.key.aux_bits + TLOG)) & tmask;
        poff = (int)((y0l << 8) | x0l);
        org = poff;
        bin = (int)(k.key & qmask);
        coff = bin * (G::TMEM ? NA * NB : G::SUB_BYTES);
    }
    int *bin_coff = reinterpret_cast<int *>(bins + 2 * G::NBINS);             // (general path) table offset of a bin
    const bool valid = lane < cnt;
    const float4 ra = raw[lane], rb = raw[32 + lane];
    const float w = p.weight ? reinterpret_cast<const float *>(raw + 64)[lane] : 1.0f;
    const float o[8] = {ra.x * w, ra.y * w, ra.z * w, ra.w * w, rb.x * w, rb.y * w, rb.z * w, rb.w * w};
    float sum[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) sum[i] = o[i];
    // merge inside the batch (as stage_write)
    const unsigned gkey = valid ? (((unsigned)org << 5) | (unsigned)bin) : (0xF0000000u | (unsigned)lane);
    const unsigned grp = __match_any_sync(0xffffffffu, gkey);
    bool keep = valid && (__ffs(grp) - 1 == lane);
    unsigned rest = keep ? (grp & ~(1u << lane)) : 0u;
    while (__any_sync(0xffffffffu, rest != 0u)) {
        const int src = rest ? __ffs(rest) - 1 : lane;
        const bool add = rest != 0u;
        rest &= rest - 1u;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const float t = __shfl_sync(0xffffffffu, o[i], src);
            if (add) sum[i] += t;
        }
    }
    // (a) records of the carried run join its bins
    const bool to_old = keep && org == bin_org;
    if (to_old) {
        float4 a = bins[2 * bin], b = bins[2 * bin + 1];
        a.x += sum[0]; a.y += sum[1]; a.z += sum[2]; a.w += sum[3];
        b.x += sum[4]; b.y += sum[5]; b.z += sum[6]; b.w += sum[7];
        bins[2 * bin] = a; bins[2 * bin + 1] = b;
        if (G::GEN) bin_coff[bin] = coff;
    }
    bin_occ |= __reduce_or_sync(0xffffffffu, to_old ? (1u << bin) : 0u);
    keep = keep && !to_old;
    // (b) does the carried run end here, and which run is carried on?
    const int tail_org = __shfl_sync(0xffffffffu, org, cnt - 1);
    const int tail_poff = __shfl_sync(0xffffffffu, poff, cnt - 1);
    const bool carry = !d.last();                              // the last batch of an item hands everything over
    const bool flush_bins = bin_org >= 0 && (!carry || tail_org != bin_org);
    const bool to_new = keep && carry && org == tail_org && tail_org != bin_org;
    const bool emit = keep && !to_new;
    // (c) the ring: first the finished run's bins in bin order, then the batch's own records
    const unsigned occ = flush_bins ? bin_occ : 0u;
    const int n_bin = __popc(occ);
    const unsigned kept = __ballot_sync(0xffffffffu, emit);
    const int n_rec = n_bin + __popc(kept);
    GR_CHECK(p.counters, n_rec + G::PIPE <= G::SLOTS_BINS);
    const int first_kept_coff = kept ? __shfl_sync(0xffffffffu, coff, __ffs(kept) - 1) : 0;
    __syncwarp();
    if (lane < G::NBINS && ((occ >> lane) & 1u)) {
        const unsigned higher = occ & ~((2u << lane) - 1u);
        const int hb = higher ? __ffs(higher) - 1 : 0;
        const int cstride = G::TMEM ? NA * NB : G::SUB_BYTES;
        const int next_coff = higher ? (G::GEN ? bin_coff[hb] : hb * cstride) : first_kept_coff;
        float4 *slot = half + __popc(occ & ((1u << lane) - 1u)) * G::SLOT_F4;
        slot[0] = bins[2 * lane];
        slot[1] = bins[2 * lane + 1];
        slot[G::VF4] = make_float4(__int_as_float(next_coff), __int_as_float(bin_poff),
                                   __int_as_float(G::GEN ? bin_coff[lane] : lane * cstride), 0.f);
        bins[2 * lane] = make_float4(0.f, 0.f, 0.f, 0.f);
        bins[2 * lane + 1] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    const unsigned above = kept & ~((2u << lane) - 1u);             // emitted lanes after this one
    int next_coff = __shfl_sync(0xffffffffu, coff, above ? __ffs(above) - 1 : lane);
    if (!above) next_coff = 0;
    int last_poff = kept ? __shfl_sync(0xffffffffu, poff, 31 - __clz(kept | 1u)) : bin_poff;
    if (emit) {
        float4 *slot = half + (n_bin + __popc(kept & ((1u << lane) - 1u))) * G::SLOT_F4;
        slot[0] = make_float4(sum[0], sum[1], sum[2], sum[3]);
        slot[1] = make_float4(sum[4], sum[5], sum[6], sum[7]);
        slot[G::VF4] = make_float4(__int_as_float(next_coff), __int_as_float(poff), __int_as_float(coff), 0.f);
    }
    if (lane < G::PIPE) {    // sentinel + pads (last batch of an item) or pads (count not a multiple of PIPE)
        float4 *s2 = half + (n_rec + lane) * G::SLOT_F4;
#pragma unroll
        for (int i = 0; i < G::VF4; ++i) s2[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        s2[G::VF4] = make_float4(__int_as_float(0), __int_as_float(d.last() ? kSentinel : last_poff), __int_as_float(0), 0.f);
    }
    if (flush_bins) { bin_org = -1; bin_occ = 0; }
    __syncwarp();
    // (d) the batch's last run moves into the (now empty) bins
    if (to_new) {
        bins[2 * bin] = make_float4(sum[0], sum[1], sum[2], sum[3]);
        bins[2 * bin + 1] = make_float4(sum[4], sum[5], sum[6], sum[7]);
        if (G::GEN) bin_coff[bin] = coff;
    }
    const unsigned moved = __reduce_or_sync(0xffffffffu, to_new ? (1u << bin) : 0u);
    if (moved) { bin_org = tail_org; bin_poff = tail_poff; bin_occ = moved; }
    return n_rec;
}

// One staged record in registers: the weighted visibility (broadcast loads) and this lane's taps.
template <int NA, int NB, int MODE>
struct RecRegs {
    static constexpr bool CPLX = MODE == 2;
    static constexpr int VF4 = 2;
    static constexpr int CF = NB * (CPLX ? 2 : 1);            // floats per column block
    float4 v[VF4];
    uint32_t sgn;                                             // MODE 2: sign bit of s (s = -1: conjugate table)
    float c[NA][CF];
    // MODE 0: `coef_lane` is the shared-space address of this lane's taps of sub-table 0 (the table
    // sits at the start of dynamic shared memory), else a global pointer.
    __device__ __forceinline__ void fetch(const float4 *slot, int coff, const char *coef_lane) {
#pragma unroll
        for (int i = 0; i < VF4; ++i) v[i] = slot[i];
        fetch_taps(coff, coef_lane);
    }
    // the two halves of the weighted visibility from two places (the per-origin bins are kept as planes)
    __device__ __forceinline__ void fetch2(const float4 *lo, const float4 *hi, int coff, const char *coef_lane) {
        v[0] = *lo;
        v[1] = *hi;
        fetch_taps(coff, coef_lane);
    }
    __device__ __forceinline__ void fetch_taps(int coff, const char *coef_lane) {
        if (MODE == 2) {
            sgn = (uint32_t)coff << 31;
            coff &= ~1;
        }
        if (MODE == 3) {                                       // tensor memory: one load for all NA*NB taps
            const uint32_t ta = (uint32_t)(uintptr_t)coef_lane + (uint32_t)coff;
            if (NA * NB == 8) {
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                             : "=f"(c[0][0]), "=f"(c[0][1]), "=f"(c[0][2]), "=f"(c[0][3]),
                               "=f"(c[NA - 1][0]), "=f"(c[NA - 1][1]), "=f"(c[NA - 1][2]), "=f"(c[NA - 1][3]) : "r"(ta));
            } else {
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0,%1}, [%2];" : "=f"(c[0][0]), "=f"(c[0][1]) : "r"(ta));
            }
            return;
        }
        const char *cp = coef_lane + coff;
#pragma unroll
        for (int a = 0; a < NA; ++a) {
            const char *ca = cp + a * 32 * CF * (int)sizeof(float);
            if (MODE == 0) {                                   // shared memory, explicit state space
                const uint32_t sa = (uint32_t)(uintptr_t)ca;
                if (CF == 4) {
                    asm("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];"
                        : "=f"(c[a][0]), "=f"(c[a][1]), "=f"(c[a][2]), "=f"(c[a][3]) : "r"(sa));
                } else {
                    asm("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(c[a][0]), "=f"(c[a][1]) : "r"(sa));
                }
            } else {                                           // global memory through L1
                // (CF == 8: the two float4 of a lane are 512 bytes apart, [j][lane][4], so that each warp load is one
                // contiguous 512-byte run -- bin.cu relayout_kernel)
#pragma unroll
                for (int j = 0; j < CF / 4; ++j) {
                    const float4 t = __ldg(reinterpret_cast<const float4 *>(ca) + j * 32);
                    c[a][4 * j] = t.x; c[a][4 * j + 1] = t.y; c[a][4 * j + 2] = t.z; c[a][4 * j + 3] = t.w;
                }
                if (CF == 2) {
                    const float2 t = __ldg(reinterpret_cast<const float2 *>(ca));
                    c[a][0] = t.x; c[a][1] = t.y;
                }
            }
        }
    }
    // MODE 3: the taps are usable only after this (it waits for the warp's outstanding tcgen05.ld);
    // the registers go through the statement so that no use is scheduled above it.
    __device__ __forceinline__ void wait() {
        if (MODE == 3) {
            if (NA * NB == 8) {
                asm volatile("tcgen05.wait::ld.sync.aligned;"
                             : "+f"(c[0][0]), "+f"(c[0][1]), "+f"(c[0][2]), "+f"(c[0][3]),
                               "+f"(c[NA - 1][0]), "+f"(c[NA - 1][1]), "+f"(c[NA - 1][2]), "+f"(c[NA - 1][3]));
            } else {
                asm volatile("tcgen05.wait::ld.sync.aligned;" : "+f"(c[0][0]), "+f"(c[0][1]));
            }
        }
    }
};

// Two-level accumulation: the register patch holds a short FP32 chain (one run
// of equal patch origins, at most fold_batches*32 entries); it is then ADDED to the shared region and
// cleared.  A long single chain is not good enough: neighbouring channels of one baseline give
// nearly equal terms, whose rounding errors do not cancel (measured 1.2e-5 relative at 2048 terms).
template <int NA, int NB, int RW, bool CIRC>
__device__ __forceinline__ void fold_patch(float4 *regA, float4 *regB, int cur, int lane, float (&acc)[NA][NB][8],
                                           Counters *ck) {
    __syncwarp();       // a cell changes owner lane from one origin to the next
    constexpr int SPY = 4 * NB, CB = RW * (CIRC ? SPY : 1);     // (CB: plane stride is passed by the caller via regB)
    (void)CB;
    const int rq = lane >> 3, c8 = lane & 7;
    const int y0 = CIRC ? (cur >> 8) : 0, xo = CIRC ? (cur & 255) + c8 : cur + rq * RW + c8;
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const int o = CIRC ? ((y0 + rq + 4 * b) & (SPY - 1)) * RW + xo + 8 * a : xo + 4 * b * RW + 8 * a;
            GR_CHECK(ck, o >= 0 && o < (int)(regB - regA) && (!CIRC || xo + 8 * a < RW));
            float4 x = regA[o], y = regB[o];
            x.x += acc[a][b][0]; x.y += acc[a][b][1]; x.z += acc[a][b][2]; x.w += acc[a][b][3];
            y.x += acc[a][b][4]; y.y += acc[a][b][5]; y.z += acc[a][b][6]; y.w += acc[a][b][7];
            regA[o] = x; regB[o] = y;
#pragma unroll
            for (int k = 0; k < 8; ++k) acc[a][b][k] = 0.f;
        }
}

// Ring of region rows: rows [from, to) of the item's region are complete -- to the item's partial, slots cleared.
template <int RW, int SPY, int CELLS>
__device__ __forceinline__ void flush_rows(float4 *regA, float4 *regB, float4 *dst, int from, int to, int lane, Counters *ck) {
    __syncwarp();
    GR_CHECK(ck, from >= 0 && from <= to && to * RW <= CELLS);
    for (int y = from; y < to; ++y) {
        if (lane < RW) {
            const int o = (y & (SPY - 1)) * RW + lane;
            stg_stream(dst + y * RW + lane, regA[o]);
            stg_stream(dst + CELLS + y * RW + lane, regB[o]);
            regA[o] = make_float4(0.f, 0.f, 0.f, 0.f);
            regB[o] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
    }
    __syncwarp();
}

// (d0, d1) += c * (v0, v1), each product-sum rounded once (two independent IEEE FMAs in one instruction).
__device__ __forceinline__ void ffma2(float &d0, float &d1, float c, float v0, float v1) {
    unsigned long long d, a, b;
    asm("mov.b64 %0, {%1,%2};" : "=l"(d) : "f"(d0), "f"(d1));
    asm("mov.b64 %0, {%1,%2};" : "=l"(a) : "f"(c), "f"(c));
    asm("mov.b64 %0, {%1,%2};" : "=l"(b) : "f"(v0), "f"(v1));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(d) : "l"(a), "l"(b));
    asm("mov.b64 {%0,%1}, %2;" : "=f"(d0), "=f"(d1) : "l"(d));
}

// `cmp` is the origin the patch was last matched against (kForce forces a fold at the next record, used
// to bound the chain length); `cur` is the origin the registers really belong to (-1: none).
// `rows_done` (ring of rows only): region rows already written to the item's partial `dst`.
template <int NA, int NB, int RW, int CELLS, int MODE>
__device__ __forceinline__ void consume(const RecRegs<NA, NB, MODE> &R, const int poff, int &cur, int &cmp,
                                        float4 *regA, float4 *regB, int lane, float (&acc)[NA][NB][8],
                                        int &rows_done, float4 *dst, Counters *ck) {
    constexpr bool CIRC = MODE == 0 || MODE == 3;
    if (poff != cmp) {                                      // warp-uniform
        if (cur >= 0) fold_patch<NA, NB, RW, CIRC>(regA, regB, cur, lane, acc, ck);
        if (CIRC && poff >= 0 && (poff >> 8) > rows_done) {     // the origin moved up: the rows below it are complete
            flush_rows<RW, 4 * NB, CELLS>(regA, regB, dst, rows_done, poff >> 8, lane, ck);
            rows_done = poff >> 8;
        }
        cur = cmp = poff;
    }
    // Packed FP32 pairs (Blackwell fma.rn.f32x2 -> FFMA2 with the tap as a scalar broadcast operand): one
    // instruction updates (re, im) of one polarisation of one cell, halving the issue slots of the loop.
    if (MODE == 2) {
        // (re, im) += cr (v.re, v.im) + ci (-s v.im, s v.re), s = -1 for the conjugate table: the second
        // pair is made here with sign-bit XORs (ALU pipe, idle in this loop) instead of being staged,
        // which keeps the shared-memory traffic of a complex entry at that of a real one
        const uint32_t sq = R.sgn, sp = R.sgn ^ 0x80000000u;
        const float4 va = R.v[0], vb = R.v[1];
        const float p0 = __uint_as_float(__float_as_uint(va.y) ^ sp), q0 = __uint_as_float(__float_as_uint(va.x) ^ sq);
        const float p1 = __uint_as_float(__float_as_uint(va.w) ^ sp), q1 = __uint_as_float(__float_as_uint(va.z) ^ sq);
        const float p2 = __uint_as_float(__float_as_uint(vb.y) ^ sp), q2 = __uint_as_float(__float_as_uint(vb.x) ^ sq);
        const float p3 = __uint_as_float(__float_as_uint(vb.w) ^ sp), q3 = __uint_as_float(__float_as_uint(vb.z) ^ sq);
#pragma unroll
        for (int a = 0; a < NA; ++a)
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const float cr = R.c[a][2 * b], ci = R.c[a][2 * b + 1];
                ffma2(acc[a][b][0], acc[a][b][1], cr, va.x, va.y);
                ffma2(acc[a][b][2], acc[a][b][3], cr, va.z, va.w);
                ffma2(acc[a][b][4], acc[a][b][5], cr, vb.x, vb.y);
                ffma2(acc[a][b][6], acc[a][b][7], cr, vb.z, vb.w);
                ffma2(acc[a][b][0], acc[a][b][1], ci, p0, q0);
                ffma2(acc[a][b][2], acc[a][b][3], ci, p1, q1);
                ffma2(acc[a][b][4], acc[a][b][5], ci, p2, q2);
                ffma2(acc[a][b][6], acc[a][b][7], ci, p3, q3);
            }
    } else {
#pragma unroll
        for (int a = 0; a < NA; ++a)
#pragma unroll
            for (int b = 0; b < NB; ++b) {
                const float c = R.c[a][b];
                ffma2(acc[a][b][0], acc[a][b][1], c, R.v[0].x, R.v[0].y);
                ffma2(acc[a][b][2], acc[a][b][3], c, R.v[0].z, R.v[0].w);
                ffma2(acc[a][b][4], acc[a][b][5], c, R.v[1].x, R.v[1].y);
                ffma2(acc[a][b][6], acc[a][b][7], c, R.v[1].z, R.v[1].w);
            }
    }
}

template <int NA, int NB, int NSUB, int TLOG, int MODE, int MAXW>
__global__ void __launch_bounds__(MAXW * 32, 1) grid_kernel(const GridParams p) {
    using G = Geo<NA, NB, NSUB, TLOG, MODE>;
    extern __shared__ float4 smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int table_f4 = MODE == 0 ? p.coef_f4 : 0;
    const bool bins_on = p.bins != 0;
    const int slots = bins_on ? G::SLOTS_BINS : G::SLOTS, warp_f4 = G::warp_f4(bins_on);
    float4 *region = smem + table_f4 + warp * warp_f4;         // plane A (XX, XY) then plane B (YX, YY)
    float4 *regA = region, *regB = region + G::CELLS_B;
    float4 *ring = region + 2 * G::CELLS_B;                    // 2 halves x SLOTS x VF4
    float4 *raw = ring + 2 * slots * G::SLOT_F4;               // cp.async landing buffer
    float4 *bins = raw + G::RAW_F4;                            // (bins_on) sums of w V of the carried origin, per offset

    if (MODE == 0)
        for (int i = threadIdx.x; i < p.coef_f4; i += blockDim.x) smem[i] = p.coef[i];
    // everything is cleared: records are fetched one ahead, also past the end of a batch, and
    // whatever a slot holds must be a valid table offset
    for (int i = lane; i < warp_f4; i += 32) region[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncthreads();

    const char *coef_lane;
    uint32_t tmem_base = 0;
    if constexpr (MODE == 3) {
        // the table goes to tensor memory: warp w (< 4) fills lane quadrant w, lane l its own taps
        __shared__ uint32_t tmem_base_s;
        if (warp == 0) {
            asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                         :: "r"((uint32_t)__cvta_generic_to_shared(&tmem_base_s)), "r"((uint32_t)p.tmem_cols) : "memory");
            asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        tmem_base = tmem_base_s;
        if (warp < 4) {
            const uint32_t tl = tmem_base + ((uint32_t)(warp * 32) << 16);
            const float *tab = reinterpret_cast<const float *>(p.coef);
            for (int q = 0; q < p.n_q; ++q) {
                float t[NA * NB];
#pragma unroll
                for (int a = 0; a < NA; ++a)
#pragma unroll
                    for (int b = 0; b < NB; ++b) t[a * NB + b] = tab[((q * NA + a) * 32 + lane) * NB + b];
                const uint32_t ta = tl + (uint32_t)(q * NA * NB);
                if (NA * NB == 8) {
                    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                                 :: "r"(ta), "f"(t[0]), "f"(t[1]), "f"(t[2]), "f"(t[3]), "f"(t[4 % (NA * NB)]),
                                    "f"(t[5 % (NA * NB)]), "f"(t[6 % (NA * NB)]), "f"(t[7 % (NA * NB)]) : "memory");
                } else {
                    asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1,%2};" :: "r"(ta), "f"(t[0]), "f"(t[1]) : "memory");
                }
            }
            asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
        }
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        coef_lane = reinterpret_cast<const char *>((uintptr_t)(tmem_base + ((uint32_t)((warp & 3) * 32) << 16)));
    } else if constexpr (MODE == 0)
        coef_lane = reinterpret_cast<const char *>((uintptr_t)((uint32_t)__cvta_generic_to_shared(smem) +
                                                              lane * RecRegs<NA, NB, MODE>::CF * (int)sizeof(float)));
    else
        coef_lane = reinterpret_cast<const char *>(p.coef) +
                    lane * (RecRegs<NA, NB, MODE>::CF > 4 ? 4 : RecRegs<NA, NB, MODE>::CF) * (int)sizeof(float);

    float acc[NA][NB][8];
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int k = 0; k < 8; ++k) acc[a][b][k] = 0.f;

    Producer prod;
    prod.init(p, lane, G::VSHIFT);
    Desc dC, dL, dK;                     // being consumed | landing in the raw buffer | keys in flight
    dC.bits = 0; dC.item = 0;
    dL = dC;
    unsigned start;
    dK = prod.next(p, lane, start);
    Entry eK = load_entry<G::GEN>(p, start + lane, lane < dK.cnt());
    Entry eL;
    eL.key = eL.idx = eL.aux = 0u;
    int par = 0, cur = -1, cmp = kSentinel;
    int rows_done = 0;                   // ring of rows: region rows of the current item already in its partial
    int bin_org = -1;                    // (bins_on) run the bins hold (origin; general path: plane | origin), -1: none
    int bin_poff = 0;                    // ... and its origin's region offset
    unsigned bin_occ = 0;                // ... and which of its offsets have something
    unsigned long long n_exec = 0;       // records gridded by this warp (after merging)

    while (true) {
        const float4 *half = ring + par * (slots * G::SLOT_F4);
        // the batch that landed goes to the other half (last read one iteration ago)
        cp_async_wait_all();
        __syncwarp();
        Desc dS = dL;
        if (dS.cnt() > 0) {
            float4 *other = ring + (par ^ 1) * (slots * G::SLOT_F4);
            const int n_rec = bins_on ? stage_write_bins<NA, NB, NSUB, TLOG, MODE>(p, raw, other, lane, dS, eL, bins, bin_org, bin_poff, bin_occ)
                                      : stage_write<NA, NB, NSUB, TLOG, MODE>(p, raw, other, lane, dS, eL);
            dS.bits = (dS.bits & ~63) | n_rec;          // the consumer sees the merged records
            n_exec += (unsigned)n_rec;
        }
        __syncwarp();
        // next batch's visibilities start to move, the one after that gets its keys
        issue_vis<G::GEN>(p, raw, lane, eK, lane < dK.cnt());
        dL = dK;
        eL = eK;
        dK = prod.next(p, lane, start);
        eK = load_entry<G::GEN>(p, start + lane, lane < dK.cnt());

        if (dC.end()) break;
        const int cnt = dC.cnt();
        if (cnt > 0) {
            // + sentinel (last batch of an item), padded to a multiple of the consumer's pipeline depth
            const int cnt1 = cnt + (dC.last() ? 1 : 0);
            const int cntp = G::PIPE == 3 ? ((cnt1 + 2) / 3) * 3 : ((cnt1 + 1) & ~1);
            const float4 *send = half + cntp * G::SLOT_F4;
            {
                // NSUB == 2: the virtual item's sub-patch selects its quarter of the table
                constexpr int sub_poff = 0;
                const char *cl = NSUB > 1 ? coef_lane + (int)(dC.item & 3u) * p.sub_stride_bytes : coef_lane;
                const float4 *sp = half;
                float4 *dst = p.partials + (size_t)dC.item * (2 * G::CELLS);      // (virtual) item id inside the class
                // meta of a slot: x = table offset of the next record, y = origin of this one
                if constexpr (G::PIPE == 3) {
                    // general path: the taps come from global memory (L1 / L2): three records in flight, taps
                    // fetched two records ahead (255 registers per thread are there at 8 warps per SM)
                    RecRegs<NA, NB, MODE> A, B, C;
                    int2 mA, mB, mC;
                    {
                        const float4 m0 = sp[G::VF4];
                        A.fetch(sp, __float_as_int(m0.z), cl);
                        mA = make_int2(__float_as_int(m0.x), __float_as_int(m0.y));
                        mB = *reinterpret_cast<const int2 *>(sp + G::SLOT_F4 + G::VF4);
                        B.fetch(sp + G::SLOT_F4, mA.x, cl);
                    }
                    do {
                        mC = *reinterpret_cast<const int2 *>(sp + 2 * G::SLOT_F4 + G::VF4);
                        C.fetch(sp + 2 * G::SLOT_F4, mB.x, cl);
                        consume<NA, NB, G::RW, G::CELLS, MODE>(A, mA.y + sub_poff, cur, cmp, regA, regB, lane, acc, rows_done, dst, p.counters);
                        mA = *reinterpret_cast<const int2 *>(sp + 3 * G::SLOT_F4 + G::VF4);
                        A.fetch(sp + 3 * G::SLOT_F4, mC.x, cl);
                        consume<NA, NB, G::RW, G::CELLS, MODE>(B, mB.y + sub_poff, cur, cmp, regA, regB, lane, acc, rows_done, dst, p.counters);
                        mB = *reinterpret_cast<const int2 *>(sp + 4 * G::SLOT_F4 + G::VF4);
                        B.fetch(sp + 4 * G::SLOT_F4, mA.x, cl);
                        consume<NA, NB, G::RW, G::CELLS, MODE>(C, mC.y + sub_poff, cur, cmp, regA, regB, lane, acc, rows_done, dst, p.counters);
                        sp += 3 * G::SLOT_F4;
                    } while (sp < send);
                } else {
                    RecRegs<NA, NB, MODE> A, B;
                    int2 mA, mB;
                    {
                        const float4 m0 = sp[G::VF4];
                        A.fetch(sp, __float_as_int(m0.z), cl);
                        mA = make_int2(__float_as_int(m0.x), __float_as_int(m0.y));
                    }
                    do {
                        mB = *reinterpret_cast<const int2 *>(sp + G::SLOT_F4 + G::VF4);
                        A.wait();
                        B.fetch(sp + G::SLOT_F4, mA.x, cl);
                        consume<NA, NB, G::RW, G::CELLS, MODE>(A, mA.y + sub_poff, cur, cmp, regA, regB, lane, acc, rows_done, dst, p.counters);
                        mA = *reinterpret_cast<const int2 *>(sp + 2 * G::SLOT_F4 + G::VF4);
                        B.wait();
                        A.fetch(sp + 2 * G::SLOT_F4, mB.x, cl);
                        consume<NA, NB, G::RW, G::CELLS, MODE>(B, mB.y + sub_poff, cur, cmp, regA, regB, lane, acc, rows_done, dst, p.counters);
                        sp += 2 * G::SLOT_F4;
                    } while (sp < send);
                }
            }
            if (dC.last()) {
                // the sentinel has folded the last patch in; move the region to this item's
                // partial and clear it
                cur = -1;
                cmp = kSentinel;
                __syncwarp();
                float4 *dst = p.partials + (size_t)dC.item * (2 * G::CELLS);      // (virtual) item id inside the class
                GR_CHECK(p.counters, (dC.item >> G::VSHIFT) < p.max_items_cls);
                if (G::CIRC) {
                    // the rest of the region: the rows still in the ring, then rows no entry reached (their slots
                    // were cleared when the rows SPY below them were written: zeros)
                    flush_rows<G::RW, G::SPY, G::CELLS>(regA, regB, dst, rows_done, G::RH, lane, p.counters);
                    rows_done = 0;
                } else {
                    for (int i = lane; i < 2 * G::CELLS; i += 32) {
                        stg_stream(dst + i, region[i]);
                        region[i] = make_float4(0.f, 0.f, 0.f, 0.f);
                    }
                }
                __syncwarp();
            } else if ((dC.bidx() & p.fold_mask) == p.fold_mask) {
                cmp = kForce;                               // bound the register chain
            }
        }
        dC = dS;
        par ^= 1;
    }
    cp_async_wait_all();
    if (lane == 0 && n_exec) atomicAdd(&p.counters->n_exec[p.cls], n_exec);     // integer: order-independent
    if constexpr (MODE == 3) {
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
        __syncthreads();
        if (warp == 0)
            asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(tmem_base), "r"((uint32_t)p.tmem_cols) : "memory");
    }
}

// ------------------------------------------------------------------------------------------
// Flush: one thread per grid cell.  The partial regions covering cell (x, y) belong to the tiles
// (ty, tx) with tx*T <= x < tx*T + RW (same in y); each tile's work items are added in id order
// (full chunks, then the tail).  FP64 accumulation, one rounding to FP32 at the end.  One launch
// per patch class (its tile table, its region geometry); the second class adds to the first.
// ------------------------------------------------------------------------------------------
template <int SP, int TLOG>
struct FlushGeo {
    static constexpr int T = 1 << TLOG;
    static constexpr int NSUB = SP > 16 ? 2 : 1;               // 32-cell class: 2 x 2 virtual items per work item
    static constexpr int PATCH = SP / NSUB;
    static constexpr int RW = T + PATCH - 1, RH = T + PATCH - 1, CELLS = RW * RH;
};

// cover[tile] = 1 when some occupied tile's region (all its sub-patches) can reach a cell of `tile`:
// the later classes' flushes (which only add to the grid) skip every cell of an uncovered tile.
__global__ void __launch_bounds__(256) tile_cover_kernel(const TileInfo *__restrict__ tiles, int ntx, int nty, int reach,
                                                          unsigned char *__restrict__ cover) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntx * nty) return;
    const int tx = t % ntx, ty = t / ntx;
    unsigned char c = 0;
    for (int yy = max(0, ty - reach); yy <= ty && !c; ++yy)
        for (int xx = max(0, tx - reach); xx <= tx; ++xx)
            if (tiles[yy * ntx + xx].count) { c = 1; break; }
    cover[t] = c;
}

template <int SP, int TLOG>
__global__ void __launch_bounds__(256, 6) flush_kernel(const FlushParams p) {
    using G = FlushGeo<SP, TLOG>;
    const int x = blockIdx.x * 32 + threadIdx.x;
    const int y = blockIdx.y * 8 + threadIdx.y;
    if (x >= p.n_grid || y >= p.n_grid) return;
    if (p.cover && !p.cover[min(y >> TLOG, p.nty - 1) * p.ntx + min(x >> TLOG, p.ntx - 1)]) return;
    double acc[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) acc[k] = 0.0;
    const uint32_t first_item = p.counters->cls_begin[p.cls];
#pragma unroll 1
    for (int sub = 0; sub < G::NSUB * G::NSUB; ++sub) {
        // sub-patch (sy, sx) regions are anchored PATCH (sx, sy) cells above their tile
        const int xs = x - (sub % G::NSUB) * G::PATCH, ys = y - (sub / G::NSUB) * G::PATCH;
        if (xs < 0 || ys < 0) continue;
        const int tx_hi = min(xs >> TLOG, p.ntx - 1), ty_hi = min(ys >> TLOG, p.nty - 1);
        const int tx_lo = max(0, (xs - G::RW + G::T) >> TLOG), ty_lo = max(0, (ys - G::RH + G::T) >> TLOG);
        for (int ty = ty_lo; ty <= ty_hi; ++ty)
            for (int tx = tx_lo; tx <= tx_hi; ++tx) {
                const TileInfo ti = p.tiles[ty * p.ntx + tx];
                if (ti.count == 0) continue;
                const int cell = (ys - (ty << TLOG)) * G::RW + (xs - (tx << TLOG));
                if (xs - (tx << TLOG) >= G::RW || ys - (ty << TLOG) >= G::RH) continue;
                const uint32_t n_it = ti.n_full + (ti.tail_item != 0xFFFFFFFFu ? 1u : 0u);
                for (uint32_t c = 0; c < n_it; ++c) {
                    const uint32_t item = c < ti.n_full ? ti.full_base + c : ti.tail_item;
                    const size_t vitem = (size_t)(item - first_item) * (G::NSUB * G::NSUB) + sub;
                    GR_CHECK(const_cast<Counters *>(p.counters), item >= first_item && item - first_item < p.max_items_cls && cell >= 0 && cell < G::CELLS);
                    const float4 *part = p.partials + vitem * (2 * G::CELLS);
                    const float4 a = __ldcs(part + cell), b = __ldcs(part + G::CELLS + cell);
                    acc[0] += (double)a.x; acc[1] += (double)a.y; acc[2] += (double)a.z; acc[3] += (double)a.w;
                    acc[4] += (double)b.x; acc[5] += (double)b.y; acc[6] += (double)b.z; acc[7] += (double)b.w;
                }
            }
    }
    const size_t nn = (size_t)p.n_grid * p.n_grid;
    const size_t c0 = (size_t)y * p.n_grid + x;
#pragma unroll
    for (int pol = 0; pol < 4; ++pol) {
        double re = acc[2 * pol], im = acc[2 * pol + 1];
        if (p.accumulate) {
            const float2 old = p.grid[pol * nn + c0];
            re += (double)old.x;
            im += (double)old.y;
        }
        p.grid[pol * nn + c0] = make_float2((float)re, (float)im);
    }
}

// ------------------------------------------------------------------------------------------
// Host side: kernel selection.  The register patch (NA x NB), the sub-patch count and the table
// mode follow from the plan; TLOG is a plan parameter; the block size is chosen at run time.
// ------------------------------------------------------------------------------------------
size_t grid_smem_bytes(const ClassGeo &g, int tlog, int mode, size_t table_bytes, int warps, bool bins) {
    const int vf4 = 2;
    const bool gen = mode == 1 || mode == 2;
    const int nbins = gen ? 32 : 16;                                   // Geo::NBINS
    const int slots = gen ? 40 : 36;                                   // Geo::SLOTS
    const int rows = (mode == 0 || mode == 3) ? 4 * g.NB : g.RH;       // fast path: a ring of SPY region rows (Geo::RHB)
    const size_t per_warp = (size_t)(2 * g.RW * rows + 2 * (bins ? slots + nbins : slots) * (vf4 + 1) + 32 * 2 + 8 + (bins ? 2 * nbins + (gen ? nbins / 4 : 0) : 0)) * sizeof(float4);   // Geo::warp_f4
    (void)tlog;
    return (mode == 0 ? table_bytes : 0) + per_warp * warps;
}

typedef void (*grid_fn_t)(const GridParams);
typedef void (*flush_fn_t)(const FlushParams);

constexpr int kMaxWarpsFast = 12, kMaxWarpsGeneral = 8;     // launch bounds: 168 / 255 registers

template <int NA, int NB, int NSUB, int MODE, int MAXW>
static grid_fn_t pick_tlog(int tlog) {
    switch (tlog) {
        case 2: return grid_kernel<NA, NB, NSUB, 2, MODE, MAXW>;
        case 3: return grid_kernel<NA, NB, NSUB, 3, MODE, MAXW>;
        case 4: return grid_kernel<NA, NB, NSUB, 4, MODE, MAXW>;
        default: return nullptr;
    }
}

template <int MODE, int MAXW>
static grid_fn_t pick_shape(const ClassGeo &g, int tlog) {
    if (g.NA == 1 && g.nsub == 1) return pick_tlog<1, 2, 1, MODE, MAXW>(tlog);
    if (g.NA == 2 && g.nsub == 1) return pick_tlog<2, 4, 1, MODE, MAXW>(tlog);
    if constexpr (MODE == 1 || MODE == 2) {
        if (g.NA == 2 && g.nsub == 2) return pick_tlog<2, 4, 2, MODE, MAXW>(tlog);
    }
    return nullptr;
}

static int kernel_mode(const Plan &p) { return (p.mode == 0 && p.tmem_cols > 0) ? 3 : p.mode; }

static grid_fn_t pick_grid(const ClassGeo &g, int tlog, int mode) {
    switch (mode) {
        case 0: return pick_shape<0, kMaxWarpsFast>(g, tlog);
        case 3: return pick_shape<3, kMaxWarpsFast>(g, tlog);
        case 1: return pick_shape<1, kMaxWarpsGeneral>(g, tlog);
        case 2: return pick_shape<2, kMaxWarpsGeneral>(g, tlog);
        default: return nullptr;
    }
}

template <int SP>
static flush_fn_t pick_flush_tlog(int tlog) {
    switch (tlog) {
        case 2: return flush_kernel<SP, 2>;
        case 3: return flush_kernel<SP, 3>;
        case 4: return flush_kernel<SP, 4>;
        default: return nullptr;
    }
}

static flush_fn_t pick_flush(const ClassGeo &g, int tlog) {
    switch (g.SP) {
        case 8: return pick_flush_tlog<8>(tlog);
        case 16: return pick_flush_tlog<16>(tlog);
        case 32: return pick_flush_tlog<32>(tlog);
        default: return nullptr;
    }
}

static const int kWarpChoices[] = {12, 10, 8, 6, 4, 2, 1};

cudaError_t configure_grid_kernel(Plan &p) {
    int dev = 0, smem_max = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return e;
    const int cap = p.mode == 0 ? kMaxWarpsFast : kMaxWarpsGeneral;
    for (int c = 0; c < p.n_cls; ++c) {
        ClassGeo &g = p.cls[c];
        int chosen = 0;
        for (int w : kWarpChoices) {
            if (w > cap) continue;
            if (p.warps_forced > 0 && w > p.warps_forced) continue;      // the caller's limit (tuning, tests)
            if (grid_smem_bytes(g, p.tlog, kernel_mode(p), p.coef_bytes, w, p.bins != 0) <= (size_t)smem_max) { chosen = w; break; }
        }
        if (!chosen) return cudaErrorInvalidConfiguration;
        g.warps = chosen;
        g.smem_bytes = (int)grid_smem_bytes(g, p.tlog, kernel_mode(p), p.coef_bytes, chosen, p.bins != 0);
        grid_fn_t fn = pick_grid(g, p.tlog, kernel_mode(p));
        if (!fn) return cudaErrorInvalidConfiguration;
        e = cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, g.smem_bytes);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

cudaError_t launch_grid(Plan &p, const float *vis, const float *weight, float *grid, int accumulate,
                        cudaStream_t s) {
    stage_mark(p, 4, s);
    // reset the work queues (a previous grid call leaves them past the end)
    cudaError_t e = cudaMemsetAsync(p.counters->queue_head, 0, sizeof(unsigned int) * kMaxClasses, s);
    if (e == cudaSuccess) e = cudaMemsetAsync(p.counters->n_exec, 0, sizeof(unsigned long long) * kMaxClasses, s);
    if (e != cudaSuccess) return e;
    if (p.presum_active) {           // sum the visibilities into the partial records of the plan, in input order
        e = launch_presum(p, vis, weight, s);
        if (e != cudaSuccess) return e;
        stage_mark(p, 7, s);
    }
    for (int c = 0; c < p.n_cls; ++c) {
        const ClassGeo &g = p.cls[c];
        grid_fn_t gfn = pick_grid(g, p.tlog, kernel_mode(p));
        if (!gfn) return cudaErrorInvalidConfiguration;
        GridParams gp;
        gp.keys = p.keys[p.sorted_sel];
        gp.vals = p.vals[p.sorted_sel];
        gp.items = p.items;
        gp.counters = p.counters;
        gp.vis = reinterpret_cast<const float4 *>(vis);
        gp.weight = weight;
        gp.coef = p.coef;
        gp.partials = p.partials + g.part_off_f4;
        gp.coef_f4 = p.mode == 0 ? (int)(p.coef_bytes / sizeof(float4)) : 0;
        gp.key = p.key;
        gp.fold_mask = p.fold_batches - 1;
        gp.cls = c;
        gp.sub_stride_bytes = p.cfg.oversample * p.cfg.oversample * g.sub_bytes;
        gp.tmem_cols = p.tmem_cols;
        gp.merge = p.merge;
        gp.n_q = p.cfg.oversample * p.cfg.oversample;
        gp.bins = p.bins;
        gp.n_sorted = (uint32_t)p.n_sorted;
        gp.n_src = (uint32_t)p.n_vis;                    // (record sums live in visibility slots: the same bound)
        gp.max_items_cls = (uint32_t)p.max_items_cls;
        if (p.presum_active) {       // the sorted list names partial records: their sums are the "visibilities"
            gp.vis = p.ps_sum;
            gp.weight = nullptr;
            if (gp.fold_mask > 3) gp.fold_mask = 3;
        }
        gfn<<<p.n_sm, g.warps * 32, g.smem_bytes, s>>>(gp);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        p.n_launches += 1;
    }
    stage_mark(p, 5, s);
    const size_t grid_floats = (size_t)8 * p.cfg.grid_size * p.cfg.grid_size;
    for (int c = 0; c < p.n_cls; ++c) {
        const ClassGeo &g = p.cls[c];
        flush_fn_t ffn = pick_flush(g, p.tlog);
        if (!ffn) return cudaErrorInvalidConfiguration;
        for (int gi = 0; gi < p.n_grids; ++gi) {         // (one grid, or one per channel block: gridder_bin_channels)
            FlushParams fp;
            fp.tiles = p.tile_info + (size_t)c * p.n_tiles_cls + (size_t)gi * p.n_tiles;
            fp.partials = p.partials + g.part_off_f4;
            fp.counters = p.counters;
            fp.cls = c;
            fp.grid = reinterpret_cast<float2 *>(grid + gi * grid_floats);
            fp.n_grid = p.cfg.grid_size;
            fp.ntx = p.ntx;
            fp.nty = p.nty;
            fp.accumulate = (c > 0 || accumulate) ? 1 : 0;
            fp.cover = nullptr;
            fp.max_items_cls = (uint32_t)p.max_items_cls;
            if (c > 0) {
                // a later class only adds: cells no region of the class can reach are skipped (sparse classes)
                const int reach = (g.RW - 1 + (g.nsub - 1) * 8 * g.NA + p.T - 1) / p.T;
                tile_cover_kernel<<<(p.n_tiles + 255) / 256, 256, 0, s>>>(fp.tiles, p.ntx, p.nty, reach, p.tile_cover);
                e = cudaGetLastError();
                if (e != cudaSuccess) return e;
                fp.cover = p.tile_cover;
                p.n_launches += 1;
            }
            dim3 blk(32, 8), grd((p.cfg.grid_size + 31) / 32, (p.cfg.grid_size + 7) / 8);
            ffn<<<grd, blk, 0, s>>>(fp);
            e = cudaGetLastError();
            if (e != cudaSuccess) return e;
            p.n_launches += 1;
        }
    }
    stage_mark(p, 6, s);
    if (p.profiling) p.prof_grid_calls++;
    return cudaSuccess;
}

}  // namespace gridder
