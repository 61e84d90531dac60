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
    static constexpr int CELLS = RW * RH;
    static constexpr int VF4 = 2;                              // float4 per staged visibility
    static constexpr int SLOT_F4 = VF4 + 1;                    // + (table offset of the NEXT record, origin)
    static constexpr int SLOTS = 36;                           // 32 records + sentinel + pad + look-ahead
    static constexpr int RING_F4 = 2 * SLOTS * SLOT_F4;        // two halves
    static constexpr int RAW_F4 = 32 * 2 + 8;                  // cp.async landing: 32 x {a, b}, 32 weights
    static constexpr int WARP_F4 = 2 * CELLS + RING_F4 + RAW_F4;
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

constexpr int kClaim = 4;       // work items claimed per queue access (descriptors live in lanes 0..3)

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
        coff = (int)((k.aux & 0x3fffffffu) << 8);          // table offset in 256-byte units
        if (G::CPLX) coff |= (int)(k.aux >> 31);           // bit 0: use the conjugate table (w < 0)
    } else {
        const uint32_t qmask = (1u << (2 * p.key.bits_q)) - 1u;
        x0l = (k.key >> p.key.aux_bits) & tmask;
        y0l = (k.key >> (p.key.aux_bits + TLOG)) & tmask;
        coff = (int)((k.key & qmask) * (uint32_t)(G::TMEM ? NA * NB : G::SUB_BYTES));   // bytes, or TMEM columns
    }
    const int poff = (int)(y0l * G::RW + x0l);
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
    if (keep) {
        // slot r carries the table offset of record r + 1 (the consumer loads taps one record ahead)
        // and the origin of record r; every slot also carries its own table offset (slot 0's is used)
        float4 *slot = half + slot_id * G::SLOT_F4;
        slot[0] = make_float4(sum[0], sum[1], sum[2], sum[3]);
        slot[1] = make_float4(sum[4], sum[5], sum[6], sum[7]);
        slot[G::VF4] = make_float4(__int_as_float(next_coff), __int_as_float(poff), __int_as_float(coff), 0.f);
    }
    if (lane < 2) {          // sentinel + pad (last batch of an item) or pad (odd count)
        float4 *s2 = half + (n_rec + lane) * G::SLOT_F4;
#pragma unroll
        for (int i = 0; i < G::VF4; ++i) s2[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        s2[G::VF4] = make_float4(__int_as_float(0), __int_as_float(d.last() ? kSentinel : last_poff), __int_as_float(0), 0.f);
    }
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
#pragma unroll
                for (int j = 0; j < CF / 4; ++j) {
                    const float4 t = __ldg(reinterpret_cast<const float4 *>(ca) + j);
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
template <int NA, int NB, int RW>
__device__ __forceinline__ void fold_patch(float4 *regA, float4 *regB, int base, float (&acc)[NA][NB][8]) {
    __syncwarp();       // a cell changes owner lane from one origin to the next
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
        for (int b = 0; b < NB; ++b) {
            const int o = base + 4 * b * RW + 8 * a;
            float4 x = regA[o], y = regB[o];
            x.x += acc[a][b][0]; x.y += acc[a][b][1]; x.z += acc[a][b][2]; x.w += acc[a][b][3];
            y.x += acc[a][b][4]; y.y += acc[a][b][5]; y.z += acc[a][b][6]; y.w += acc[a][b][7];
            regA[o] = x; regB[o] = y;
#pragma unroll
            for (int k = 0; k < 8; ++k) acc[a][b][k] = 0.f;
        }
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
template <int NA, int NB, int RW, int MODE>
__device__ __forceinline__ void consume(const RecRegs<NA, NB, MODE> &R, const int poff, int &cur, int &cmp,
                                        float4 *regA, float4 *regB, int lane_cell, float (&acc)[NA][NB][8]) {
    if (poff != cmp) {                                      // warp-uniform
        if (cur >= 0) fold_patch<NA, NB, RW>(regA, regB, cur + lane_cell, acc);
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
    float4 *region = smem + table_f4 + warp * G::WARP_F4;      // plane A (XX, XY) then plane B (YX, YY)
    float4 *regA = region, *regB = region + G::CELLS;
    float4 *ring = region + 2 * G::CELLS;                      // 2 halves x SLOTS x VF4
    float4 *raw = ring + G::RING_F4;                           // cp.async landing buffer

    if (MODE == 0)
        for (int i = threadIdx.x; i < p.coef_f4; i += blockDim.x) smem[i] = p.coef[i];
    // everything is cleared: records are fetched one ahead, also past the end of a batch, and
    // whatever a slot holds must be a valid table offset
    for (int i = lane; i < G::WARP_F4; i += 32) region[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncthreads();

    const int lane_cell = (lane >> 3) * G::RW + (lane & 7);      // tap (a=0, b=0) of this lane
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
        coef_lane = reinterpret_cast<const char *>(p.coef) + lane * RecRegs<NA, NB, MODE>::CF * (int)sizeof(float);

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
    unsigned long long n_exec = 0;       // records gridded by this warp (after merging)

    while (true) {
        const float4 *half = ring + par * (G::SLOTS * G::SLOT_F4);
        // the batch that landed goes to the other half (last read one iteration ago)
        cp_async_wait_all();
        __syncwarp();
        Desc dS = dL;
        if (dS.cnt() > 0) {
            const int n_rec = stage_write<NA, NB, NSUB, TLOG, MODE>(p, raw, ring + (par ^ 1) * (G::SLOTS * G::SLOT_F4),
                                                                   lane, dS, eL);
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
            const int cntp = dC.last() ? ((cnt + 2) & ~1) : ((cnt + 1) & ~1);   // + sentinel / pad, even
            const float4 *send = half + cntp * G::SLOT_F4;
            {
                // NSUB == 2: the virtual item's sub-patch selects its quarter of the table
                constexpr int sub_poff = 0;
                const char *cl = NSUB > 1 ? coef_lane + (int)(dC.item & 3u) * p.sub_stride_bytes : coef_lane;
                RecRegs<NA, NB, MODE> A, B;
                const float4 *sp = half;
                // meta of a slot: x = table offset of the next record, y = origin of this one
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
                    consume<NA, NB, G::RW, MODE>(A, mA.y + sub_poff, cur, cmp, regA, regB, lane_cell, acc);
                    mA = *reinterpret_cast<const int2 *>(sp + 2 * G::SLOT_F4 + G::VF4);
                    B.wait();
                    A.fetch(sp + 2 * G::SLOT_F4, mB.x, cl);
                    consume<NA, NB, G::RW, MODE>(B, mB.y + sub_poff, cur, cmp, regA, regB, lane_cell, acc);
                    sp += 2 * G::SLOT_F4;
                } while (sp < send);
            }
            if (dC.last()) {
                // the sentinel has folded the last patch in; move the region to this item's
                // partial and clear it
                cur = -1;
                cmp = kSentinel;
                __syncwarp();
                float4 *dst = p.partials + (size_t)dC.item * (2 * G::CELLS);      // (virtual) item id inside the class
                for (int i = lane; i < 2 * G::CELLS; i += 32) {
                    stg_stream(dst + i, region[i]);
                    region[i] = make_float4(0.f, 0.f, 0.f, 0.f);
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
// The fast path with PER-ORIGIN BINS (one real table in shared memory, 16 x 16 patch, merging on).
// Entries of a work item are sorted by patch origin, and for one origin there are only O^2 possible
// sub-cell offsets, i.e. O^2 different sets of taps.  So the weighted visibilities of an origin are
// first summed into O^2 bins of shared memory (512 B per warp at O = 4) and only when the origin
// changes are the non-empty bins gridded (256 FMAs each) -- at most O^2 records per (item, origin)
// however many entries it has; exact by linearity like the per-batch merging of stage_write, of
// which this is the complete form.  Fixed order: inside a batch the first lane of a group adds the
// others in ascending lane order, batches are added to the bins in sequence, bins are gridded in
// offset order: bit-identical reruns.  FP32 chains: <= 32 (batch), <= K/32 (bin), <= O^2 records
// in registers per origin, then the fold: inside the budget of DESIGN.md section 7.
// Pipeline per warp: sorted (key, index) pairs three batches ahead in registers, visibilities two
// batches ahead (cp.async into three landing buffers); a batch is accumulated straight out of its
// landing buffer, there is no record ring.
// ------------------------------------------------------------------------------------------
template <int TLOG, int MAXW>
__global__ void __launch_bounds__(MAXW * 32, 1) grid_kernel_qbins(const GridParams p) {
    constexpr int NA = 2, NB = 4, NRAW = 3;
    using G = Geo<NA, NB, 1, TLOG, 0>;
    extern __shared__ float4 smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_q = p.n_q;                                     // O^2 <= 64 bins
    const int warp_f4 = 2 * G::CELLS + 2 * n_q + NRAW * G::RAW_F4;
    float4 *region = smem + p.coef_f4 + warp * warp_f4;        // plane A (XX, XY) then plane B (YX, YY)
    float4 *regA = region, *regB = region + G::CELLS;
    float4 *bins = region + 2 * G::CELLS;                      // [2][q] float4: sum of w V of the current origin
    float4 *raw = bins + 2 * n_q;                              // NRAW cp.async landing buffers

    for (int i = threadIdx.x; i < p.coef_f4; i += blockDim.x) smem[i] = p.coef[i];
    for (int i = lane; i < warp_f4; i += 32) region[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncthreads();

    const int lane_cell = (lane >> 3) * G::RW + (lane & 7);
    const char *coef_lane = reinterpret_cast<const char *>((uintptr_t)((uint32_t)__cvta_generic_to_shared(smem) +
                                                                        lane * NB * (int)sizeof(float)));
    float acc[NA][NB][8];
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int k = 0; k < 8; ++k) acc[a][b][k] = 0.f;

    Producer prod;
    prod.init(p, lane, 0);
    // batch i is processed while i+1 and i+2 are landing and i+3 has its pairs in flight
    Desc d0, d1, d2, d3;
    Entry e0, e1, e2, e3;
    d0.bits = 0; d0.item = 0; d1 = d0; d2 = d0;
    e0.key = e0.idx = e0.aux = 0u; e1 = e0; e2 = e0;
    {
        unsigned start;
        d3 = prod.next(p, lane, start);
        e3 = load_entry<false>(p, start + lane, lane < d3.cnt());
    }
    unsigned long long n_exec = 0;
    const uint32_t tmask = (1u << TLOG) - 1u, qmask = (1u << (2 * p.key.bits_q)) - 1u;
    int cur = -1, cmp = kSentinel;
    int bin_org = kSentinel;             // origin the bins belong to
    unsigned long long occ = 0;          // its non-empty bins
    int slot = 0;                        // landing buffer of batch i

    while (true) {
        // batch i+2's visibilities start to move; batch i+3 gets its pairs; then batch i must have landed
        d0 = d1; e0 = e1; d1 = d2; e1 = e2; d2 = d3; e2 = e3;
        issue_vis<false>(p, raw + ((slot + 2) % NRAW) * G::RAW_F4, lane, e2, lane < d2.cnt());
        {
            unsigned start;
            d3 = prod.next(p, lane, start);
            e3 = load_entry<false>(p, start + lane, lane < d3.cnt());
        }
        asm volatile("cp.async.wait_group 2;" ::: "memory");
        __syncwarp();
        if (d0.end()) break;
        const int cnt = d0.cnt();
        if (cnt > 0) {
            const float4 *rw = raw + slot * G::RAW_F4;
            const uint32_t x0l = (e0.key >> p.key.aux_bits) & tmask, y0l = (e0.key >> (p.key.aux_bits + TLOG)) & tmask;
            const bool valid = lane < cnt;
            const int poff = valid ? (int)(y0l * G::RW + x0l) : kForce;
            const int q = (int)(e0.key & qmask);
            const float4 ra = rw[lane], rb = rw[32 + lane];
            const float w = p.weight ? reinterpret_cast<const float *>(rw + 64)[lane] : 1.0f;
            const float o[8] = {ra.x * w, ra.y * w, ra.z * w, ra.w * w, rb.x * w, rb.y * w, rb.z * w, rb.w * w};
            float sum[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) sum[k] = o[k];
            // Sum inside the batch.  Neighbouring channels of a baseline are neighbours in the sorted list and
            // mostly share (origin, offset): first a segmented tree reduction over RUNS of equal lanes (five
            // shuffle steps whatever the run lengths), then the heads of runs with equal (origin, offset) --
            // rare -- are added into the first of them one by one.  Fixed order, so reruns are bit-identical.
            const unsigned gkey = valid ? (((unsigned)poff << 8) | (unsigned)q) : (0xFFFF0000u | lane);
            const unsigned gprev = __shfl_up_sync(0xffffffffu, gkey, 1);
            const bool head = lane == 0 || gprev != gkey;
            const unsigned heads = __ballot_sync(0xffffffffu, head);
            const unsigned above = lane == 31 ? 0u : (heads & (0xFFFFFFFEu << lane));
            const int run_end = above ? __ffs(above) - 1 : 32;         // first lane of the next run
#pragma unroll
            for (int dlt = 1; dlt < 32; dlt <<= 1) {
                const bool add = lane + dlt < run_end;
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const float t = __shfl_down_sync(0xffffffffu, sum[k], dlt);
                    if (add) sum[k] += t;
                }
            }
            const unsigned grp = __match_any_sync(0xffffffffu, head ? gkey : (0xFFFF0000u | lane));
            const bool keep = valid && head && (__ffs(grp) - 1 == lane);
            unsigned rest = keep ? (grp & ~(1u << lane)) : 0u;
            if (__any_sync(0xffffffffu, rest != 0u)) {
                float hs[8];                                           // the run sums as the heads hold them now
#pragma unroll
                for (int k = 0; k < 8; ++k) hs[k] = sum[k];
                do {
                    const int src = rest ? __ffs(rest) - 1 : lane;
                    const bool add = rest != 0u;
                    rest &= rest - 1u;
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        const float t = __shfl_sync(0xffffffffu, hs[k], src);
                        if (add) sum[k] += t;
                    }
                } while (__any_sync(0xffffffffu, rest != 0u));
            }
            // origin by origin (the batch is sorted by origin); one more round with no origin ends the item
            int lp = 0;
            const bool last = d0.last();
            while (lp < cnt || (last && lp == cnt)) {
                const int seg = lp < cnt ? __shfl_sync(0xffffffffu, poff, lp) : kSentinel;
                if (seg != bin_org) {
                    // ---- grid the bins of the finished origin ------------------------------------------
                    if (occ) {
                        RecRegs<NA, NB, 0> A, B;
                        unsigned long long m = occ;
                        int qa = __ffsll((long long)m) - 1, qb;
                        m &= m - 1ull;
                        A.fetch2(bins + qa, bins + n_q + qa, qa * G::SUB_BYTES, coef_lane);
                        while (true) {
                            qb = m ? __ffsll((long long)m) - 1 : -1;
                            m &= m - 1ull;
                            if (qb >= 0) B.fetch2(bins + qb, bins + n_q + qb, qb * G::SUB_BYTES, coef_lane);
                            consume<NA, NB, G::RW, 0>(A, bin_org, cur, cmp, regA, regB, lane_cell, acc);
                            if (qb < 0) break;
                            qa = m ? __ffsll((long long)m) - 1 : -1;
                            m &= m - 1ull;
                            if (qa >= 0) A.fetch2(bins + qa, bins + n_q + qa, qa * G::SUB_BYTES, coef_lane);
                            consume<NA, NB, G::RW, 0>(B, bin_org, cur, cmp, regA, regB, lane_cell, acc);
                            if (qa < 0) break;
                        }
                        n_exec += (unsigned)__popcll(occ);
                        __syncwarp();
                        for (int k = lane; k < 2 * n_q; k += 32) bins[k] = make_float4(0.f, 0.f, 0.f, 0.f);
                        occ = 0;
                        __syncwarp();
                    }
                    bin_org = seg;
                }
                if (lp >= cnt) break;
                // ---- this origin's lanes of the batch go into the bins ---------------------------------
                const bool in_seg = poff == seg;
                const bool put = in_seg && keep;
                if (put) {               // the kept lanes of one origin have distinct offsets
                    float4 x = bins[q], y = bins[n_q + q];
                    x.x += sum[0]; x.y += sum[1]; x.z += sum[2]; x.w += sum[3];
                    y.x += sum[4]; y.y += sum[5]; y.z += sum[6]; y.w += sum[7];
                    bins[q] = x; bins[n_q + q] = y;
                }
                const unsigned lo = __reduce_or_sync(0xffffffffu, (put && q < 32) ? (1u << q) : 0u);
                const unsigned hi = __reduce_or_sync(0xffffffffu, (put && q >= 32) ? (1u << (q - 32)) : 0u);
                occ |= ((unsigned long long)hi << 32) | lo;
                lp += __popc(__ballot_sync(0xffffffffu, in_seg));
                __syncwarp();
            }
            if (last) {
                // the item's last origin has been gridded; fold it, write the region out, clear it
                if (cur >= 0) fold_patch<NA, NB, G::RW>(regA, regB, cur + lane_cell, acc);
                cur = -1; cmp = kSentinel; bin_org = kSentinel;
                __syncwarp();
                float4 *dst = p.partials + (size_t)d0.item * (2 * G::CELLS);
                for (int k = lane; k < 2 * G::CELLS; k += 32) {
                    stg_stream(dst + k, region[k]);
                    region[k] = make_float4(0.f, 0.f, 0.f, 0.f);
                }
                __syncwarp();
            }
        }
        slot = (slot + 1) % NRAW;
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    if (lane == 0 && n_exec) atomicAdd(&p.counters->n_exec[p.cls], n_exec);
}

// ------------------------------------------------------------------------------------------
// PRE-SUMMATION of a dense plan's entries (fast path, O^2 <= 16 sub-cell offsets).
// When a tile holds many more entries than it has (origin, offset) pairs -- T^2 O^2 = 256 at
// T = O = 4 -- it pays to add the weighted visibilities of every pair first (8 FMAs per entry) and to
// grid each non-empty pair once (2048 FMAs): sum_i C_q w_i V_i = C_q sum_i w_i V_i, exact by
// linearity like the per-batch merging of stage_write, of which this is the complete form.  This
// kernel does the adding: per work item it writes RECORDS (origin | offset, sum of w V), origin by
// origin; grid_kernel then runs on the records exactly as it runs on entries (keys = record keys,
// visibilities = record sums, no weights, nothing left to merge).  BASELINE.json config 4: 16.5
// entries per record.
//
// A warp walks its items' entries 64 at a time, two per lane (its own queue of work items; sorted pairs
// and visibilities land in rings of shared memory by cp.async, two to four batches ahead).  Entries of one origin are consecutive.
// Every lane PAIR (l, l + 16) keeps private bins for the O^2 offsets of the current origin in shared
// memory ([offset][half][l] float4: conflict-free whatever the offsets are); the two half-warps add
// their entries to their bins in turn, so no two lanes ever touch the same word at the same time and
// there is nothing to match, merge or serialise.
// When the origin changes (or after 1024 entries, which bounds the FP32 chain of a bin copy at 64) the 16
// private copies of each bin are added in a fixed order -- lane (q, h) adds the 16 copies of half h of bin
// q one after the other -- into registers, and at the end of the origin the non-empty bins are
// written out as records in offset order.  All orders are fixed: reruns are bit-identical.
// ------------------------------------------------------------------------------------------
constexpr int kRedWarps = 13, kRedPiece = 32;      // (a copy is shared by two lanes: chains <= 64)
constexpr int kRedBins = 16;                                   // O^2 <= 16
constexpr int kRedCopies = 16;                                 // private copies of a bin: lanes l and l + 16 share one
constexpr int kRedBatch = 64;                                  // entries per batch: two per lane
constexpr int kRedVis = 3, kRedVisF4 = 2 * (32 * 2 + 8);       // landing ring of the visibilities: 2 x (a, b, weight)
constexpr int kRedKey = 5, kRedKeyF4 = 32;                     // ring of the sorted pairs: 64 keys, 64 indices
constexpr int kRedWarpF4 = kRedBins * 2 * kRedCopies + kRedVis * kRedVisF4 + kRedKey * kRedKeyF4 + 8;

__global__ void __launch_bounds__(kRedWarps * 32, 1) reduce_kernel(const GridParams p) {
    extern __shared__ float4 smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float4 *priv = smem + (size_t)warp * kRedWarpF4;           // [q][half][lane & 15]
    float4 *vring = priv + kRedBins * 2 * kRedCopies;                  // kRedVis x 2 x {a[32], b[32], w[32]}
    uint32_t *kring = reinterpret_cast<uint32_t *>(vring + kRedVis * kRedVisF4);   // kRedKey x {key[64], idx[64]}
    uint4 *dring = reinterpret_cast<uint4 *>(kring + kRedKey * 128);                // kRedKey batch descriptors
    for (int i = lane; i < kRedWarpF4; i += 32) priv[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncwarp();

    const int tl2 = 2 * p.key.tlog;
    const uint32_t omask = (1u << tl2) - 1u, qmask = (1u << (2 * p.key.bits_q)) - 1u;
    const uint32_t dropbit = 1u << (2 * p.key.bits_q);
    const unsigned item_begin = p.counters->cls_begin[p.cls], item_end = p.counters->cls_end[p.cls];
    const uint32_t *idx_sorted = reinterpret_cast<const uint32_t *>(p.vals);
    // the lane's part in adding the private copies: half bh of bin bq (row lane of the [q][half] table)
    const int bq = lane >> 1, bh = lane & 1;
    const int cl = lane & (kRedCopies - 1);

    float4 bacc = make_float4(0.f, 0.f, 0.f, 0.f);     // sum of (bq, bh) over the pieces of the origin
    unsigned touched = 0;                // this lane's private bins that hold something
    unsigned occ = 0;                    // bins of the origin that hold something (all pieces)
    int bin_org = -1, piece = 0;
    unsigned n_rec = 0;
    size_t rec_base = 0;

    // ---- the warp's stream of batches: <= 64 consecutive entries of one work item (lane: e and e + 32) ---
    // descriptor: x = first entry, y = count | first batch of its item << 8 | last << 9 | end of stream << 10,
    // z = item (relative to the class)
    unsigned cur_id = 0, cur_start = 0, cur_len = 0, cur_off = 0;      // the item the batches are cut from
    unsigned nxt_id = 0, nxt_start = 0, nxt_len = 0;                   // claimed one item ahead
    bool nxt_ok = false, gen_end = false;
    auto claim = [&]() {
        unsigned it = 0;
        if (lane == 0) it = atomicAdd(&p.counters->queue_head[p.cls], 1u);
        nxt_id = __shfl_sync(0xffffffffu, it, 0);
        nxt_ok = item_begin + nxt_id < item_end;
        nxt_start = nxt_len = 0;
        if (nxt_ok) {
            const WorkItem w = p.items[item_begin + nxt_id];
            nxt_start = w.start;
            nxt_len = w.len;
        }
    };
    // batch m: its descriptor into the ring, the copies of its sorted pairs started
    auto gen_batch = [&](int ks) {
        if (!gen_end && cur_off >= cur_len) {
            if (!nxt_ok) gen_end = true;
            else {
                cur_id = nxt_id; cur_start = nxt_start; cur_len = nxt_len; cur_off = 0;
                claim();
            }
        }
        uint4 d = make_uint4(0u, 1u << 10, 0u, 0u);
        if (!gen_end) {
            const unsigned left = cur_len - cur_off;
            d.x = cur_start + cur_off;
            d.y = min((unsigned)kRedBatch, left) | (cur_off == 0u ? 256u : 0u) | (left <= (unsigned)kRedBatch ? 512u : 0u);
            d.z = cur_id;
            cur_off += (unsigned)kRedBatch;
        }
        if (lane == 0) dring[ks] = d;
        const int cnt = (int)(d.y & 255u);
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const bool v = lane + 32 * u < cnt;
            cp_async_4(kring + ks * 128 + 32 * u + lane, p.keys + d.x + (v ? 32 * u + lane : 0), v);
            cp_async_4(kring + ks * 128 + 64 + 32 * u + lane, idx_sorted + d.x + (v ? 32 * u + lane : 0), v);
        }
    };
    // batch m (its pairs have landed): the copies of its visibilities started
    auto gen_vis = [&](int ks, int vs) {
        const int cnt = (int)(dring[ks].y & 255u);
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const uint32_t key = kring[ks * 128 + 32 * u + lane], idx = kring[ks * 128 + 64 + 32 * u + lane];
            const bool live = lane + 32 * u < cnt && !(key & dropbit);
            float4 *dst = vring + vs * kRedVisF4 + u * (kRedVisF4 / 2);
            const float4 *src = p.vis + 2 * (size_t)(live ? idx : 0u);
            cp_async_16(dst + lane, src, live);
            cp_async_16(dst + 32 + lane, src + 1, live);
            if (p.weight) cp_async_4(reinterpret_cast<float *>(dst + 64) + lane, p.weight + (live ? idx : 0u), live);
        }
    };

    claim();
    // prologue: batches 0..3 have their pairs moving, then 0 and 1 their visibilities
    for (int m = 0; m < 4; ++m) {
        gen_batch(m);
        cp_async_commit();
    }
    asm volatile("cp.async.wait_group 2;" ::: "memory");          // pairs of batches 0 and 1
    __syncwarp();
    for (int m = 0; m < 2; ++m) {
        gen_vis(m, m);
        cp_async_commit();
    }

    // iteration n: pairs of batch n+4 and visibilities of batch n+2 start to move (one group), batch n is added
    int kn = 0, vn = 0;                  // ring slots of batch n
#pragma unroll 1
    while (true) {
        asm volatile("cp.async.wait_group 1;" ::: "memory");      // groups up to iteration n-2: pairs(n+2), vis(n)
        __syncwarp();
        gen_batch(kn + 4 < kRedKey ? kn + 4 : kn + 4 - kRedKey);
        gen_vis(kn + 2 < kRedKey ? kn + 2 : kn + 2 - kRedKey, vn + 2 < kRedVis ? vn + 2 : vn + 2 - kRedVis);
        cp_async_commit();
        const uint4 d = dring[kn];
        if (d.y & 1024u) break;
        const int cnt = (int)(d.y & 255u);
        {
            const float4 *rw = vring + vn * kRedVisF4;
            if (d.y & 256u) {            // first batch of an item: where its records go
                n_rec = 0;
                rec_base = p.rec_slot ? (size_t)d.z * p.rec_slot : (size_t)d.x;
            }
            const uint32_t key0 = kring[kn * 128 + lane], key1 = kring[kn * 128 + 32 + lane];
            const int org0 = lane < cnt ? (int)((key0 >> p.key.aux_bits) & omask) : -2;
            const int org1 = lane + 32 < cnt ? (int)((key1 >> p.key.aux_bits) & omask) : -2;
            const int q0 = (int)(key0 & qmask), q1 = (int)(key1 & qmask);
            const float w0 = p.weight ? reinterpret_cast<const float *>(rw + 64)[lane] : 1.0f;
            const float w1 = p.weight ? reinterpret_cast<const float *>(rw + kRedVisF4 / 2 + 64)[lane] : 1.0f;
            const float4 a0 = rw[lane], b0 = rw[32 + lane];
            const float4 a1 = rw[kRedVisF4 / 2 + lane], b1 = rw[kRedVisF4 / 2 + 32 + lane];
            const bool last = d.y & 512u;
            int lp = 0;
            // origin by origin; one more round with no origin ends the item
#pragma unroll 1
            while (lp < cnt || (last && lp == cnt)) {
                const int seg = lp < cnt ? __shfl_sync(0xffffffffu, lp < 32 ? org0 : org1, lp & 31) : -1;
                const bool change = seg != bin_org;
                if ((change && bin_org >= 0) || piece >= kRedPiece) {
                    // ---- the 16 private copies of every bin are added into bacc and cleared: lane (q, h) adds
                    // half h of bin q, copy by copy in a fixed (rotated: conflict-free) order
                    __syncwarp();
                    occ |= __reduce_or_sync(0xffffffffu, touched);
                    {
                        const float4 *src = priv + lane * kRedCopies;        // row (q * 2 + h) = lane
                        float4 t = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                        for (int j = 0; j < kRedCopies; ++j) {
                            const float4 v = src[(j + lane) & (kRedCopies - 1)];
                            t.x += v.x; t.y += v.y; t.z += v.z; t.w += v.w;
                        }
                        bacc.x += t.x; bacc.y += t.y; bacc.z += t.z; bacc.w += t.w;
                    }
                    __syncwarp();
                    for (unsigned m = touched; m; m &= m - 1u) {     // (lanes l and l + 16 may clear the same words)
                        const int qq = __ffs(m) - 1;
                        priv[(qq * 2) * kRedCopies + cl] = make_float4(0.f, 0.f, 0.f, 0.f);
                        priv[(qq * 2 + 1) * kRedCopies + cl] = make_float4(0.f, 0.f, 0.f, 0.f);
                    }
                    touched = 0;
                    piece = 0;
                    __syncwarp();
                    if (change) {
                        // ---- the origin is complete: its non-empty bins become records, in offset order ----
                        if ((occ >> bq) & 1u) {
                            const size_t r = rec_base + n_rec + (unsigned)__popc(occ & ((1u << bq) - 1u));
                            p.rec_sum[2 * r + bh] = bacc;
                            if (bh == 0) p.rec_key[r] = ((uint32_t)bin_org << p.key.aux_bits) | (uint32_t)bq;
                        }
                        bacc = make_float4(0.f, 0.f, 0.f, 0.f);
                        n_rec += (unsigned)__popc(occ);
                        occ = 0;
                    }
                }
                bin_org = seg;
                if (lp >= cnt) break;
                // the lane's two entries: into its copy of the bins (one read-modify-write when they share the
                // offset); lanes l and l + 16 share a copy, so the two half-warps take turns
                const bool in0 = org0 == seg, in1 = org1 == seg;
                const bool same = in0 && in1 && q0 == q1;
                float4 *pa0 = priv + (q0 * 2) * kRedCopies + cl, *pa1 = priv + (q1 * 2) * kRedCopies + cl;
#pragma unroll 1
                for (int ph = 0; ph < 2; ++ph) {
                    if ((lane >> 4) == ph) {
                        // (the addresses are valid whatever the lane holds: loads are unconditional, stores are not)
                        float4 x0 = pa0[0], y0 = pa0[kRedCopies];
                        float4 x1 = pa1[0], y1 = pa1[kRedCopies];
                        x0.x = fmaf(w0, a0.x, x0.x); x0.y = fmaf(w0, a0.y, x0.y); x0.z = fmaf(w0, a0.z, x0.z); x0.w = fmaf(w0, a0.w, x0.w);
                        y0.x = fmaf(w0, b0.x, y0.x); y0.y = fmaf(w0, b0.y, y0.y); y0.z = fmaf(w0, b0.z, y0.z); y0.w = fmaf(w0, b0.w, y0.w);
                        if (same) { x1 = x0; y1 = y0; }
                        x1.x = fmaf(w1, a1.x, x1.x); x1.y = fmaf(w1, a1.y, x1.y); x1.z = fmaf(w1, a1.z, x1.z); x1.w = fmaf(w1, a1.w, x1.w);
                        y1.x = fmaf(w1, b1.x, y1.x); y1.y = fmaf(w1, b1.y, y1.y); y1.z = fmaf(w1, b1.z, y1.z); y1.w = fmaf(w1, b1.w, y1.w);
                        if (in0 && !same) { pa0[0] = x0; pa0[kRedCopies] = y0; }
                        if (in1) { pa1[0] = x1; pa1[kRedCopies] = y1; }
                    }
                    __syncwarp();
                }
                if (in0) touched |= 1u << q0;
                if (in1) touched |= 1u << q1;
                piece += 2;
                lp += __popc(__ballot_sync(0xffffffffu, in0)) + __popc(__ballot_sync(0xffffffffu, in1));
            }
            if (last && lane == 0) {     // the item's entry in the record items
                WorkItem ri;
                ri.start = (uint32_t)rec_base;
                ri.len = n_rec;
                ri.tile = 0;
                ri.pad = 0;
                p.rec_items[item_begin + d.z] = ri;
            }
        }
        kn = kn + 1 < kRedKey ? kn + 1 : 0;
        vn = vn + 1 < kRedVis ? vn + 1 : 0;
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
}

// The same pre-summation straight from the SORTED CHANNEL RUNS (runs.cu), so that the per-entry sorted
// list never has to be written (expand_kernel: 3.7 ms and 6.4 GB on config 4) or read.  Entry e of the
// sorted order belongs to the run r with rcum[r] <= e < rcum[r + 1]; it is visibility start[r] + (e - rcum[r]),
// its origin is in the run's key and its sub-cell offsets (and drop flag) are the byte qaux[visibility].
// Batches are cut at multiples of 64 of the global entry position, and blk_run[e / 64] (block_run_kernel)
// names the run holding position 64 (e / 64): the 64 runs from there on cover the batch (a run has at least
// one entry), so a lane finds its run by a 6-step search in a window of shared memory.  Four stages run
// ahead of the adding, each through its own ring: descriptor + blk_run word (6 batches ahead), run window
// (4), visibilities + weight + qaux word (2).  Same records, same order of additions, same bits as
// reduce_kernel.
constexpr int kRunWin = 4, kRunWinU32 = 192;                   // ring of run windows: cum[64], start[64], key[64]
constexpr int kRunEnt = 3, kRunEntF4 = 2 * (32 * 2 + 8) + 32;  // ring of entries: 2 x (a, b, weight), then okey[64], qword[64]
constexpr int kRunDesc = 8;
constexpr int kRunWarps = 11;
constexpr int kRunWarpF4 = kRedBins * 2 * kRedCopies + kRunEnt * kRunEntF4 + kRunWin * kRunWinU32 / 4 + kRunDesc;

__global__ void __launch_bounds__(kRunWarps * 32, 1) reduce_runs_kernel(const GridParams p) {
    extern __shared__ float4 smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float4 *priv = smem + (size_t)warp * kRunWarpF4;           // [q][half][lane & 15]
    float4 *ering = priv + kRedBins * 2 * kRedCopies;
    uint32_t *wring = reinterpret_cast<uint32_t *>(ering + kRunEnt * kRunEntF4);
    uint4 *dring = reinterpret_cast<uint4 *>(wring + kRunWin * kRunWinU32);
    for (int i = lane; i < kRunWarpF4; i += 32) priv[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncwarp();

    const int tl2 = 2 * p.key.tlog;
    const uint32_t omask = (1u << tl2) - 1u, qmask = (1u << (2 * p.key.bits_q)) - 1u;
    const int dropshift = 2 * p.key.bits_q;
    const unsigned item_begin = p.counters->cls_begin[p.cls], item_end = p.counters->cls_end[p.cls];
    // the lane's part in adding the private copies: half bh of bin bq (row lane of the [q][half] table)
    const int bq = lane >> 1, bh = lane & 1;
    const int cl = lane & (kRedCopies - 1);

    float4 bacc = make_float4(0.f, 0.f, 0.f, 0.f);     // sum of (bq, bh) over the pieces of the origin
    unsigned touched = 0;                // this lane's private bins that hold something
    unsigned occ = 0;                    // bins of the origin that hold something (all pieces)
    int bin_org = -1, piece = 0;
    unsigned n_rec = 0;
    size_t rec_base = 0;

    // ---- the warp's stream of batches: consecutive entries of one work item up to the next multiple of 64
    // of the global position (lane: positions x + lane and x + 32 + lane).  descriptor: x = first position,
    // y = count | first batch of its item << 8 | last << 9 | end of stream << 10, z = item, w = blk_run[x / 64]
    unsigned cur_id = 0, cur_pos = 0, cur_end = 0;                     // the item the batches are cut from
    bool cur_first = false;
    unsigned nxt_id = 0, nxt_start = 0, nxt_len = 0;                   // claimed one item ahead
    bool nxt_ok = false, gen_end = false;
    auto claim = [&]() {
        unsigned it = 0;
        if (lane == 0) it = atomicAdd(&p.counters->queue_head[p.cls], 1u);
        nxt_id = __shfl_sync(0xffffffffu, it, 0);
        nxt_ok = item_begin + nxt_id < item_end;
        nxt_start = nxt_len = 0;
        if (nxt_ok) {
            const WorkItem w = p.items[item_begin + nxt_id];
            nxt_start = w.start;
            nxt_len = w.len;
        }
    };
    // stage 1, batch m: its descriptor into the ring, the copy of its blk_run word started
    auto gen_desc = [&](int m) {
        if (!gen_end && cur_pos >= cur_end) {
            if (!nxt_ok) gen_end = true;
            else {
                cur_id = nxt_id; cur_pos = nxt_start; cur_end = nxt_start + nxt_len; cur_first = true;
                claim();
            }
        }
        uint4 d = make_uint4(0u, 1u << 10, 0u, 0u);
        if (!gen_end) {
            const unsigned stop = min(cur_end, (cur_pos | 63u) + 1u);
            d.x = cur_pos;
            d.y = (stop - cur_pos) | (cur_first ? 256u : 0u) | (stop == cur_end ? 512u : 0u);
            d.z = cur_id;
            cur_pos = stop;
            cur_first = false;
        }
        uint4 *slot = dring + (m & (kRunDesc - 1));
        if (lane == 0) {
            *reinterpret_cast<uint3 *>(slot) = make_uint3(d.x, d.y, d.z);
            cp_async_4(&slot->w, p.blk_run + (d.x >> 6), !(d.y & 1024u));
        }
    };
    // stage 2, batch m (its blk_run word has landed): the copies of its window of 64 runs started
    auto gen_window = [&](int m) {
        const uint4 d = dring[m & (kRunDesc - 1)];
        uint32_t *w = wring + (m & (kRunWin - 1)) * kRunWinU32;
        const bool live = !(d.y & 1024u);
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const unsigned r = d.w + 32 * u + lane;
            const bool v = live && r < p.n_runs;
            if (v) cp_async_4(w + 32 * u + lane, p.rcum + r, true);
            else w[32 * u + lane] = 0xFFFFFFFFu;             // beyond the last run: never chosen by the search
            cp_async_4(w + 64 + 32 * u + lane, p.rstart + 2 * (size_t)(v ? r : 0u), v);
            cp_async_4(w + 128 + 32 * u + lane, p.rkey + (v ? r : 0u), v);
        }
    };
    // stage 3, batch m (its window has landed): every lane finds the runs of its two entries, notes origin
    // and byte position, and starts the copies of visibility, weight and the qaux word
    auto gen_entries = [&](int m, int es) {
        const uint4 d = dring[m & (kRunDesc - 1)];
        const uint32_t *w = wring + (m & (kRunWin - 1)) * kRunWinU32;
        const int cnt = (int)(d.y & 255u);
        float4 *dst0 = ering + es * kRunEntF4;
        uint32_t *okey = reinterpret_cast<uint32_t *>(dst0 + 2 * (32 * 2 + 8));
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const bool v = lane + 32 * u < cnt;
            const unsigned pos = d.x + 32 * u + lane;
            int j = 0;
#pragma unroll
            for (int st = 32; st >= 1; st >>= 1)
                if (w[j + st] <= pos) j += st;
            const unsigned idx = v ? w[64 + j] + (pos - w[j]) : 0u;
            okey[32 * u + lane] = ((w[128 + j] >> p.key.aux_bits) & omask) | ((idx & 3u) << 16);
            float4 *dst = dst0 + u * (32 * 2 + 8);
            const float4 *src = p.vis + 2 * (size_t)idx;
            cp_async_16(dst + lane, src, v);
            cp_async_16(dst + 32 + lane, src + 1, v);
            if (p.weight) cp_async_4(reinterpret_cast<float *>(dst + 64) + lane, p.weight + idx, v);
            cp_async_4(okey + 64 + 32 * u + lane, p.qaux + (idx & ~3u), v);
        }
    };

    claim();
    // iteration n: stages 1, 2, 3 for batches n + 6, n + 4, n + 2 (one cp.async group), batch n is added; the
    // first six iterations only fill the pipeline
    int es_n = 0, es_n2 = 2;             // entry-ring slots of batches n and n + 2 (n = -6: any)
#pragma unroll 1
    for (int n = -6;; ++n) {
        asm volatile("cp.async.wait_group 1;" ::: "memory");      // everything up to iteration n - 2 has landed
        __syncwarp();
        gen_desc(n + 6);
        if (n + 4 >= 0) gen_window(n + 4);
        if (n + 2 >= 0) gen_entries(n + 2, es_n2);
        cp_async_commit();
        if (n >= 0) {
        const uint4 d = dring[n & (kRunDesc - 1)];
        if (d.y & 1024u) break;
        const int cnt = (int)(d.y & 255u);
        {
            const float4 *rw = ering + es_n * kRunEntF4;
            const uint32_t *okey = reinterpret_cast<const uint32_t *>(rw + 2 * (32 * 2 + 8));
            if (d.y & 256u) {            // first batch of an item: where its records go
                n_rec = 0;
                rec_base = p.rec_slot ? (size_t)d.z * p.rec_slot : (size_t)d.x;
            }
            const uint32_t k0 = okey[lane], k1 = okey[32 + lane];
            const uint32_t qb0 = (okey[64 + lane] >> (8 * (k0 >> 16))) & 255u;
            const uint32_t qb1 = (okey[96 + lane] >> (8 * (k1 >> 16))) & 255u;
            const int org0 = lane < cnt ? (int)(k0 & 0xFFFFu) : -2;
            const int org1 = lane + 32 < cnt ? (int)(k1 & 0xFFFFu) : -2;
            const int q0 = (int)(qb0 & qmask), q1 = (int)(qb1 & qmask);
            const bool drop0 = (qb0 >> dropshift) & 1u, drop1 = (qb1 >> dropshift) & 1u;      // dropped: adds nothing
            const float w0 = drop0 ? 0.0f : (p.weight ? reinterpret_cast<const float *>(rw + 64)[lane] : 1.0f);
            const float w1 = drop1 ? 0.0f : (p.weight ? reinterpret_cast<const float *>(rw + (32 * 2 + 8) + 64)[lane] : 1.0f);
            const float4 z4 = make_float4(0.f, 0.f, 0.f, 0.f);
            const float4 a0 = drop0 ? z4 : rw[lane], b0 = drop0 ? z4 : rw[32 + lane];
            const float4 a1 = drop1 ? z4 : rw[(32 * 2 + 8) + lane], b1 = drop1 ? z4 : rw[(32 * 2 + 8) + 32 + lane];
            const bool last = d.y & 512u;
            int lp = 0;
            // origin by origin; one more round with no origin ends the item
#pragma unroll 1
            while (lp < cnt || (last && lp == cnt)) {
                const int seg = lp < cnt ? __shfl_sync(0xffffffffu, lp < 32 ? org0 : org1, lp & 31) : -1;
                const bool change = seg != bin_org;
                if ((change && bin_org >= 0) || piece >= kRedPiece) {
                    // ---- the 16 private copies of every bin are added into bacc and cleared: lane (q, h) adds
                    // half h of bin q, copy by copy in a fixed (rotated: conflict-free) order
                    __syncwarp();
                    occ |= __reduce_or_sync(0xffffffffu, touched);
                    {
                        const float4 *src = priv + lane * kRedCopies;        // row (q * 2 + h) = lane
                        float4 t = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
                        for (int j = 0; j < kRedCopies; ++j) {
                            const float4 v = src[(j + lane) & (kRedCopies - 1)];
                            t.x += v.x; t.y += v.y; t.z += v.z; t.w += v.w;
                        }
                        bacc.x += t.x; bacc.y += t.y; bacc.z += t.z; bacc.w += t.w;
                    }
                    __syncwarp();
                    for (unsigned m = touched; m; m &= m - 1u) {     // (lanes l and l + 16 may clear the same words)
                        const int qq = __ffs(m) - 1;
                        priv[(qq * 2) * kRedCopies + cl] = make_float4(0.f, 0.f, 0.f, 0.f);
                        priv[(qq * 2 + 1) * kRedCopies + cl] = make_float4(0.f, 0.f, 0.f, 0.f);
                    }
                    touched = 0;
                    piece = 0;
                    __syncwarp();
                    if (change) {
                        // ---- the origin is complete: its non-empty bins become records, in offset order ----
                        if ((occ >> bq) & 1u) {
                            const size_t r = rec_base + n_rec + (unsigned)__popc(occ & ((1u << bq) - 1u));
                            p.rec_sum[2 * r + bh] = bacc;
                            if (bh == 0) p.rec_key[r] = ((uint32_t)bin_org << p.key.aux_bits) | (uint32_t)bq;
                        }
                        bacc = make_float4(0.f, 0.f, 0.f, 0.f);
                        n_rec += (unsigned)__popc(occ);
                        occ = 0;
                    }
                }
                bin_org = seg;
                if (lp >= cnt) break;
                // the lane's two entries: into its copy of the bins (one read-modify-write when they share the
                // offset); lanes l and l + 16 share a copy, so the two half-warps take turns
                const bool in0 = org0 == seg, in1 = org1 == seg;
                const bool same = in0 && in1 && q0 == q1;
                float4 *pa0 = priv + (q0 * 2) * kRedCopies + cl, *pa1 = priv + (q1 * 2) * kRedCopies + cl;
#pragma unroll 1
                for (int ph = 0; ph < 2; ++ph) {
                    if ((lane >> 4) == ph) {
                        // (the addresses are valid whatever the lane holds: loads are unconditional, stores are not)
                        float4 x0 = pa0[0], y0 = pa0[kRedCopies];
                        float4 x1 = pa1[0], y1 = pa1[kRedCopies];
                        x0.x = fmaf(w0, a0.x, x0.x); x0.y = fmaf(w0, a0.y, x0.y); x0.z = fmaf(w0, a0.z, x0.z); x0.w = fmaf(w0, a0.w, x0.w);
                        y0.x = fmaf(w0, b0.x, y0.x); y0.y = fmaf(w0, b0.y, y0.y); y0.z = fmaf(w0, b0.z, y0.z); y0.w = fmaf(w0, b0.w, y0.w);
                        if (same) { x1 = x0; y1 = y0; }
                        x1.x = fmaf(w1, a1.x, x1.x); x1.y = fmaf(w1, a1.y, x1.y); x1.z = fmaf(w1, a1.z, x1.z); x1.w = fmaf(w1, a1.w, x1.w);
                        y1.x = fmaf(w1, b1.x, y1.x); y1.y = fmaf(w1, b1.y, y1.y); y1.z = fmaf(w1, b1.z, y1.z); y1.w = fmaf(w1, b1.w, y1.w);
                        if (in0 && !same) { pa0[0] = x0; pa0[kRedCopies] = y0; }
                        if (in1) { pa1[0] = x1; pa1[kRedCopies] = y1; }
                    }
                    __syncwarp();
                }
                if (in0) touched |= 1u << q0;
                if (in1) touched |= 1u << q1;
                piece += 2;
                lp += __popc(__ballot_sync(0xffffffffu, in0)) + __popc(__ballot_sync(0xffffffffu, in1));
            }
            if (last && lane == 0) {     // the item's entry in the record items
                WorkItem ri;
                ri.start = (uint32_t)rec_base;
                ri.len = n_rec;
                ri.tile = 0;
                ri.pad = 0;
                p.rec_items[item_begin + d.z] = ri;
            }
        }
        }
        es_n = es_n + 1 < kRunEnt ? es_n + 1 : 0;
        es_n2 = es_n2 + 1 < kRunEnt ? es_n2 + 1 : 0;
    }
    asm volatile("cp.async.wait_group 0;" ::: "memory");
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
__global__ void __launch_bounds__(256) flush_kernel(const FlushParams p) {
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
size_t grid_smem_bytes(const ClassGeo &g, int tlog, int mode, size_t table_bytes, int warps, int qbins) {
    const int vf4 = 2;
    if (qbins > 0)      // grid_kernel_qbins: region, O^2 bins, three landing buffers
        return table_bytes + (size_t)(2 * g.RW * g.RH + 2 * qbins + 3 * (32 * 2 + 8)) * sizeof(float4) * warps;
    (void)mode;
    const size_t per_warp = (size_t)(2 * g.RW * g.RH + 2 * 36 * (vf4 + 1) + 32 * 2 + 8) * sizeof(float4);   // Geo::WARP_F4
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

static int kernel_qbins(const Plan &p) { return p.reduce ? 0 : p.qbins; }      // the kernel with its own bins
static int kernel_mode(const Plan &p) { return (p.mode == 0 && p.tmem_cols > 0) ? 3 : p.mode; }

static grid_fn_t pick_qbins(int tlog) {
    switch (tlog) {
        case 2: return grid_kernel_qbins<2, kMaxWarpsFast>;
        case 3: return grid_kernel_qbins<3, kMaxWarpsFast>;
        case 4: return grid_kernel_qbins<4, kMaxWarpsFast>;
        default: return nullptr;
    }
}

static grid_fn_t pick_grid(const ClassGeo &g, int tlog, int mode, int qbins = 0) {
    if (qbins > 0) return pick_qbins(tlog);
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
            if (grid_smem_bytes(g, p.tlog, kernel_mode(p), p.coef_bytes, w, kernel_qbins(p)) <= (size_t)smem_max) { chosen = w; break; }
        }
        if (!chosen) return cudaErrorInvalidConfiguration;
        g.warps = chosen;
        g.smem_bytes = (int)grid_smem_bytes(g, p.tlog, kernel_mode(p), p.coef_bytes, chosen, kernel_qbins(p));
        grid_fn_t fn = pick_grid(g, p.tlog, kernel_mode(p), kernel_qbins(p));
        if (!fn) return cudaErrorInvalidConfiguration;
        e = cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, g.smem_bytes);
        if (e != cudaSuccess) return e;
    }
    if (p.reduce) {
        e = cudaFuncSetAttribute((const void *)reduce_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)(kRedWarps * kRedWarpF4 * sizeof(float4)));
        if (e == cudaSuccess && p.fuse)
            e = cudaFuncSetAttribute((const void *)reduce_runs_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)(kRunWarps * kRunWarpF4 * sizeof(float4)));
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
    if (p.reduce) {                  // sum the entries into records first; the grid kernel then takes those
        GridParams rp;
        memset(&rp, 0, sizeof(rp));
        rp.keys = p.keys[p.sorted_sel];
        rp.vals = p.vals[p.sorted_sel];
        rp.items = p.items;
        rp.counters = p.counters;
        rp.vis = reinterpret_cast<const float4 *>(vis);
        rp.weight = weight;
        if (p.presum_active) {       // the sorted list names partial records: their sums are the "visibilities"
            rp.vis = p.ps_sum;
            rp.weight = nullptr;
        }
        rp.key = p.key;
        rp.cls = 0;
        rp.rec_key = p.rec_key;
        rp.rec_sum = p.rec_sum;
        rp.rec_items = p.rec_items;
        rp.rec_slot = (uint32_t)p.rec_slot;
        if (p.fused_bin) {           // binned by runs and not expanded: straight from the sorted runs
            rp.rkey = p.srun_key;
            rp.rstart = reinterpret_cast<const uint32_t *>(p.srun_val);
            rp.rcum = p.run_cum;
            rp.n_runs = (uint32_t)p.n_runs;
            rp.qaux = p.qaux;
            rp.blk_run = p.blk_run;
            reduce_runs_kernel<<<p.n_sm, kRunWarps * 32, kRunWarps * kRunWarpF4 * sizeof(float4), s>>>(rp);
        } else {
            reduce_kernel<<<p.n_sm, kRedWarps * 32, kRedWarps * kRedWarpF4 * sizeof(float4), s>>>(rp);
        }
        e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaMemsetAsync(p.counters->queue_head, 0, sizeof(unsigned int) * kMaxClasses, s);
        if (e != cudaSuccess) return e;
        p.n_launches += 1;
        stage_mark(p, 8, s);
    }
    for (int c = 0; c < p.n_cls; ++c) {
        const ClassGeo &g = p.cls[c];
        grid_fn_t gfn = pick_grid(g, p.tlog, kernel_mode(p), kernel_qbins(p));
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
        if (p.reduce) {              // the entries were summed into records: grid those, as they are
            gp.keys = p.rec_key;
            gp.vals = nullptr;
            gp.items = p.rec_items;
            gp.vis = p.rec_sum;
            gp.weight = nullptr;
            gp.merge = 0;
            if (gp.fold_mask > 3) gp.fold_mask = 3;      // a record is a sum already: shorter register chains
        }
        if (p.presum_active && !p.reduce) {       // the sorted list names partial records: their sums are the "visibilities"
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
    for (int c = 0; c < p.n_cls; ++c) {
        const ClassGeo &g = p.cls[c];
        flush_fn_t ffn = pick_flush(g, p.tlog);
        if (!ffn) return cudaErrorInvalidConfiguration;
        FlushParams fp;
        fp.tiles = p.tile_info + (size_t)c * p.n_tiles;
        fp.partials = p.partials + g.part_off_f4;
        fp.counters = p.counters;
        fp.cls = c;
        fp.grid = reinterpret_cast<float2 *>(grid);
        fp.n_grid = p.cfg.grid_size;
        fp.ntx = p.ntx;
        fp.nty = p.nty;
        fp.accumulate = (c > 0 || accumulate) ? 1 : 0;
        fp.cover = nullptr;
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
    stage_mark(p, 6, s);
    if (p.profiling) p.prof_grid_calls++;
    return cudaSuccess;
}

}  // namespace gridder
