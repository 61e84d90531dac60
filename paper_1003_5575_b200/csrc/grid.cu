// gridder_grid: the gridding kernel (FP32 FMA, registers + shared memory) and the deterministic flush.
//
// Grid kernel.  PAPER.md :197-199 gathers per pixel from 9 bins; here the work
// is turned round so that every lane does useful FMAs on every visibility:
//   * a work item is <= K consecutive entries of one uv tile's sorted list; ONE WARP owns it;
//   * the warp keeps the item's (T + SP - 1)^2-cell region (tile + halo) in shared memory;
//   * for the current patch origin the SP x SP patch lives in REGISTERS, NA*NB cells (x 4 pol
//     complex = 8 floats) per lane; entries are sorted by origin, so the patch is exchanged with
//     the shared region only when the origin changes;
//   * per entry a lane does 3 broadcast LDS.128 (visibility + meta), NA vector LDS (its taps of the
//     GCF sub-table) and 8*NA*NB FFMA; visibilities are fetched one batch of 32 ahead with
//     128-bit loads (float4 per polarisation pair) and pre-multiplied by their weight;
//   * no atomics anywhere: every region cell has one owner lane, every work item its own partial
//     region in HBM.
// Flush kernel: each grid cell sums, in FP64 and in a fixed (tile row, tile column, chunk) order,
// the partial regions that cover it, and writes the complex64 grid once.
#include "gridder_internal.cuh"

namespace gridder {

template <int NA, int NB, int TLOG>
struct Geo {
    static constexpr int SPX = 8 * NA, SPY = 4 * NB;         // padded patch
    static constexpr int T = 1 << TLOG;
    static constexpr int RW = T + SPX - 1, RH = T + SPY - 1;   // region = tile + halo
    static constexpr int CELLS = RW * RH;
    static constexpr int HALF_SLOTS = 32 + 3;                  // (3 = the consumer's look-ahead)
    static constexpr int HALF_SLOTS_UNUSED = 0;                  // a batch + copies of the next batch's first records
    static constexpr int STAGE_F4 = 2 * HALF_SLOTS * 3;        // 2 halves x slots x 3 float4
    static constexpr int RAW_F4 = 32 * 3;                      // cp.async landing buffer: one batch
    static constexpr int WARP_F4 = 2 * CELLS + STAGE_F4 + RAW_F4;   // shared float4 per warp
};

__device__ __forceinline__ float4 ldg_stream(const float4 *p) {
    float4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
                 : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
}

__device__ __forceinline__ void stg_stream(float4 *p, const float4 &v) {
    asm volatile("st.global.L1::no_allocate.v4.f32 [%0], {%1,%2,%3,%4};"
                 :: "l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

// ---- staging pipeline, three batches deep -------------------------------------------------------
// Batch j+3: sorted (key, visibility index) loads in flight (two registers).  Batch j+2: its
// visibilities and weights in flight as cp.async copies into the warp's raw buffer -- no register
// holds them, so nothing is spilled while the FFMA loop runs.  Batch j+1: read back from the raw
// buffer by its own lane, multiplied by its weight and written to the record ring while batch j is
// being gridded.  No load is consumed in the step that issued it.
struct KeyIdx {
    uint32_t key, idx;
};

__device__ __forceinline__ KeyIdx load_keyidx(const GridParams &p, uint32_t e, bool valid) {
    KeyIdx k;
    k.key = 0u;
    k.idx = 0u;
    if (valid) {
        k.key = __ldg(p.keys + e);
        k.idx = __ldg(p.vals + e);
    }
    return k;
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

// Starts the copies of one batch: lane's record goes to raw[lane] = {a, b, (w, -, -, -)}.
// A lane past the end of the item, or a dropped visibility, gets zeros (and so adds nothing).
__device__ __forceinline__ void issue_vis(const GridParams &p, float4 *raw, int lane, const KeyIdx k, bool valid) {
    const bool dropped = (k.key >> (2 * p.key.bits_q)) & 1u;
    const bool live = valid && !dropped;
    const float4 *src = p.vis + 2 * (size_t)(live ? k.idx : 0u);
    float4 *dst = raw + lane * 3;
    cp_async_16(dst, src, live);
    cp_async_16(dst + 1, src + 1, live);
    if (p.weight) cp_async_4(dst + 2, p.weight + (live ? k.idx : 0u), live);
    cp_async_commit();
}

// Moves a landed batch of `cnt` <= 32 records from the raw buffer into `half` of the ring in the
// consumer's format {w*a, w*b, (table offset, origin)}; lanes past the end write a record that adds
// nothing (zero visibility, the last record's origin) so that the consumer can work in fours.  The
// first records are repeated in the extension slots of the other half, where the consumer's
// look-ahead finds them without wrapping.
template <int NA, int NB, int TLOG>
__device__ __forceinline__ void stage_write(const GridParams &p, const float4 *raw, float4 *half, float4 *other_ext,
                                            int lane, int cnt, uint32_t key) {
    using G = Geo<NA, NB, TLOG>;
    const uint32_t qmask = (1u << (2 * p.key.bits_q)) - 1u;
    const uint32_t tmask = (1u << TLOG) - 1u;
    const uint32_t x0l = (key >> p.key.aux_bits) & tmask;
    const uint32_t y0l = (key >> (p.key.aux_bits + TLOG)) & tmask;
    const int coff = (int)((key & qmask) * (NA * 32 * NB * (uint32_t)sizeof(float)));
    const int poff = (int)(y0l * G::RW + x0l);
    const int last_poff = __shfl_sync(0xffffffffu, poff, cnt - 1);
    const bool pad = lane >= cnt;
    const float4 ra = raw[lane * 3], rb = raw[lane * 3 + 1];
    const float w = p.weight ? raw[lane * 3 + 2].x : 1.0f;
    const float4 a = make_float4(ra.x * w, ra.y * w, ra.z * w, ra.w * w);
    const float4 b = make_float4(rb.x * w, rb.y * w, rb.z * w, rb.w * w);
    const float4 m = make_float4(__int_as_float(pad ? 0 : coff), __int_as_float(pad ? last_poff : poff), 0.f, 0.f);
    float4 *slot = half + lane * 3;
    slot[0] = a; slot[1] = b; slot[2] = m;
    if (lane < 3) {
        float4 *e = other_ext + lane * 3;
        e[0] = a; e[1] = b; e[2] = m;
    }
}

template <int NB> struct CoefVec;
template <> struct CoefVec<4> {
    float c[4];
    __device__ __forceinline__ void load(const float *p) {
        const float4 v = *reinterpret_cast<const float4 *>(p);
        c[0] = v.x; c[1] = v.y; c[2] = v.z; c[3] = v.w;
    }
};
template <> struct CoefVec<2> {
    float c[2];
    __device__ __forceinline__ void load(const float *p) {
        const float2 v = *reinterpret_cast<const float2 *>(p);
        c[0] = v.x; c[1] = v.y;
    }
};

// One staged record in registers: the weighted visibility (broadcast loads) and this lane's taps.
template <int NA, int NB>
struct RecRegs {
    float4 va, vb;
    CoefVec<NB> c[NA];
    // `coff` = table byte offset of the record in `slot`, loaded one record earlier (load_meta), so
    // that no address here waits on a load issued in the same step.
    __device__ __forceinline__ void fetch(const float4 *slot, const int coff, const char *coef_lane) {
        va = slot[0];
        vb = slot[1];
        const float *cp = reinterpret_cast<const float *>(coef_lane + coff);
#pragma unroll
        for (int a = 0; a < NA; ++a) c[a].load(cp + a * 32 * NB);
    }
};

__device__ __forceinline__ int2 load_meta(const float4 *slot) {
    const float2 m = *reinterpret_cast<const float2 *>(slot + 2);
    return make_int2(__float_as_int(m.x), __float_as_int(m.y));
}

// Two-level accumulation: the register patch holds a short FP32 chain (one run
// of equal patch origins, at most 64 entries); it is then ADDED to the shared region and cleared.
// A long single chain is not good enough: neighbouring channels of one baseline give nearly equal
// terms, whose rounding errors do not cancel (measured 1.2e-5 relative at 2048 terms).
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

template <int NA, int NB, int RW>
__device__ __forceinline__ void consume(const RecRegs<NA, NB> &R, const int poff, int &cur, float4 *regA,
                                        float4 *regB, int lane_cell, float (&acc)[NA][NB][8]) {
    if (poff != cur) {                                      // warp-uniform
        if (cur >= 0) fold_patch<NA, NB, RW>(regA, regB, cur + lane_cell, acc);
        cur = poff;
    }
    const float v[8] = {R.va.x, R.va.y, R.va.z, R.va.w, R.vb.x, R.vb.y, R.vb.z, R.vb.w};
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int k = 0; k < 8; ++k) acc[a][b][k] = fmaf(R.c[a].c[b], v[k], acc[a][b][k]);
}

template <int NA, int NB, int TLOG, int WARPS>
__global__ void __launch_bounds__(WARPS * 32, 1) grid_kernel(const GridParams p) {
    using G = Geo<NA, NB, TLOG>;
    extern __shared__ float4 smem[];
    float4 *coef4 = smem;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    float4 *region = smem + p.coef_f4 + warp * G::WARP_F4;     // plane A then plane B
    float4 *regA = region, *regB = region + G::CELLS;
    float4 *stage = region + 2 * G::CELLS;                     // record ring: 2 halves x 35 slots x 3 float4
    float4 *raw = stage + G::STAGE_F4;                         // cp.async landing buffer

    for (int i = threadIdx.x; i < p.coef_f4; i += WARPS * 32) coef4[i] = p.coef[i];
    // the ring is cleared too: records are fetched one ahead, also past the end of an item, and
    // whatever a slot holds must be a valid table offset
    for (int i = lane; i < G::WARP_F4; i += 32) region[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncthreads();

    const unsigned int n_items = p.counters_ro->n_items;
    const int lane_cell = (lane >> 3) * G::RW + (lane & 7);      // tap (a=0, b=0) of this lane
    const char *coef_lane = reinterpret_cast<const char *>(smem) + lane * NB * sizeof(float);

    float acc[NA][NB][8];
#pragma unroll
    for (int a = 0; a < NA; ++a)
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
            for (int k = 0; k < 8; ++k) acc[a][b][k] = 0.f;

    while (true) {
        unsigned int item = 0;
        if (lane == 0) item = atomicAdd(&p.counters->queue_head, 1u);
        item = __shfl_sync(0xffffffffu, item, 0);
        if (item >= n_items) break;
        const WorkItem wi = p.items[item];
        const int len = (int)wi.len;

        const int n_batches = (len + 31) >> 5;

        // prologue: batch 0 staged, batch 1's visibilities (cp.async) and batch 2's keys in flight
        uint32_t key_landing;                                   // key of the batch in the raw buffer
        KeyIdx ki_next;                                         // batch after that
        {
            const KeyIdx k0 = load_keyidx(p, wi.start + lane, lane < len);
            const KeyIdx k1 = load_keyidx(p, wi.start + 32 + lane, 32 + lane < len);
            ki_next = load_keyidx(p, wi.start + 64 + lane, 64 + lane < len);
            issue_vis(p, raw, lane, k0, lane < len);
            cp_async_wait_all();
            stage_write<NA, NB, TLOG>(p, raw, stage, stage + (G::HALF_SLOTS + 32) * 3, lane, min(32, len), k0.key);
            issue_vis(p, raw, lane, k1, 32 + lane < len);
            key_landing = k1.key;
        }
        __syncwarp();

        // The loop body handles four records so that every prefetched (table offset, origin) pair
        // lands in a register nobody else is still reading: no copy waits on a load just issued.
        RecRegs<NA, NB> A, B;
        int2 mA = load_meta(stage);
        A.fetch(stage, mA.x, coef_lane);
        int2 mB = load_meta(stage + 3);
        int cur = -1;
        for (int jb = 0; jb < n_batches; ++jb) {
            float4 *half = stage + (jb & 1) * (G::HALF_SLOTS * 3);
            float4 *other = stage + ((jb + 1) & 1) * (G::HALF_SLOTS * 3);
            const int n_quads = (min(32, len - 32 * jb) + 3) >> 2;
            const float4 *sp = half;
            auto quad_step = [&]() {
                // in: A = record 0 (origin mA.y), mB = meta of record 1
                const int2 mC = load_meta(sp + 6);
                B.fetch(sp + 3, mB.x, coef_lane);
                consume<NA, NB, G::RW>(A, mA.y, cur, regA, regB, lane_cell, acc);
                const int2 mD = load_meta(sp + 9);
                A.fetch(sp + 6, mC.x, coef_lane);
                consume<NA, NB, G::RW>(B, mB.y, cur, regA, regB, lane_cell, acc);
                mA = load_meta(sp + 12);
                B.fetch(sp + 9, mD.x, coef_lane);
                consume<NA, NB, G::RW>(A, mC.y, cur, regA, regB, lane_cell, acc);
                mB = load_meta(sp + 15);
                A.fetch(sp + 12, mA.x, coef_lane);
                consume<NA, NB, G::RW>(B, mD.y, cur, regA, regB, lane_cell, acc);
                sp += 12;
            };
            const int first = min(n_quads, 4);
            for (int i = 0; i < first; ++i) quad_step();
            // mid-batch (warp-uniform): bound the register chain, then move the staging pipeline on
            if ((jb & p.fold_mask) == p.fold_mask && cur >= 0) {
                fold_patch<NA, NB, G::RW>(regA, regB, cur + lane_cell, acc);
                cur = -1;
            }
            if (jb + 1 < n_batches) {
                __syncwarp();                                   // the other half was last read in batch jb-1
                cp_async_wait_all();
                stage_write<NA, NB, TLOG>(p, raw, other, half + 32 * 3, lane, min(32, len - 32 * (jb + 1)), key_landing);
                __syncwarp();
                const int o2 = (jb + 2) * 32 + lane, o3 = (jb + 3) * 32 + lane;
                if ((jb + 2) * 32 < len) {
                    issue_vis(p, raw, lane, ki_next, o2 < len);
                    key_landing = ki_next.key;
                    ki_next = load_keyidx(p, wi.start + o3, o3 < len);
                }
            }
            for (int i = 4; i < n_quads; ++i) quad_step();
        }
        // fold the last patch in, then move the region to this item's partial and clear it
        if (cur >= 0) fold_patch<NA, NB, G::RW>(regA, regB, cur + lane_cell, acc);
        __syncwarp();
        float4 *dst = p.partials + (size_t)item * (2 * G::CELLS);
        for (int i = lane; i < 2 * G::CELLS; i += 32) {
            stg_stream(dst + i, region[i]);
            region[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        __syncwarp();
    }
}

// ------------------------------------------------------------------------------------------
// Flush: one thread per grid cell.  The partial regions covering cell (x, y) belong to the tiles
// (ty, tx) with tx*T <= x < tx*T + RW (same in y); each tile's work items are added in id order
// (full chunks, then the tail).  FP64 accumulation, one rounding to FP32 at the end.
// ------------------------------------------------------------------------------------------
template <int NA, int NB, int TLOG>
__global__ void __launch_bounds__(256) flush_kernel(const FlushParams p) {
    using G = Geo<NA, NB, TLOG>;
    const int x = blockIdx.x * 32 + threadIdx.x;
    const int y = blockIdx.y * 8 + threadIdx.y;
    if (x >= p.n_grid || y >= p.n_grid) return;
    double acc[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) acc[k] = 0.0;
    const int tx_hi = min(x >> TLOG, p.ntx - 1), ty_hi = min(y >> TLOG, p.nty - 1);
    const int tx_lo = max(0, (x - G::RW + G::T) >> TLOG), ty_lo = max(0, (y - G::RH + G::T) >> TLOG);
    for (int ty = ty_lo; ty <= ty_hi; ++ty)
        for (int tx = tx_lo; tx <= tx_hi; ++tx) {
            const TileInfo ti = p.tiles[ty * p.ntx + tx];
            if (ti.count == 0) continue;
            const int cell = (y - (ty << TLOG)) * G::RW + (x - (tx << TLOG));
            const uint32_t n_it = ti.n_full + (ti.tail_item != 0xFFFFFFFFu ? 1u : 0u);
            for (uint32_t c = 0; c < n_it; ++c) {
                const uint32_t item = c < ti.n_full ? ti.full_base + c : ti.tail_item;
                const float4 *part = p.partials + (size_t)item * (2 * G::CELLS);
                const float4 a = __ldcs(part + cell), b = __ldcs(part + G::CELLS + cell);
                acc[0] += (double)a.x; acc[1] += (double)a.y; acc[2] += (double)a.z; acc[3] += (double)a.w;
                acc[4] += (double)b.x; acc[5] += (double)b.y; acc[6] += (double)b.z; acc[7] += (double)b.w;
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
// Host side: kernel selection.  NA x NB is fixed by the padded patch (16: 2x4, 8: 1x2), TLOG and
// the number of warps per block are plan parameters.
// ------------------------------------------------------------------------------------------
size_t grid_smem_bytes(int NA, int NB, int tlog, int oversample, int warps) {
    const int T = 1 << tlog;
    const int RW = T + 8 * NA - 1, RH = T + 4 * NB - 1;
    const size_t coef = (size_t)oversample * oversample * NA * NB * 32 * sizeof(float);
    const size_t per_warp = (size_t)(2 * RW * RH + 2 * (32 + 3) * 3 + 32 * 3) * sizeof(float4);   // Geo::WARP_F4
    return coef + per_warp * warps;
}

typedef void (*grid_fn_t)(const GridParams);
typedef void (*flush_fn_t)(const FlushParams);

template <int NA, int NB, int TLOG>
static grid_fn_t pick_warps(int warps) {
    switch (warps) {
        case 4: return grid_kernel<NA, NB, TLOG, 4>;
        case 6: return grid_kernel<NA, NB, TLOG, 6>;
        case 8: return grid_kernel<NA, NB, TLOG, 8>;
        case 10: return grid_kernel<NA, NB, TLOG, 10>;
        case 12: return grid_kernel<NA, NB, TLOG, 12>;
        case 16: return grid_kernel<NA, NB, TLOG, 16>;
        default: return nullptr;
    }
}

static grid_fn_t pick_grid(int NA, int tlog, int warps) {
    if (NA == 2) {
        if (tlog == 2) return pick_warps<2, 4, 2>(warps);
        if (tlog == 3) return pick_warps<2, 4, 3>(warps);
        if (tlog == 4) return pick_warps<2, 4, 4>(warps);
    } else {
        if (tlog == 2) return pick_warps<1, 2, 2>(warps);
        if (tlog == 3) return pick_warps<1, 2, 3>(warps);
        if (tlog == 4) return pick_warps<1, 2, 4>(warps);
    }
    return nullptr;
}

static flush_fn_t pick_flush(int NA, int tlog) {
    if (NA == 2) {
        if (tlog == 2) return flush_kernel<2, 4, 2>;
        if (tlog == 3) return flush_kernel<2, 4, 3>;
        if (tlog == 4) return flush_kernel<2, 4, 4>;
    } else {
        if (tlog == 2) return flush_kernel<1, 2, 2>;
        if (tlog == 3) return flush_kernel<1, 2, 3>;
        if (tlog == 4) return flush_kernel<1, 2, 4>;
    }
    return nullptr;
}

static const int kWarpChoices[] = {16, 12, 10, 8, 6, 4};

cudaError_t configure_grid_kernel(Plan &p) {
    int dev = 0, smem_max = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&smem_max, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e != cudaSuccess) return e;
    int chosen = 0;
    for (int w : kWarpChoices) {
        if (p.warps > 0 && w != p.warps) continue;             // forced by the caller (tuning)
        if (grid_smem_bytes(p.NA, p.NB, p.tlog, p.cfg.oversample, w) <= (size_t)smem_max) { chosen = w; break; }
    }
    if (!chosen) return cudaErrorInvalidConfiguration;
    p.warps = chosen;
    p.smem_bytes = (int)grid_smem_bytes(p.NA, p.NB, p.tlog, p.cfg.oversample, chosen);
    grid_fn_t fn = pick_grid(p.NA, p.tlog, p.warps);
    if (!fn) return cudaErrorInvalidConfiguration;
    return cudaFuncSetAttribute((const void *)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, p.smem_bytes);
}

cudaError_t launch_grid(Plan &p, const float *vis, const float *weight, float *grid, int accumulate,
                        cudaStream_t s) {
    grid_fn_t gfn = pick_grid(p.NA, p.tlog, p.warps);
    flush_fn_t ffn = pick_flush(p.NA, p.tlog);
    if (!gfn || !ffn) return cudaErrorInvalidConfiguration;
    stage_mark(p, 4, s);
    // reset the work queue (bin leaves it at 0, a previous grid call leaves it past the end)
    cudaError_t e = cudaMemsetAsync(&p.counters->queue_head, 0, sizeof(unsigned int), s);
    if (e != cudaSuccess) return e;
    GridParams gp;
    gp.keys = p.keys[p.sorted_sel];
    gp.vals = p.vals[p.sorted_sel];
    gp.items = p.items;
    gp.counters_ro = p.counters;
    gp.counters = p.counters;
    gp.vis = reinterpret_cast<const float4 *>(vis);
    gp.weight = weight;
    gp.coef = p.coef;
    gp.partials = p.partials;
    gp.coef_f4 = p.coef_f4;
    gp.key = p.key;
    gp.fold_mask = p.fold_batches - 1;
    gfn<<<p.n_sm, p.warps * 32, p.smem_bytes, s>>>(gp);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    stage_mark(p, 5, s);
    FlushParams fp;
    fp.tiles = p.tile_info;
    fp.counters = p.counters;
    fp.partials = p.partials;
    fp.grid = reinterpret_cast<float2 *>(grid);
    fp.n_grid = p.cfg.grid_size;
    fp.ntx = p.ntx;
    fp.nty = p.nty;
    fp.accumulate = accumulate;
    dim3 blk(32, 8), grd((p.cfg.grid_size + 31) / 32, (p.cfg.grid_size + 7) / 8);
    ffn<<<grd, blk, 0, s>>>(fp);
    e = cudaGetLastError();
    stage_mark(p, 6, s);
    if (p.profiling) p.prof_grid_calls++;
    p.n_launches += 2;
    return e;
}

}  // namespace gridder
