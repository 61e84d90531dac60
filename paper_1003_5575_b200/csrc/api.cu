// The C ABI of include/gridder.h: plan management, argument checks, error codes.
#include <cstdio>
#include <cstring>
#include <new>

#include "gridder_internal.cuh"

using namespace gridder;

namespace {

size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

int ceil_log2(unsigned long long v) {   // smallest b with 2^b >= v
    int b = 0;
    while ((1ull << b) < v) ++b;
    return b;
}

// Everything that follows from the config and the tuning alone (no device access).
int derive(const gridder_config *cfg, const gridder_tuning *tuning, Plan &p) {
    if (!cfg) return GRIDDER_ERR_INVALID_ARG;
    if (cfg->grid_size < 2 || (cfg->grid_size & 1) || cfg->grid_size > 32768) return GRIDDER_ERR_INVALID_ARG;
    if (!(cfg->cell_size > 0.0) || cfg->n_pol != 4) return GRIDDER_ERR_INVALID_ARG;
    if (cfg->oversample < 1 || cfg->oversample > 64) return GRIDDER_ERR_INVALID_ARG;
    if (cfg->n_wplanes < 1 || cfg->n_wplanes > kMaxPlanes || !cfg->support) return GRIDDER_ERR_INVALID_ARG;
    if (cfg->max_vis < 0 || cfg->max_vis > 0xFFFFF000ll) return GRIDDER_ERR_INVALID_ARG;
    for (int i = 0; i < cfg->n_wplanes; ++i) {
        const int s = cfg->support[i];
        if (s < 1 || s > 32 || ((s * cfg->oversample) & 1)) return GRIDDER_ERR_INVALID_ARG;
        if (s > cfg->grid_size) return GRIDDER_ERR_INVALID_ARG;
    }
    if (cfg->n_wplanes > 1 && !(cfg->w_max > 0.0)) return GRIDDER_ERR_INVALID_ARG;
    gridder_tuning t;
    memset(&t, 0, sizeof(t));
    if (tuning) t = *tuning;
    if ((t.tile_log2 != 0 && (t.tile_log2 < 2 || t.tile_log2 > 4)) || (t.chunk != 0 && (t.chunk < 32 || t.chunk > (1 << 20))) ||
        t.max_warps < 0 || t.merge < 0 || t.merge > 2 || t.presum < 0 || t.presum > 2 || t.table_in_tmem < 0 ||
        t.table_in_tmem > 2 || t.fold_batches < 0 || t.fold_batches > 64 || (t.fold_batches & (t.fold_batches - 1)) ||
        t.force_general < 0 || t.force_general > 1 || t.host_slices < 0 || t.host_slices > 64 || t.host_slice_min_mb < 0)
        return GRIDDER_ERR_INVALID_ARG;
    for (int i = 0; i < 6; ++i)
        if (t.reserved[i]) return GRIDDER_ERR_INVALID_ARG;

    p.cfg = *cfg;
    p.tune = t;
    memcpy(p.support_copy, cfg->support, sizeof(int32_t) * cfg->n_wplanes);
    p.cfg.support = p.support_copy;
    const bool cplx = cfg->kernel_is_complex != 0;
    const size_t oo = (size_t)cfg->oversample * cfg->oversample;
    const int q_bits = ceil_log2((unsigned long long)cfg->oversample);
    p.merge = t.merge == 2 ? 0 : 1;
    // fast path: one real table with S <= 16 (table in shared or tensor memory, 32-bit sort values)
    p.mode = cplx ? 2 : ((cfg->n_wplanes == 1 && cfg->support[0] <= 16 && !t.force_general) ? 0 : 1);
    // PRE-SUMMATION IN INPUT ORDER (presum.cu): fast path, merging allowed (a per-visibility GCF forbids it),
    // sub-cell offsets and drop flag in one byte.  By default for plans of 1 Mi visibilities and more: below
    // that sorting every visibility is cheap and the one host synchronisation it costs gridder_bin is not.
    // Whether an input then really takes it is decided per gridder_bin, from its shape and the number of partial
    // records the plan kernel COUNTED (the data, not the capacity): see launch_bin.
    p.presum = (p.mode == 0 && p.merge && 2 * q_bits + 1 <= 8 &&
                (t.presum == 1 || (t.presum == 0 && cfg->max_vis >= (1ll << 20)))) ? 1 : 0;
    // (its mapper packs the two lattice coordinates of a visibility into 16 bits each: map.cuh FastMap2::lat)
    if ((int64_t)cfg->grid_size * cfg->oversample + cfg->oversample >= 65533) p.presum = 0;
    p.tlog = t.tile_log2 ? t.tile_log2 : ((p.presum || p.mode != 0) ? 3 : 2);
    p.T = 1 << p.tlog;
    p.ntx = (cfg->grid_size + p.T - 1) / p.T;
    p.nty = p.ntx;
    p.n_tiles = p.ntx * p.nty;
    if (cfg->max_grids < 0 || cfg->max_grids > 4096) return GRIDDER_ERR_INVALID_ARG;
    p.max_grids = cfg->max_grids > 1 ? cfg->max_grids : 1;
    if ((int64_t)p.n_tiles * p.max_grids > (1ll << 30)) return GRIDDER_ERR_UNSUPPORTED;
    p.n_tiles_cls = p.n_tiles * p.max_grids;
    p.n_grids = 1;
    // the fast path keeps the sub-cell offsets in the 32-bit sort key; a grid too large for that
    // (2 log2 N + 2 log2 O + 1 > 32 bits) goes through the general path, whose values carry them
    if (p.mode == 0 && 2 * q_bits + 1 + 2 * p.tlog + ceil_log2((unsigned long long)p.n_tiles_cls) > 32) {
        p.mode = 1;
        p.presum = 0;
    }

    // patch classes in use (ascending), and each plane's slot and table offset
    int slot_of_class[kMaxClasses] = {-1, -1, -1};
    bool used[kMaxClasses] = {false, false, false};
    for (int i = 0; i < cfg->n_wplanes; ++i) {
        const int s = cfg->support[i];
        used[s <= 8 ? 0 : (s <= 16 ? 1 : 2)] = true;
    }
    p.n_cls = 0;
    for (int c = 0; c < kMaxClasses; ++c) {
        if (!used[c]) continue;
        ClassGeo g;
        memset(&g, 0, sizeof(g));
        g.NA = c == 0 ? 1 : 2;
        g.NB = c == 0 ? 2 : 4;
        g.nsub = c == 2 ? 2 : 1;
        g.SP = 8 * g.NA * g.nsub;
        g.RW = g.RH = p.T + 8 * g.NA - 1;            // region of ONE register patch (tile + halo)
        g.sub_bytes = g.NA * g.NB * 32 * (cplx ? 8 : 4);
        g.region_f4 = g.nsub * g.nsub * 2 * g.RW * g.RH;     // nsub^2 virtual items per work item
        slot_of_class[c] = p.n_cls;
        p.cls[p.n_cls++] = g;
    }
    size_t off = 0;
    for (int i = 0; i < cfg->n_wplanes; ++i) {
        const int s = cfg->support[i];
        p.plane_slot[i] = slot_of_class[s <= 8 ? 0 : (s <= 16 ? 1 : 2)];
        const ClassGeo &g = p.cls[p.plane_slot[i]];
        p.plane_off256[i] = (uint32_t)(off / 256);
        off += (size_t)g.nsub * g.nsub * oo * g.sub_bytes;
    }
    if (off >= (1ull << 31)) return GRIDDER_ERR_UNSUPPORTED;       // table offsets are 32-bit byte offsets
    p.coef_bytes = off;
    // a fast-path table that cannot sit in shared memory beside one warp's region (e.g. S = 16 with O = 16:
    // 256 KB) is read from global memory instead: the general path
    if (p.mode == 0 && p.coef_bytes + 24 * 1024 > 227 * 1024) {
        p.mode = 1;
        p.presum = 0;
    }

    // fast path: the table in tensor memory (512 columns x 32 bit per lane) when it fits.  Measured on B200:
    // same speed as the shared-memory table while the kernel is FMA-bound, faster on the records of a
    // pre-summed plan, where the shared-memory path is the busiest unit: on by default there.
    p.tmem_cols = 0;
    if (p.mode == 0 && (t.table_in_tmem == 1 || (t.table_in_tmem == 0 && p.presum))) {
        const size_t cols = oo * p.cls[0].NA * p.cls[0].NB;
        if (cols <= 512) {
            p.tmem_cols = 32;
            while ((size_t)p.tmem_cols < cols) p.tmem_cols *= 2;
        }
    }
    // K: most entries per work item, ~ max_vis / 2^14 as a power of two in [256, 4096]: small inputs get
    // short items so that a hot tile still spreads over the ~1800 resident warps; larger K means fewer partial
    // regions for the flush, smaller K a better balanced end of the grid kernel (warps claim one item at a time);
    // measured on configs 3 and 4, 2048 .. 8192 are within 1 % of each other (the accuracy budget of DESIGN.md
    // section 7 holds up to 8192)
    int k_auto = 4096;
    while (k_auto > 256 && (int64_t)k_auto * 16384 > cfg->max_vis) k_auto >>= 1;
    p.chunk = t.chunk ? t.chunk : k_auto;
    p.warps_forced = t.max_warps;
    // per-origin bins carried across the batches of the grid kernel (grid.cu stage_write_bins)
    p.bins = (p.merge && oo <= 16) ? 1 : 0;
    p.fold_batches = t.fold_batches ? t.fold_batches : 8;

    KeyLayout k;
    k.bits_q = q_bits;
    k.tlog = p.tlog;
    k.aux_bits = p.mode == 0 ? 2 * k.bits_q + 1 : 0;
    k.plane_shift = k.aux_bits + 2 * k.tlog;
    k.plane_bits = cfg->n_wplanes > 1 ? ceil_log2((unsigned long long)cfg->n_wplanes) : 0;
    k.tile_bits = ceil_log2((unsigned long long)p.n_tiles_cls * p.n_cls);
    if (k.tile_bits < 1) k.tile_bits = 1;
    // sorting on the plane inside a tile only helps table locality: dropped when the key is full
    if (k.plane_shift + k.plane_bits + k.tile_bits > 32) k.plane_bits = 0;
    k.tile_shift = k.plane_shift + k.plane_bits;
    k.total_bits = k.tile_shift + k.tile_bits;
    if (k.total_bits > 32) return GRIDDER_ERR_UNSUPPORTED;
    p.key = k;
    // general path: a carried run is (plane, origin), so the sort must keep the entries of a plane together
    if (p.mode != 0 && ((cfg->n_wplanes > 1 && k.plane_bits == 0) || k.tile_shift > 26)) p.bins = 0;

    const int64_t n = cfg->max_vis;
    const int64_t n_vtiles = (int64_t)p.n_tiles_cls * p.n_cls;
    int64_t occ = n < n_vtiles ? n : n_vtiles;
    p.max_items = occ + n / p.chunk + 1;
    // each class has its own partial-region array, sized for the case that every entry is of that class
    p.max_items_cls = (n < p.n_tiles_cls ? n : p.n_tiles_cls) + n / p.chunk + 1;
    if (p.presum) {
        // The sums of a group's partial records live in the group's own visibility slots (presum.cu slot_index), so
        // they need an array as large as the visibilities.  Inputs that merge into more than 3/4 n records take the per-visibility path (decided
        // per gridder_bin from the count the plan kernel returns).  The plan kernel stages the record keys in the
        // sort's second key buffer.
        p.ps_cap = n * 3 / 4 + 1024;
        p.ps_group_cap = n / 8 + 1024;
    }
    p.partials_f4 = 0;
    for (int c = 0; c < p.n_cls; ++c) {
        p.cls[c].part_off_f4 = p.partials_f4;
        p.partials_f4 += p.max_items_cls * p.cls[c].region_f4;
    }
    return GRIDDER_OK;
}

// Lay the workspace out; with base == nullptr only the size is computed.
cudaError_t carve(Plan &p, char *base) {
    size_t off = 0;
    auto take = [&](size_t bytes) { char *ptr = base ? base + off : nullptr; off += align_up(bytes); return ptr; };
    const size_t n = (size_t)(p.cfg.max_vis > 0 ? p.cfg.max_vis : 1);
    const size_t n_vtiles = (size_t)p.n_tiles_cls * p.n_cls;
    const size_t val_bytes = p.mode == 0 ? sizeof(uint32_t) : sizeof(unsigned long long);
    // (keys[1] and vals[1] next to each other: together they are the staging area of the pre-summed plans)
    p.keys[0] = (uint32_t *)take(n * sizeof(uint32_t));
    p.vals[0] = (void *)take(n * val_bytes);
    p.keys[1] = (uint32_t *)take(n * sizeof(uint32_t));
    p.vals[1] = (void *)take(n * val_bytes);
    size_t t1 = 0, t2 = 0;
    cudaError_t e = sort_temp_bytes((int64_t)n, p.key.aux_bits, p.key.total_bits, p.mode != 0, &t1);
    if (e == cudaSuccess) e = scan_temp_bytes((int64_t)n_vtiles + 1, &t2);
    if (e == cudaSuccess && p.presum) {
        size_t t3 = 0;
        e = presum_scan_temp_bytes(p.ps_group_cap + 1, &t3);
        if (t3 > t2) t2 = t3;
    }
    if (e == cudaErrorNoDevice || e == cudaErrorInsufficientDriver || e == cudaErrorInvalidDevice) {
        // no GPU on this machine (size query only): CUB cannot be asked, so report a generous bound
        (void)cudaGetLastError();
        t1 = ((size_t)32 << 20) + n / 2;
        t2 = (size_t)1 << 20;
        e = cudaSuccess;
    }
    if (e != cudaSuccess) return e;
    p.cub_temp_bytes = align_up(t1 > t2 ? t1 : t2);
    p.cub_temp = take(p.cub_temp_bytes);
    p.freq_scale = (double *)take(sizeof(double) * kMaxChannels);
    p.tile_start = (uint32_t *)take(sizeof(uint32_t) * 2 * n_vtiles);        // [start | end]
    p.tile_chunks = (unsigned long long *)take(sizeof(unsigned long long) * (n_vtiles + 1));
    p.tile_chunks_scan = (unsigned long long *)take(sizeof(unsigned long long) * (n_vtiles + 1));
    p.tile_info = (TileInfo *)take(sizeof(TileInfo) * n_vtiles);
    p.tile_cover = (unsigned char *)take((size_t)p.n_tiles);
    p.items = (WorkItem *)take(sizeof(WorkItem) * (size_t)p.max_items);
    p.partials = (float4 *)take(sizeof(float4) * (size_t)p.partials_f4);
    if (p.presum) {
        p.ps_flags = (unsigned char *)take(n);
        p.ps_count = (uint32_t *)take(sizeof(uint32_t) * (size_t)(p.ps_group_cap + 1));
        p.ps_base = (uint32_t *)take(sizeof(uint32_t) * (size_t)(p.ps_group_cap + 1));
        p.ps_sum = (float4 *)take(sizeof(float4) * 2 * n);
    }
    p.coef = (float4 *)take(p.coef_bytes);
    p.counters = (Counters *)take(sizeof(Counters));
    p.workspace_needed = off;
    return cudaSuccess;
}

// GRIDDER_CHECKED builds: failed index checks of all plans of this process (see gridder_internal.cuh GR_CHECK)
long long g_check_violations = 0;

// Adds the device counter of the plan's last bin / grid to the process total (synchronises the device).
void collect_violations(Plan *p) {
#ifdef GRIDDER_CHECKED
    if (!p || !p->counters) return;
    unsigned int v = 0;
    if (cudaDeviceSynchronize() == cudaSuccess &&
        cudaMemcpy(&v, &p->counters->violations, sizeof(v), cudaMemcpyDeviceToHost) == cudaSuccess && v) {
        g_check_violations += v;
        cudaMemset(&p->counters->violations, 0, sizeof(v));
    }
#else
    (void)p;
#endif
}

int cuda_fail(Plan *p, cudaError_t e) {
    if (p) p->last_cuda_error = (int)e;
    return GRIDDER_ERR_CUDA;
}

}  // namespace

extern "C" {

int gridder_workspace_size(const gridder_config *cfg, size_t *bytes_needed) {
    return gridder_workspace_size_tuned(cfg, nullptr, bytes_needed);
}

int gridder_plan(const gridder_config *cfg, gridder_plan_t **plan_out, size_t *workspace_needed) {
    return gridder_plan_tuned(cfg, nullptr, plan_out, workspace_needed);
}

int gridder_workspace_size_tuned(const gridder_config *cfg, const gridder_tuning *tuning, size_t *bytes_needed) {
    if (!bytes_needed) return GRIDDER_ERR_INVALID_ARG;
    Plan p;
    memset(&p, 0, sizeof(p));
    const int rc = derive(cfg, tuning, p);
    if (rc != GRIDDER_OK) return rc;
    if (carve(p, nullptr) != cudaSuccess) return GRIDDER_ERR_CUDA;
    *bytes_needed = p.workspace_needed;
    return GRIDDER_OK;
}

int gridder_plan_tuned(const gridder_config *cfg, const gridder_tuning *tuning, gridder_plan_t **plan_out,
                       size_t *workspace_needed) {
    if (!plan_out) return GRIDDER_ERR_INVALID_ARG;
    *plan_out = nullptr;
    Plan *p = new (std::nothrow) Plan;
    if (!p) return GRIDDER_ERR_INVALID_ARG;
    memset(p, 0, sizeof(Plan));
    int rc = derive(cfg, tuning, *p);
    if (rc != GRIDDER_OK) { delete p; return rc; }
    if (carve(*p, nullptr) != cudaSuccess) { delete p; return GRIDDER_ERR_CUDA; }
    if (workspace_needed) *workspace_needed = p->workspace_needed;
    if (!cfg->kernel || !cfg->workspace || ((uintptr_t)cfg->workspace & 255)) { delete p; return GRIDDER_ERR_INVALID_ARG; }
    if (cfg->workspace_bytes < p->workspace_needed) { delete p; return GRIDDER_ERR_WORKSPACE; }
    if (carve(*p, (char *)cfg->workspace) != cudaSuccess) { delete p; return GRIDDER_ERR_CUDA; }

    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&p->n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = configure_grid_kernel(*p);
    if (e == cudaSuccess) e = launch_relayout(*p, 0);
    if (e == cudaSuccess) e = cudaMemsetAsync(p->counters, 0, sizeof(Counters), 0);
    if (e == cudaSuccess) e = cudaStreamSynchronize(0);
    if (e != cudaSuccess) { delete p; return GRIDDER_ERR_CUDA; }
    *plan_out = reinterpret_cast<gridder_plan_t *>(p);
    return GRIDDER_OK;
}

int gridder_bin(gridder_plan_t *plan, const double *uvw_m, int32_t n_time, int32_t n_baseline,
                const double *freq_hz, int32_t n_chan, void *cuda_stream) {
    return gridder_bin_tables(plan, uvw_m, n_time, n_baseline, freq_hz, n_chan, nullptr, cuda_stream);
}

static int bin_common(gridder_plan_t *plan, const double *uvw_m, int32_t n_time, int32_t n_baseline, const double *freq_hz,
                      int32_t n_chan, const int32_t *table_index, int32_t chans_per_grid, void *cuda_stream);

int gridder_bin_tables(gridder_plan_t *plan, const double *uvw_m, int32_t n_time, int32_t n_baseline,
                       const double *freq_hz, int32_t n_chan, const int32_t *table_index, void *cuda_stream) {
    return bin_common(plan, uvw_m, n_time, n_baseline, freq_hz, n_chan, table_index, 0, cuda_stream);
}

int gridder_bin_channels(gridder_plan_t *plan, const double *uvw_m, int32_t n_time, int32_t n_baseline,
                         const double *freq_hz, int32_t n_chan, int32_t chans_per_grid, void *cuda_stream) {
    if (chans_per_grid < 1) return GRIDDER_ERR_INVALID_ARG;
    return bin_common(plan, uvw_m, n_time, n_baseline, freq_hz, n_chan, nullptr, chans_per_grid, cuda_stream);
}

static int bin_common(gridder_plan_t *plan, const double *uvw_m, int32_t n_time, int32_t n_baseline, const double *freq_hz,
                      int32_t n_chan, const int32_t *table_index, int32_t chans_per_grid, void *cuda_stream) {
    Plan *p = reinterpret_cast<Plan *>(plan);
    if (!p || n_time < 0 || n_baseline < 0 || n_chan < 0) return GRIDDER_ERR_INVALID_ARG;
    const int32_t n_grids = chans_per_grid > 0 && n_chan > 0 ? (n_chan + chans_per_grid - 1) / chans_per_grid : 1;
    if (n_grids > p->max_grids) return GRIDDER_ERR_CAPACITY;
    const int64_t n = (int64_t)n_time * n_baseline * n_chan;
    if (n > 0 && (!uvw_m || !freq_hz)) return GRIDDER_ERR_INVALID_ARG;
    if (n > p->cfg.max_vis) return GRIDDER_ERR_CAPACITY;
    if (n_chan > kMaxChannels) return GRIDDER_ERR_UNSUPPORTED;
    collect_violations(p);           // (the bin resets the device counters)
    p->binned = false;
    p->n_grids = n_grids;
    p->chans_per_grid = chans_per_grid;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaError_t e = launch_bin(*p, uvw_m, n_time, n_baseline, freq_hz, n_chan, table_index, s);
    if (e != cudaSuccess) return cuda_fail(p, e);
    p->n_vis = n;
    p->binned = true;
    p->last_stream = s;
    return GRIDDER_OK;
}

int gridder_grid(gridder_plan_t *plan, const float *vis, const float *weight, float *grid,
                 int32_t accumulate, void *cuda_stream) {
    Plan *p = reinterpret_cast<Plan *>(plan);
    if (p && p->binned && p->n_grids > 1) return GRIDDER_ERR_INVALID_ARG;       // binned for several grids
    return gridder_grid_channels(plan, vis, weight, grid, accumulate, cuda_stream);
}

int gridder_grid_channels(gridder_plan_t *plan, const float *vis, const float *weight, float *grid,
                          int32_t accumulate, void *cuda_stream) {
    Plan *p = reinterpret_cast<Plan *>(plan);
    if (!p || !grid) return GRIDDER_ERR_INVALID_ARG;
    if (!p->binned) return GRIDDER_ERR_NOT_BINNED;
    if (p->n_vis > 0 && !vis) return GRIDDER_ERR_INVALID_ARG;
    if (((uintptr_t)vis & 15) || ((uintptr_t)grid & 7)) return GRIDDER_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaError_t e = launch_grid(*p, vis, weight, grid, accumulate ? 1 : 0, s);
    if (e != cudaSuccess) return cuda_fail(p, e);
    p->last_stream = s;
    return GRIDDER_OK;
}

int gridder_destroy(gridder_plan_t *plan) {
    Plan *p = reinterpret_cast<Plan *>(plan);
    if (!p) return GRIDDER_ERR_INVALID_ARG;
    cudaError_t e = cudaDeviceSynchronize();     // the caller may free the workspace after this
    collect_violations(p);
    image_destroy(*p);
    if (p->copy_stream) cudaStreamDestroy(p->copy_stream);
    if (p->count_ev) cudaEventDestroy(p->count_ev);
    for (int r = 0; r < kProfRing; ++r)
        for (int i = 0; i < 10; ++i) if (p->ev[r][i]) cudaEventDestroy(p->ev[r][i]);
    delete p;
    return e == cudaSuccess ? GRIDDER_OK : GRIDDER_ERR_CUDA;
}

int gridder_get_stats(gridder_plan_t *plan, gridder_stats *out) {
    Plan *p = reinterpret_cast<Plan *>(plan);
    if (!p || !out) return GRIDDER_ERR_INVALID_ARG;
    if (!p->binned) return GRIDDER_ERR_NOT_BINNED;
    Counters c;
    cudaError_t e = cudaMemcpyAsync(&c, p->counters, sizeof(Counters), cudaMemcpyDeviceToHost, p->last_stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->last_stream);
    if (e != cudaSuccess) return cuda_fail(p, e);
    memset(out, 0, sizeof(*out));
    out->n_vis = p->n_vis;
    out->n_dropped = (int64_t)c.n_dropped;
    out->n_entries = p->n_vis - (int64_t)c.n_dropped;
    out->vis_taps = (int64_t)c.vis_taps;
    out->n_tiles = p->n_tiles;
    out->n_tiles_occupied = c.n_occupied;      /* (class, tile) pairs when several patch classes are in use */
    out->max_tile_load = c.max_tile_load;
    out->n_work_items = c.n_items;
    out->tile_size = p->T;
    out->patch_size = p->cls[p->n_cls - 1].SP;
    out->chunk_size = p->chunk;
    out->grid_warps_per_sm = p->cls[p->n_cls - 1].warps;
    out->n_presum_records = p->presum_active ? p->n_sorted : 0;
    for (int k = 0; k < p->n_cls; ++k) {
        const ClassGeo &g = p->cls[k];
        out->n_records_gridded += (int64_t)c.n_exec[k];
        out->fma_executed += (int64_t)c.n_exec[k] * (8 * g.NA) * (4 * g.NB) * (p->cfg.kernel_is_complex ? 16 : 8);
    }
    return GRIDDER_OK;
}

int gridder_map(gridder_plan_t *plan, const double *uvw_m, int32_t n_time, int32_t n_baseline,
                const double *freq_hz, int32_t n_chan, const int32_t *table_index, int32_t *out, void *cuda_stream) {
    Plan *p = reinterpret_cast<Plan *>(plan);
    if (!p || !uvw_m || !freq_hz || !out || n_time < 0 || n_baseline < 0 || n_chan < 0)
        return GRIDDER_ERR_INVALID_ARG;
    if ((int64_t)n_time * n_baseline * n_chan == 0) return GRIDDER_OK;
    cudaError_t e = launch_map_debug(*p, uvw_m, n_time, n_baseline, freq_hz, n_chan, table_index, out,
                                     (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(p, e);
    return GRIDDER_OK;
}

int gridder_map_presum(gridder_plan_t *plan, const double *uvw_m, int32_t n_time, int32_t n_baseline,
                       const double *freq_hz, int32_t n_chan, int32_t *out, void *cuda_stream) {
    Plan *p = reinterpret_cast<Plan *>(plan);
    if (!p || !uvw_m || !freq_hz || !out || n_time < 0 || n_baseline < 0 || n_chan < 0)
        return GRIDDER_ERR_INVALID_ARG;
    if ((int64_t)n_time * n_baseline * n_chan == 0) return GRIDDER_OK;
    cudaError_t e = launch_map_presum_debug(*p, uvw_m, n_time, n_baseline, freq_hz, n_chan, out, (cudaStream_t)cuda_stream);
    if (e == cudaErrorNotSupported) return GRIDDER_ERR_UNSUPPORTED;
    if (e != cudaSuccess) return cuda_fail(p, e);
    return GRIDDER_OK;
}

int gridder_scatter_atomic(gridder_plan_t *plan, const double *uvw_m, int32_t n_time, int32_t n_baseline,
                           const double *freq_hz, int32_t n_chan, const float *vis, const float *weight, float *grid,
                           int32_t accumulate, void *cuda_stream) {
    Plan *p = reinterpret_cast<Plan *>(plan);
    if (!p || !grid || n_time < 0 || n_baseline < 0 || n_chan < 0) return GRIDDER_ERR_INVALID_ARG;
    const int64_t n = (int64_t)n_time * n_baseline * n_chan;
    if (n > 0 && (!uvw_m || !freq_hz || !vis)) return GRIDDER_ERR_INVALID_ARG;
    if (n > 0xFFFFF000ll) return GRIDDER_ERR_CAPACITY;
    if (((uintptr_t)vis & 15) || ((uintptr_t)grid & 7)) return GRIDDER_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    cudaError_t e = launch_scatter_atomic(*p, uvw_m, n_time, n_baseline, freq_hz, n_chan, vis, weight, grid,
                                          accumulate ? 1 : 0, s);
    if (e != cudaSuccess) return cuda_fail(p, e);
    p->last_stream = s;
    return GRIDDER_OK;
}

int gridder_sum_parts(const float *parts, int32_t n_parts, int64_t len, int64_t stride, float *out,
                      void *cuda_stream) {
    if (!parts || !out || n_parts < 1 || len < 0 || stride < len || (len & 3) || (stride & 3)) return GRIDDER_ERR_INVALID_ARG;
    if (((uintptr_t)parts & 15) || ((uintptr_t)out & 15)) return GRIDDER_ERR_INVALID_ARG;
    if (len == 0) return GRIDDER_OK;
    const cudaError_t e = launch_sum_parts(parts, n_parts, len, stride, out, (cudaStream_t)cuda_stream);
    return e == cudaSuccess ? GRIDDER_OK : GRIDDER_ERR_CUDA;
}

int gridder_image_workspace_size(gridder_plan_t *plan, size_t *bytes) {
    Plan *p = reinterpret_cast<Plan *>(plan);
    if (!p || !bytes) return GRIDDER_ERR_INVALID_ARG;
    return image_workspace(*p, bytes);
}

int gridder_image(gridder_plan_t *plan, const float *grid, float *image, const float *corr, void *work,
                  size_t work_bytes, void *cuda_stream) {
    Plan *p = reinterpret_cast<Plan *>(plan);
    if (!p || !grid || !image) return GRIDDER_ERR_INVALID_ARG;
    if (((uintptr_t)grid & 15) || ((uintptr_t)image & 15)) return GRIDDER_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const int rc = launch_image(*p, grid, image, corr, work, work_bytes, s);
    if (rc == GRIDDER_OK) p->last_stream = s;
    return rc;
}

int gridder_run_host(gridder_plan_t *plan, const double *h_uvw_m, int32_t n_time, int32_t n_baseline,
                     const double *h_freq_hz, int32_t n_chan, const float *h_vis, const float *h_weight,
                     float *h_grid, double *d_uvw_m, double *d_freq_hz, float *d_vis, float *d_weight,
                     float *d_grid, void *cuda_stream) {
    Plan *p = reinterpret_cast<Plan *>(plan);
    if (!p || !h_uvw_m || !h_freq_hz || !h_vis || !h_grid || !d_uvw_m || !d_freq_hz || !d_vis || !d_grid)
        return GRIDDER_ERR_INVALID_ARG;
    if (h_weight && !d_weight) return GRIDDER_ERR_INVALID_ARG;
    if (n_time < 0 || n_baseline < 0 || n_chan < 0) return GRIDDER_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const size_t n_tb = (size_t)n_time * n_baseline, n = n_tb * n_chan;
    const size_t gbytes = (size_t)4 * p->cfg.grid_size * p->cfg.grid_size * 2 * sizeof(float);
    cudaError_t e = cudaMemcpyAsync(d_uvw_m, h_uvw_m, n_tb * 3 * sizeof(double), cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_freq_hz, h_freq_hz, (size_t)n_chan * sizeof(double), cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return cuda_fail(p, e);

    // Large inputs are copied and gridded in slices of the flattened (integration, baseline) axis: the
    // copies run on a second stream, slice k is binned and gridded (added to the grid) while slice k+1
    // is still on the wire.  Gridding is linear, so the slices sum to the same grid (each slice's
    // result is rounded to FP32 once more when it is added; deterministic all the same).
    const size_t want = (size_t)(p->tune.host_slices ? p->tune.host_slices : 8);
    const size_t min_mb = (size_t)(p->tune.host_slice_min_mb ? p->tune.host_slice_min_mb : 256);
    const int n_slices = (n * 32 >= (min_mb << 20) && n_tb >= 8 && want > 1) ? (int)(n_tb < want ? n_tb : want) : 1;
    if (n_slices == 1) {
        // the binning only needs uvw and freq: it is enqueued ahead of the visibility copy
        int rc = gridder_bin(plan, d_uvw_m, n_time, n_baseline, d_freq_hz, n_chan, cuda_stream);
        if (rc != GRIDDER_OK) return rc;
        e = cudaMemcpyAsync(d_vis, h_vis, n * 8 * sizeof(float), cudaMemcpyHostToDevice, s);
        if (e == cudaSuccess && h_weight) e = cudaMemcpyAsync(d_weight, h_weight, n * sizeof(float), cudaMemcpyHostToDevice, s);
        if (e != cudaSuccess) return cuda_fail(p, e);
        rc = gridder_grid(plan, d_vis, h_weight ? d_weight : nullptr, d_grid, 0, cuda_stream);
        if (rc != GRIDDER_OK) return rc;
    } else {
        if (!p->copy_stream && cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking) != cudaSuccess)
            return cuda_fail(p, cudaGetLastError());
        cudaEvent_t ev[64], ev_start;
        int n_ev = 0;
        int rc = GRIDDER_OK;
        // the copy stream starts after whatever the caller's stream was doing with the staging buffers
        e = cudaEventCreateWithFlags(&ev_start, cudaEventDisableTiming);
        if (e != cudaSuccess) return cuda_fail(p, e);
        e = cudaEventRecord(ev_start, s);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(p->copy_stream, ev_start, 0);
        cudaEventDestroy(ev_start);
        // all copies are enqueued first (their stream never waits for the compute stream)
        for (int k = 0; k < n_slices && e == cudaSuccess; ++k) {
            const size_t r0 = n_tb * k / n_slices, r1 = n_tb * (k + 1) / n_slices, cnt = (r1 - r0) * n_chan;
            e = cudaMemcpyAsync(d_vis + r0 * n_chan * 8, h_vis + r0 * n_chan * 8, cnt * 8 * sizeof(float),
                                cudaMemcpyHostToDevice, p->copy_stream);
            if (e == cudaSuccess && h_weight)
                e = cudaMemcpyAsync(d_weight + r0 * n_chan, h_weight + r0 * n_chan, cnt * sizeof(float),
                                    cudaMemcpyHostToDevice, p->copy_stream);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ev[k], cudaEventDisableTiming);
            if (e == cudaSuccess) { ++n_ev; e = cudaEventRecord(ev[k], p->copy_stream); }
        }
        for (int k = 0; k < n_slices && e == cudaSuccess && rc == GRIDDER_OK; ++k) {
            const size_t r0 = n_tb * k / n_slices, r1 = n_tb * (k + 1) / n_slices;
            e = cudaStreamWaitEvent(s, ev[k], 0);
            if (e != cudaSuccess) break;
            rc = gridder_bin(plan, d_uvw_m + r0 * 3, 1, (int32_t)(r1 - r0), d_freq_hz, n_chan, cuda_stream);
            if (rc == GRIDDER_OK)
                rc = gridder_grid(plan, d_vis + r0 * n_chan * 8, h_weight ? d_weight + r0 * n_chan : nullptr, d_grid,
                                  k > 0 ? 1 : 0, cuda_stream);
        }
        if (e != cudaSuccess || rc != GRIDDER_OK) cudaStreamSynchronize(p->copy_stream);
        for (int k = 0; k < n_ev; ++k) cudaEventDestroy(ev[k]);
        if (e != cudaSuccess) return cuda_fail(p, e);
        if (rc != GRIDDER_OK) return rc;
    }
    e = cudaMemcpyAsync(h_grid, d_grid, gbytes, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return cuda_fail(p, e);
    return GRIDDER_OK;
}

int gridder_set_profiling(gridder_plan_t *plan, int32_t enable) {
    Plan *p = reinterpret_cast<Plan *>(plan);
    if (!p) return GRIDDER_ERR_INVALID_ARG;
    if (enable && !p->ev[0][0]) {
        for (int r = 0; r < kProfRing; ++r)
            for (int i = 0; i < 10; ++i)
                if (cudaEventCreate(&p->ev[r][i]) != cudaSuccess) return cuda_fail(p, cudaGetLastError());
    }
    p->profiling = enable != 0;
    p->prof_bin_calls = p->prof_grid_calls = 0;
    return GRIDDER_OK;
}

int gridder_get_stage_ms(gridder_plan_t *plan, float *ms_out) {
    Plan *p = reinterpret_cast<Plan *>(plan);
    if (!p || !ms_out) return GRIDDER_ERR_INVALID_ARG;
    double sum[6] = {0, 0, 0, 0, 0, 0};
    const int nb = (int)(p->prof_bin_calls < kProfRing ? p->prof_bin_calls : kProfRing);
    const int ng = (int)(p->prof_grid_calls < kProfRing ? p->prof_grid_calls : kProfRing);
    cudaError_t e = cudaSuccess;
    for (int r = 0; r < nb && e == cudaSuccess; ++r) {
        e = cudaEventSynchronize(p->ev[r][3]);
        for (int i = 0; i < 3 && e == cudaSuccess; ++i) {
            float ms = 0.f;
            e = cudaEventElapsedTime(&ms, p->ev[r][i], p->ev[r][i + 1]);
            sum[i] += ms;
        }
    }
    for (int r = 0; r < ng && e == cudaSuccess; ++r) {
        e = cudaEventSynchronize(p->ev[r][6]);
        // events of a grid call, in stream order: 4, [7 after the input-order pre-summation], 5 after the grid
        // kernels, 6 after the flush
        int last = 4;
        float ms = 0.f;
        if (p->presum_active && e == cudaSuccess) {
            e = cudaEventElapsedTime(&ms, p->ev[r][last], p->ev[r][7]);
            sum[5] += ms;
            last = 7;
        }
        if (e == cudaSuccess) { e = cudaEventElapsedTime(&ms, p->ev[r][last], p->ev[r][5]); sum[3] += ms; }
        if (e == cudaSuccess) { e = cudaEventElapsedTime(&ms, p->ev[r][5], p->ev[r][6]); sum[4] += ms; }
    }
    if (e != cudaSuccess) return cuda_fail(p, e);
    for (int i = 0; i < 3; ++i) ms_out[i] = nb ? (float)(sum[i] / nb) : 0.f;
    for (int i = 3; i < 6; ++i) ms_out[i] = ng ? (float)(sum[i] / ng) : 0.f;
    return GRIDDER_OK;
}

int64_t gridder_launch_count(const gridder_plan_t *plan) {
    const Plan *p = reinterpret_cast<const Plan *>(plan);
    return p ? p->n_launches : 0;
}

const char *gridder_strerror(int code) {
    switch (code) {
        case GRIDDER_OK: return "ok";
        case GRIDDER_ERR_INVALID_ARG: return "invalid argument";
        case GRIDDER_ERR_CAPACITY: return "more visibilities than the plan's max_vis";
        case GRIDDER_ERR_WORKSPACE: return "workspace too small";
        case GRIDDER_ERR_CUDA: return "CUDA runtime error";
        case GRIDDER_ERR_NOT_BINNED: return "gridder_bin has not been called on this plan";
        case GRIDDER_ERR_UNSUPPORTED: return "configuration not supported by this build";
        default: return "unknown gridder status";
    }
}

int gridder_last_cuda_error(const gridder_plan_t *plan) {
    const Plan *p = reinterpret_cast<const Plan *>(plan);
    return p ? p->last_cuda_error : 0;
}

const char *gridder_version(void) { return "0.2.0"; }

long long gridder_check_violations(void) {
#ifdef GRIDDER_CHECKED
    return g_check_violations;
#else
    return -1;
#endif
}

}  // extern "C"
