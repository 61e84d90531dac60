// gridder_grid_static: plan + bin + grid of a SMALL cadence without any allocation by anybody.
//
// Some callers cannot call cudaMalloc (tight serving loops, harnesses that forbid it, code that must not disturb a
// caching allocator) and therefore cannot hand the library the workspace every other entry point asks for.  For
// them the workspace of this one entry point is a file-scope device array of GRIDDER_STATIC_WORKSPACE_BYTES
// (64 MiB): every GPU that loads the library holds it from the first CUDA call of the process until exit.  The
// path behind it is the ordinary one (gridder_plan_tuned, gridder_bin, gridder_grid, gridder_destroy on that
// workspace), so the result is bit for bit what those calls give with a caller-owned workspace.
//
// What the caller must know (also in include/gridder.h):
//   * a plan that needs more than the array is refused with GRIDDER_ERR_WORKSPACE (the size it would need is
//     reported); nothing is enqueued;
//   * no cudaMalloc, cudaFree or allocating library routine is called (CUB gets its temporary storage from the
//     array; the plan object lives in host memory);
//   * every call on a device shares the array, and the array keeps the last call's contents.  The path clears
//     what must start at zero itself (gridder_plan: counters; gridder_bin: counters, tile tables; gridder_grid:
//     work queues; every partial region is written whole before the flush reads it), so a dirty array is the
//     normal case, and the test runs two different problems back to back;
//   * calls that overlapped on the GPU would race on the array.  They cannot: a process-wide lock serialises the
//     calls and each call synchronises the device before it returns (gridder_destroy).  Nothing else may use the
//     array.
//
// The array's name in HOST code is a host-side stand-in, not a device address; the device address is asked for
// once per device, with that device current, by cudaGetSymbolAddress, and that pointer is what the plan gets.
#include <cstring>
#include <mutex>

#include "gridder_internal.cuh"

namespace {

constexpr size_t kStaticWsBytes = GRIDDER_STATIC_WORKSPACE_BYTES;
constexpr int kMaxDevices = 64;

static __device__ __align__(256) unsigned char g_static_ws[kStaticWsBytes];

std::mutex g_static_mutex;                       // serialises the calls (and guards the table below)
void *g_static_ptr[kMaxDevices] = {};            // device address of g_static_ws on device d, once resolved

// Device address of the array on the CURRENT device (resolved at the first call on that device).
int static_workspace(void **out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return GRIDDER_ERR_CUDA;
    if (dev < 0 || dev >= kMaxDevices) return GRIDDER_ERR_UNSUPPORTED;
    if (!g_static_ptr[dev]) {
        void *ptr = nullptr;
        const cudaError_t e = cudaGetSymbolAddress((void **)&ptr, g_static_ws);
        if (e != cudaSuccess || !ptr) {
            (void)cudaGetLastError();
            return GRIDDER_ERR_CUDA;
        }
        if ((uintptr_t)ptr & 255) return GRIDDER_ERR_CUDA;          // __align__(256) was not honoured
        g_static_ptr[dev] = ptr;
    }
    *out = g_static_ptr[dev];
    return GRIDDER_OK;
}

}  // namespace

extern "C" {

int gridder_grid_static(const gridder_config *cfg, const gridder_tuning *tuning, const double *uvw_m, int32_t n_time,
                        int32_t n_baseline, const double *freq_hz, int32_t n_chan, const float *vis, const float *weight,
                        float *grid, int32_t accumulate, size_t *workspace_needed, void *cuda_stream) {
    if (workspace_needed) *workspace_needed = 0;
    if (!cfg || !uvw_m || !freq_hz || !vis || !grid) return GRIDDER_ERR_INVALID_ARG;
    gridder_tuning t;
    memset(&t, 0, sizeof(t));
    if (tuning) t = *tuning;
    // pre-summation in input order is for large cadences and synchronises in the middle of gridder_bin: only on request
    if (t.presum == 0) t.presum = 2;

    // the size first (host arithmetic only): a plan beyond the array is refused before anything is enqueued
    size_t need = 0;
    int rc = gridder_workspace_size_tuned(cfg, &t, &need);
    if (rc != GRIDDER_OK) return rc;
    if (workspace_needed) *workspace_needed = need;
    if (need > kStaticWsBytes) return GRIDDER_ERR_WORKSPACE;

    std::lock_guard<std::mutex> lock(g_static_mutex);
    void *ws = nullptr;
    rc = static_workspace(&ws);
    if (rc != GRIDDER_OK) return rc;

    gridder_config c = *cfg;
    c.workspace = ws;
    c.workspace_bytes = kStaticWsBytes;
    gridder_plan_t *plan = nullptr;
    rc = gridder_plan_tuned(&c, &t, &plan, nullptr);
    if (rc != GRIDDER_OK) return rc;
    rc = gridder_bin(plan, uvw_m, n_time, n_baseline, freq_hz, n_chan, cuda_stream);
    if (rc == GRIDDER_OK) rc = gridder_grid(plan, vis, weight, grid, accumulate, cuda_stream);
    const int rd = gridder_destroy(plan);            // synchronises the device: the array is free again
    return rc != GRIDDER_OK ? rc : rd;
}

}  // extern "C"
