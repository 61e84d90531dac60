// gridder_image: the stage right after the gridder in the paper's pipeline --
// "the gridded visibilities are then Fourier transformed" into images (PAPER.md :75; 2-D inverse FFT
// of 4 polarisations, :211, :217), with the division by the Fourier transform of the gridding
// convolution function ("grid correction") fused into the pass that re-centres the image.
//   image[pol][y][x] = corr[y] corr[x] * sum_{v,u} G[pol][v][u] exp(+2 pi i ((u-N/2)(x-N/2) + (v-N/2)(y-N/2)) / N)
// The centring of both planes on cell N/2 is done with the (-1)^(u+v) / (-1)^(x+y) sign trick (N is
// even), so the FFT itself is a plain batched C2C inverse: a library primitive (cuFFT), loaded lazily
// with dlopen so that the gridding path does not depend on it.  The two element-wise passes are ours.
#include <cufft.h>
#include <dlfcn.h>

#include "gridder_internal.cuh"

namespace gridder {

namespace {

struct CufftApi {
    void *lib = nullptr;
    cufftResult (*Create)(cufftHandle *) = nullptr;
    cufftResult (*SetAutoAllocation)(cufftHandle, int) = nullptr;
    cufftResult (*MakePlanMany)(cufftHandle, int, int *, int *, int, int, int *, int, int, cufftType, int, size_t *) = nullptr;
    cufftResult (*SetWorkArea)(cufftHandle, void *) = nullptr;
    cufftResult (*SetStream)(cufftHandle, cudaStream_t) = nullptr;
    cufftResult (*ExecC2C)(cufftHandle, cufftComplex *, cufftComplex *, int) = nullptr;
    cufftResult (*Destroy)(cufftHandle) = nullptr;
    bool ok = false;
};

CufftApi &cufft_api() {
    static CufftApi api;
    static bool tried = false;
    if (tried) return api;
    tried = true;
    const char *names[] = {"libcufft.so.11", "libcufft.so", "/usr/local/cuda/lib64/libcufft.so.11"};
    for (const char *n : names) {
        api.lib = dlopen(n, RTLD_NOW | RTLD_LOCAL);
        if (api.lib) break;
    }
    if (!api.lib) return api;
    api.Create = (decltype(api.Create))dlsym(api.lib, "cufftCreate");
    api.SetAutoAllocation = (decltype(api.SetAutoAllocation))dlsym(api.lib, "cufftSetAutoAllocation");
    api.MakePlanMany = (decltype(api.MakePlanMany))dlsym(api.lib, "cufftMakePlanMany");
    api.SetWorkArea = (decltype(api.SetWorkArea))dlsym(api.lib, "cufftSetWorkArea");
    api.SetStream = (decltype(api.SetStream))dlsym(api.lib, "cufftSetStream");
    api.ExecC2C = (decltype(api.ExecC2C))dlsym(api.lib, "cufftExecC2C");
    api.Destroy = (decltype(api.Destroy))dlsym(api.lib, "cufftDestroy");
    api.ok = api.Create && api.SetAutoAllocation && api.MakePlanMany && api.SetWorkArea && api.SetStream &&
             api.ExecC2C && api.Destroy;
    return api;
}

}  // namespace

// out = in * (-1)^(x+y) [* corr[y] corr[x]]; float4 = two complex cells (x even, x+1), so the signs
// inside one float4 are (s, s, -s, -s) with s = (-1)^y.
__global__ void __launch_bounds__(256) centre_kernel(const float4 *in, float4 *out,       // (may be the same buffer: no __restrict__)
                                                      const float *__restrict__ corr, int n_grid, size_t n_f4) {
    const int half = n_grid >> 1;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_f4; i += (size_t)gridDim.x * blockDim.x) {
        const int xh = (int)(i % half);
        const int y = (int)((i / half) % n_grid);
        float s0 = (y & 1) ? -1.f : 1.f, s1 = -s0;
        if (corr) {
            const float cy = corr[y];
            s0 *= cy * corr[2 * xh];
            s1 *= cy * corr[2 * xh + 1];
        }
        const float4 v = in[i];
        out[i] = make_float4(v.x * s0, v.y * s0, v.z * s1, v.w * s1);
    }
}

static int image_plan(Plan &p, void *work, size_t work_bytes, size_t *need) {
    CufftApi &api = cufft_api();
    if (!api.ok) return GRIDDER_ERR_UNSUPPORTED;
    if (!p.fft_ready) {
        cufftHandle h;
        if (api.Create(&h) != CUFFT_SUCCESS) return GRIDDER_ERR_CUDA;
        api.SetAutoAllocation(h, 0);
        int n[2] = {p.cfg.grid_size, p.cfg.grid_size};
        size_t ws = 0;
        if (api.MakePlanMany(h, 2, n, nullptr, 1, n[0] * n[1], nullptr, 1, n[0] * n[1], CUFFT_C2C, 4, &ws) != CUFFT_SUCCESS) {
            api.Destroy(h);
            return GRIDDER_ERR_CUDA;
        }
        p.fft_handle = (int)h;
        p.fft_work_bytes = ws;
        p.fft_ready = true;
    }
    if (need) *need = p.fft_work_bytes;
    if (!work && !need) return GRIDDER_ERR_INVALID_ARG;
    if (work && work_bytes < p.fft_work_bytes) return GRIDDER_ERR_WORKSPACE;
    return GRIDDER_OK;
}

int image_workspace(Plan &p, size_t *bytes) { return image_plan(p, nullptr, 0, bytes); }

void image_destroy(Plan &p) {
    if (p.fft_ready && cufft_api().ok) cufft_api().Destroy((cufftHandle)p.fft_handle);
    p.fft_ready = false;
}

int launch_image(Plan &p, const float *grid, float *image, const float *corr, void *work, size_t work_bytes,
                 cudaStream_t s) {
    size_t need = 0;
    const int rc = image_plan(p, work, work_bytes, &need);
    if (rc != GRIDDER_OK) return rc;
    if (need > 0 && !work) return GRIDDER_ERR_WORKSPACE;
    CufftApi &api = cufft_api();
    const cufftHandle h = (cufftHandle)p.fft_handle;
    const size_t n_f4 = (size_t)4 * p.cfg.grid_size * p.cfg.grid_size / 2;
    const int blocks = p.n_sm * 16;
    centre_kernel<<<blocks, 256, 0, s>>>(reinterpret_cast<const float4 *>(grid), reinterpret_cast<float4 *>(image),
                                         nullptr, p.cfg.grid_size, n_f4);
    if (cudaGetLastError() != cudaSuccess) return GRIDDER_ERR_CUDA;
    if (api.SetStream(h, s) != CUFFT_SUCCESS) return GRIDDER_ERR_CUDA;
    if (need > 0 && api.SetWorkArea(h, work) != CUFFT_SUCCESS) return GRIDDER_ERR_CUDA;
    if (api.ExecC2C(h, reinterpret_cast<cufftComplex *>(image), reinterpret_cast<cufftComplex *>(image), CUFFT_INVERSE) !=
        CUFFT_SUCCESS)
        return GRIDDER_ERR_CUDA;
    centre_kernel<<<blocks, 256, 0, s>>>(reinterpret_cast<const float4 *>(image), reinterpret_cast<float4 *>(image),
                                         corr, p.cfg.grid_size, n_f4);
    if (cudaGetLastError() != cudaSuccess) return GRIDDER_ERR_CUDA;
    p.n_launches += 3;
    return GRIDDER_OK;
}

}  // namespace gridder
