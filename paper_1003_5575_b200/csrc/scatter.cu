// gridder_scatter_atomic: the arithmetic of the paper's OpenGL gridder
// (PAPER.md :185-191) restated in CUDA.  "For each visibility, we simply rendered a screen-aligned
// quadrilateral texture-mapped with the appropriate GCF ... with additive blending enabled": here a
// warp takes a visibility, its lanes rasterise the S x S quad, and every (tap, polarisation) is an FP32
// atomic add into the HBM grid (red.global.add.v2.f32) -- the "atomic floating point instructions"
// the paper expected of Fermi (:187).  O(v k) work, no binning, no sort.  The order of the additions is
// not fixed, so results are NOT bit-identical from run to run and long FP32 chains are not bounded:
// this path is a same-box comparison for the binned gridder, checked against the oracle on small
// inputs only, and never used where determinism is promised.
#include "gridder_internal.cuh"
#include "map.cuh"

namespace gridder {

__device__ __forceinline__ void red_add_v2(float2 *addr, float re, float im) {
    asm volatile("red.global.add.v2.f32 [%0], {%1, %2};" :: "l"(addr), "f"(re), "f"(im) : "memory");
}

__global__ void __launch_bounds__(256) scatter_atomic_kernel(const double *__restrict__ uvw,
                                                              const double *__restrict__ freq, unsigned int n,
                                                              unsigned int n_chan, const MapParams p,
                                                              const float *__restrict__ table,   // user layout
                                                              const unsigned long long *__restrict__ plane_off,
                                                              const float4 *__restrict__ vis,
                                                              const float *__restrict__ weight,
                                                              float2 *__restrict__ grid) {
    const int lane = threadIdx.x & 31;
    const unsigned int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const unsigned int n_warps = (gridDim.x * blockDim.x) >> 5;
    const size_t nn = (size_t)p.n_grid * p.n_grid;
    const int O = p.oversample;
    for (unsigned int i = warp; i < n; i += n_warps) {
        const unsigned int tb = i / n_chan, f = i - tb * n_chan;
        const double s = __ddiv_rn(freq[f], kSpeedOfLight);
        const VisMap m = map_vis(uvw[(size_t)tb * 3], uvw[(size_t)tb * 3 + 1], uvw[(size_t)tb * 3 + 2], s, p);
        if (m.dropped) continue;                                // warp-uniform
        const int S = m.S, pitch = S * O;
        const float w = weight ? weight[i] : 1.0f;
        const float4 a = vis[2 * (size_t)i], b = vis[2 * (size_t)i + 1];
        const float v[8] = {a.x * w, a.y * w, a.z * w, a.w * w, b.x * w, b.y * w, b.z * w, b.w * w};
        const float *K = table + plane_off[m.plane];
        for (int t = lane; t < S * S; t += 32) {
            const int ty = t / S, tx = t - ty * S;
            const size_t j = (size_t)(m.qy + ty * O) * pitch + (m.qx + tx * O);
            float kr, ki = 0.f;
            if (p.is_complex) {
                const float2 k2 = reinterpret_cast<const float2 *>(K)[j];
                kr = k2.x;
                ki = m.conj ? -k2.y : k2.y;
            } else {
                kr = K[j];
            }
            float2 *cell = grid + (size_t)(m.y0 + ty) * p.n_grid + (size_t)(m.x0 + tx);
#pragma unroll
            for (int pol = 0; pol < 4; ++pol) {
                const float vr = v[2 * pol], vi = v[2 * pol + 1];
                red_add_v2(cell + pol * nn, fmaf(vr, kr, -vi * ki), fmaf(vr, ki, vi * kr));
            }
        }
    }
}

cudaError_t launch_scatter_atomic(Plan &p, const double *uvw, int n_time, int n_bl, const double *freq, int n_chan,
                                  const float *vis, const float *weight, float *grid, int accumulate,
                                  cudaStream_t s) {
    const long long n = (long long)n_time * n_bl * n_chan;
    const size_t gbytes = (size_t)4 * p.cfg.grid_size * p.cfg.grid_size * sizeof(float2);
    cudaError_t e = cudaSuccess;
    if (!accumulate) e = cudaMemsetAsync(grid, 0, gbytes, s);
    if (e != cudaSuccess || n == 0) return e;
    // element offsets of the planes in the caller's table: staged in the (otherwise unused here) scan scratch
    unsigned long long off[kMaxPlanes];
    unsigned long long o = 0;
    const int E = p.cfg.kernel_is_complex ? 2 : 1;
    for (int i = 0; i < p.cfg.n_wplanes; ++i) {
        off[i] = o;
        o += (unsigned long long)p.support_copy[i] * p.cfg.oversample * p.support_copy[i] * p.cfg.oversample * E;
    }
    e = cudaMemcpyAsync(p.tile_chunks, off, sizeof(unsigned long long) * p.cfg.n_wplanes, cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return e;
    long long blocks = (n + 7) / 8;                       // 8 warps per block, one visibility per warp per pass
    const long long cap = (long long)p.n_sm * 32;
    if (blocks > cap) blocks = cap;
    scatter_atomic_kernel<<<(int)blocks, 256, 0, s>>>(uvw, freq, (unsigned)n, (unsigned)n_chan, make_map_params(p),
                                                      (const float *)p.cfg.kernel, p.tile_chunks,
                                                      reinterpret_cast<const float4 *>(vis), weight,
                                                      reinterpret_cast<float2 *>(grid));
    p.n_launches += 1;
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------
// Row f4: out[i] = (float) sum over the parts, in part order, in double (include/gridder.h).  One float4
// per thread and part: HBM-bound, (n_parts + 1) x 4 len bytes.
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) sum_parts_kernel(const float4 *parts, int n_parts, long long len4,
                                                         long long stride4, float4 *out) {     // (out may alias part 0)
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < len4; i += (long long)gridDim.x * blockDim.x) {
        double a = 0.0, b = 0.0, c = 0.0, d = 0.0;
        for (int p = 0; p < n_parts; ++p) {
            const float4 v = parts[(long long)p * stride4 + i];
            a += (double)v.x; b += (double)v.y; c += (double)v.z; d += (double)v.w;
        }
        out[i] = make_float4((float)a, (float)b, (float)c, (float)d);
    }
}

cudaError_t launch_sum_parts(const float *parts, int n_parts, long long len, long long stride, float *out, cudaStream_t s) {
    const long long len4 = len / 4;
    long long blocks = (len4 + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    sum_parts_kernel<<<(int)blocks, 256, 0, s>>>(reinterpret_cast<const float4 *>(parts), n_parts, len4, stride / 4,
                                                 reinterpret_cast<float4 *>(out));
    return cudaGetLastError();
}

}  // namespace gridder
