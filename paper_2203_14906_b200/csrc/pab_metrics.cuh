// pab_metrics.cuh -- SURVEY.md section 8(f) row f3: image-quality metrics of the paper's evaluation on the device:
// SNR eq. (10), CR eq. (11), gCNR eq. (12) and FWHM, reading A22.
// The image is the float32 array the beamformer delivers; sums are carried in double, the histogram bin of gCNR
// is decided in float32 arithmetic with individually rounded operations.
#pragma once
#include <cuda_runtime.h>
#include "pab_types.h"

namespace pab {

__device__ __forceinline__ double block_sum(double v, double* sh) {
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) sh[warp] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x < 32) {
        t = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.0;
        for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
    }
    return t;       // valid in thread 0
}

// pass 1: sums and maximum.  grid: (blocks, 2): y = 0 target, 1 background.
__global__ void __launch_bounds__(256) metrics_sum_kernel(const float* __restrict__ img, int nx, RoiPair R, MetricAcc* acc) {
    __shared__ double sh[8];
    const int* r = blockIdx.y == 0 ? R.t : R.b;
    const int w = r[3] - r[2], n = (r[1] - r[0]) * w;
    double s = 0.0;
    float mx = 0.0f;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const float v = img[(size_t)(r[0] + i / w) * nx + r[2] + i % w];
        s += (double)v;
        mx = fmaxf(mx, v);
    }
    for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if ((threadIdx.x & 31) == 0 && mx > 0.0f) atomicMax(&acc->max_bits, __float_as_uint(mx));
    const double t = block_sum(s, sh);
    if (threadIdx.x == 0) atomicAdd(blockIdx.y == 0 ? &acc->sum_in : &acc->sum_out, t);
}

// pass 2: background variance about its mean, and the two histograms.  hist[2][n_bins] unsigned.
__global__ void __launch_bounds__(256) metrics_hist_kernel(const float* __restrict__ img, int nx, RoiPair R, MetricAcc* acc,
                                                           unsigned int* hist, int n_bins) {
    __shared__ double sh[8];
    const int* r = blockIdx.y == 0 ? R.t : R.b;
    const int w = r[3] - r[2], n = (r[1] - r[0]) * w;
    const float vmax = __uint_as_float(acc->max_bits);
    const double mu = acc->sum_out / (double)((R.b[1] - R.b[0]) * (R.b[3] - R.b[2]));
    double var = 0.0;
    unsigned int* h = hist + blockIdx.y * n_bins;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const float v = img[(size_t)(r[0] + i / w) * nx + r[2] + i % w];
        int b = vmax > 0.0f ? (int)floorf(__fmul_rn(__fdiv_rn(v, vmax), (float)n_bins)) : 0;
        b = min(max(b, 0), n_bins - 1);
        atomicAdd(h + b, 1u);
        if (blockIdx.y == 1) { const double d = (double)v - mu; var += d * d; }
    }
    if (blockIdx.y == 1) {
        const double t = block_sum(var, sh);
        if (threadIdx.x == 0) atomicAdd(&acc->var_out, t);
    }
}

// FWHM on one row inside the target's columns; one warp.  out[0] = width in pixels (double).
__global__ void metrics_fwhm_kernel(const float* __restrict__ img, int nx, int row, int c0, int c1, double* out) {
    const float* p = img + (size_t)row * nx;
    // first maximum: value descending, then column ascending
    float best = -1.0f; int pk = c0;
    for (int c = c0 + (int)threadIdx.x; c < c1; c += 32) if (p[c] > best) { best = p[c]; pk = c; }
    for (int o = 16; o > 0; o >>= 1) {
        const float ob = __shfl_xor_sync(0xffffffffu, best, o);
        const int op = __shfl_xor_sync(0xffffffffu, pk, o);
        if (ob > best || (ob == best && op < pk)) { best = ob; pk = op; }
    }
    if (threadIdx.x == 0) {
        const double half = 0.5 * (double)p[pk];
        double left = (double)c0, right = (double)(c1 - 1);
        for (int c = pk; c > c0; --c)
            if ((double)p[c - 1] < half) { left = (double)(c - 1) + (half - (double)p[c - 1]) / ((double)p[c] - (double)p[c - 1]); break; }
        for (int c = pk; c < c1 - 1; ++c)
            if ((double)p[c + 1] < half) { right = (double)c + ((double)p[c] - half) / ((double)p[c] - (double)p[c + 1]); break; }
        out[0] = right - left;
    }
}

}  // namespace pab
