// pab_tu_peaks.cu -- translation unit: the microbenchmarks behind the roofline denominators (SURVEY.md section 8(d):
// "to be confirmed on the box by two microbenchmarks, an FMA-throughput loop and a MUFU-throughput loop"), plus the
// shared-memory load rate and the pinned host <-> device copy rate that bound the secondary ceilings DESIGN.md quotes.
// Every kernel times itself with clock64() inside one CTA per SM, so the unit is lanes (or bytes) per clock per SM and
// no clock frequency enters; the SM clock is reported separately from cycles / event time.
#include <cstdint>
#include <cuda_runtime.h>
#include "../../include/pab.h"

namespace {

constexpr int kThreads = 1024, kIters = 4096, kChains = 8;

__device__ __forceinline__ float mufu_ex2(float x) { float y; asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_lg2(float x) { float y; asm volatile("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// kind 0: MUFU (alternating lg2 / ex2, the cube root's pair); 1: FFMA; 2: FFMA2 (fma.rn.f32x2)
template <int KIND>
__global__ void __launch_bounds__(kThreads, 1) peak_alu_kernel(float seed, long long* cycles, float* sink) {
    float v[kChains];
#pragma unroll
    for (int c = 0; c < kChains; ++c) v[c] = seed + 0.001f * (float)(threadIdx.x + c);
    unsigned long long w[kChains / 2];
#pragma unroll
    for (int c = 0; c < kChains / 2; ++c) w[c] = ((unsigned long long)__float_as_uint(v[2 * c + 1]) << 32) | __float_as_uint(v[2 * c]);
    const unsigned long long ab = ((unsigned long long)__float_as_uint(0.999f) << 32) | __float_as_uint(1.001f);
    const float fa = seed * 0.666f, fb = seed * 0.0007f;
    __syncthreads();
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < kIters; ++it) {
        if constexpr (KIND == 0) {
#pragma unroll
            for (int c = 0; c < kChains; ++c) v[c] = mufu_ex2(mufu_lg2(v[c]));
        } else if constexpr (KIND == 1) {
#pragma unroll
            for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int c = 0; c < kChains; ++c) v[c] = fmaf(v[c], fa, fb);          // three register operands
        } else {
#pragma unroll
            for (int r = 0; r < 2; ++r)
#pragma unroll
                for (int c = 0; c < kChains / 2; ++c) asm volatile("fma.rn.f32x2 %0, %0, %1, %1;" : "+l"(w[c]) : "l"(ab));
        }
    }
    const long long t1 = clock64();
    __syncthreads();
    float s = 0.0f;
#pragma unroll
    for (int c = 0; c < kChains; ++c) s += v[c];
#pragma unroll
    for (int c = 0; c < kChains / 2; ++c) s += __uint_as_float((unsigned)w[c]);
    if (s == 123.456f) sink[0] = s;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

// conflict-free 128-bit shared loads: lane l of a warp reads 16 bytes at l * 16 (+ a rotating offset)
__global__ void __launch_bounds__(kThreads, 1) peak_lds_kernel(long long* cycles, float* sink) {
    __shared__ __align__(16) float buf[kThreads * 4 + 64];
    for (int i = threadIdx.x; i < kThreads * 4 + 64; i += kThreads) buf[i] = (float)i;
    __syncthreads();
    const uint32_t base = (uint32_t)__cvta_generic_to_shared(buf) + threadIdx.x * 16;
    float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
    const long long t0 = clock64();
#pragma unroll 1
    for (int it = 0; it < kIters; ++it) {
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            float4 v;
            asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(base + c * 16));
            a.x += v.x; a.y += v.y; a.z += v.z; a.w += v.w;
        }
    }
    const long long t1 = clock64();
    __syncthreads();
    if (a.x + a.y + a.z + a.w == 123.456f) sink[0] = a.x;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

double slowest(const long long* h, int n) {
    long long m = 1;
    for (int i = 0; i < n; ++i) m = h[i] > m ? h[i] : m;
    return (double)m;
}

}  // namespace

// out[0] MUFU lanes/clk/SM   out[1] FFMA lanes/clk/SM   out[2] FFMA2 lanes/clk/SM (two fp32 results per lane-slot count
// as two)   out[3] LDS.128 bytes/clk/SM   out[4] pinned host->device GB/s   out[5] device->host GB/s (64 MiB copies)
// out[6] SM clock seen during the MUFU loop, MHz   out[7] SM count
extern "C" int pab_measure_peaks(double* out, int n_out) {
    if (!out || n_out < 8) return PAB_ERR_INVALID;
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess || prop.major != 10) return PAB_ERR_DEVICE;
    const int sms = prop.multiProcessorCount;
    long long* d_cyc = nullptr;
    float* d_sink = nullptr;
    long long* h_cyc = new long long[sms];
    cudaEvent_t e0, e1;
    if (cudaMalloc(&d_cyc, sms * sizeof(long long)) != cudaSuccess || cudaMalloc(&d_sink, 64) != cudaSuccess) {
        cudaFree(d_cyc); cudaFree(d_sink); delete[] h_cyc;
        cudaGetLastError();
        return PAB_ERR_ALLOC;
    }
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    auto cyc = [&]() { cudaMemcpy(h_cyc, d_cyc, sms * sizeof(long long), cudaMemcpyDeviceToHost); return slowest(h_cyc, sms); };
    for (int rep = 0; rep < 2; ++rep) {          // first pass warms clocks and caches
        cudaEventRecord(e0);
        peak_alu_kernel<0><<<sms, kThreads>>>(1.5f, d_cyc, d_sink);
        cudaEventRecord(e1);
        const double c0 = cyc();
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        out[0] = (double)kThreads * kIters * kChains * 2 / c0;
        out[6] = c0 / (ms * 1e-3) / 1e6;
        peak_alu_kernel<1><<<sms, kThreads>>>(1.5f, d_cyc, d_sink);
        out[1] = (double)kThreads * kIters * kChains * 2 / cyc();
        peak_alu_kernel<2><<<sms, kThreads>>>(1.5f, d_cyc, d_sink);
        out[2] = (double)kThreads * kIters * kChains * 2 / cyc();
        peak_lds_kernel<<<sms, kThreads>>>(d_cyc, d_sink);
        out[3] = (double)kThreads * kIters * 8 * 16 / cyc();
    }
    const size_t bytes = 64u << 20;
    void *h = nullptr, *d = nullptr;
    out[4] = out[5] = 0.0;
    if (cudaMallocHost(&h, bytes) == cudaSuccess && cudaMalloc(&d, bytes) == cudaSuccess) {
        for (int dir = 0; dir < 2; ++dir) {
            float best = 1e30f;
            for (int rep = 0; rep < 6; ++rep) {
                cudaEventRecord(e0);
                if (dir == 0) cudaMemcpyAsync(d, h, bytes, cudaMemcpyHostToDevice, 0);
                else cudaMemcpyAsync(h, d, bytes, cudaMemcpyDeviceToHost, 0);
                cudaEventRecord(e1);
                cudaEventSynchronize(e1);
                float ms = 0.f;
                cudaEventElapsedTime(&ms, e0, e1);
                if (rep > 0 && ms < best) best = ms;
            }
            out[4 + dir] = (double)bytes / (best * 1e-3) / 1e9;
        }
    }
    if (h) cudaFreeHost(h);
    cudaFree(d);
    out[7] = (double)sms;
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d_cyc); cudaFree(d_sink);
    delete[] h_cyc;
    return cudaGetLastError() == cudaSuccess ? PAB_OK : PAB_ERR_CUDA;
}
