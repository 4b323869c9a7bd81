// pab_kernels.cuh -- ingest (a1), direct beamforming (a2..a6, a10) and post (a7..a9) kernels.
// The staged (bulk-copy + mbarrier) beamforming kernel lives in pab_staged.cuh.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "pab_math.cuh"

namespace pab {

// ------------------------------------------------------------------------------------------------------
// Parameters of one beamforming launch.
//
// Staged-RF layouts (written by the ingest kernels below, device memory owned by the context):
//   V = 1 ("lin")  : rf[frame][N][Sp]        fp32, Sp = S rounded up to 4 (16-byte rows)
//   V = 4 ("quad") : rf[quad][N][S][4]       fp32, the 4 frames of a quad interleaved per sample, so one
//                    128-bit load brings a sample of 4 frames and the delay/index work of a (pixel, element)
//                    pair is shared by every frame a thread carries (step a10).
// Output: out[frame][nz][nx], x fastest.
// ------------------------------------------------------------------------------------------------------
struct BfParams {
    const float* rf;       // staged RF of this launch's first frame / quad
    float* out;            // image of this launch's first frame
    const float2* xj;      // [nx]  pixel column x_j in samples (x fs / c), fp32 hi + lo
    const float2* xe;      // [N]   element x in samples, fp32 hi + lo
    const float4* zrow;    // [nz]  (zs_hi, 2 zs_lo, zf - 1/2, zi - 2 * 0x4B400000 as int bits), zs = z fs / c = zi + zf
    int N, S, Sp, nx, nz;
    int n_frames;          // valid frames in this launch (stores beyond are skipped)
    float inv_n;           // 1 / N, for the coherence factor (row f1)
};

// ------------------------------------------------------------------------------------------------------
// a1: ingest.  T = float or int16_t.  value = scale * stored (A15; int16 -> fp32 is exact).
// ------------------------------------------------------------------------------------------------------
template <typename T> __device__ __forceinline__ float ld_as_float(const T* p) { return (float)(*p); }

// rf[F][N][S] -> quad[ceil(F/4)][N][S][4]; frames beyond F are written as zeros.
// grid: (ceil(S / (4*blockDim.x)), N, n_quads); each thread moves 4 samples x 4 frames.
template <typename T>
__global__ void __launch_bounds__(256) ingest_quad_kernel(const T* __restrict__ rf, float4* __restrict__ quad,
                                                           int F, int N, int S, float scale) {
    const int n = blockIdx.y, q = blockIdx.z;
    const int s4 = (blockIdx.x * blockDim.x + threadIdx.x) * 4;
    if (s4 >= S) return;
    float v[4][4];
#pragma unroll
    for (int fr = 0; fr < 4; ++fr) {
        const int f = q * 4 + fr;
        const T* src = rf + ((size_t)f * N + n) * (size_t)S + s4;
#pragma unroll
        for (int k = 0; k < 4; ++k) v[fr][k] = (f < F && s4 + k < S) ? scale * ld_as_float(src + k) : 0.0f;
    }
    float4* dst = quad + ((size_t)q * N + n) * (size_t)S + s4;
#pragma unroll
    for (int k = 0; k < 4; ++k)
        if (s4 + k < S) dst[k] = make_float4(v[0][k], v[1][k], v[2][k], v[3][k]);
}

// The same for fp32 records with S a multiple of 4 at a 16-byte aligned address: 128-bit loads, all 4 frames in flight.
__global__ void __launch_bounds__(256) ingest_quad_vec_kernel(const float4* __restrict__ rf, float4* __restrict__ quad,
                                                               int F, int N, int S4, float scale) {
    const int n = blockIdx.y, q = blockIdx.z;
    const int s4 = blockIdx.x * blockDim.x + threadIdx.x;     // in units of 4 samples
    if (s4 >= S4) return;
    float4 v[4];
#pragma unroll
    for (int fr = 0; fr < 4; ++fr) {
        const int f = q * 4 + fr;
        v[fr] = f < F ? __ldcs(rf + ((size_t)f * N + n) * (size_t)S4 + s4) : make_float4(0.f, 0.f, 0.f, 0.f);
    }
    float4* dst = quad + (((size_t)q * N + n) * (size_t)S4 + s4) * 4;
    dst[0] = make_float4(scale * v[0].x, scale * v[1].x, scale * v[2].x, scale * v[3].x);
    dst[1] = make_float4(scale * v[0].y, scale * v[1].y, scale * v[2].y, scale * v[3].y);
    dst[2] = make_float4(scale * v[0].z, scale * v[1].z, scale * v[2].z, scale * v[3].z);
    dst[3] = make_float4(scale * v[0].w, scale * v[1].w, scale * v[2].w, scale * v[3].w);
}

// rf[F][N][S] -> lin[F][N][Sp], Sp >= S multiple of 4, pad written as zeros.  grid: (ceil(Sp/blockDim.x), N, F)
template <typename T>
__global__ void __launch_bounds__(256) ingest_lin_kernel(const T* __restrict__ rf, float* __restrict__ lin,
                                                          int N, int S, int Sp, float scale) {
    const int n = blockIdx.y, f = blockIdx.z;
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= Sp) return;
    lin[((size_t)f * N + n) * (size_t)Sp + s] = s < S ? scale * ld_as_float(rf + ((size_t)f * N + n) * (size_t)S + s) : 0.0f;
}

// ------------------------------------------------------------------------------------------------------
// Direct beamforming kernel: one thread per pixel, lanes along depth (so a warp's gathers of one channel
// fall in one short contiguous window: adjacent rows differ by <= dz fs / c samples), 8 warps = 8 columns.
// Gathers go through L1/L2 with 128-bit loads from the quad layout (NQ quads = 4 NQ frames per thread) or
// 32-bit loads from the lin layout (NQ = 0: one frame per thread).  No shared memory; any geometry.
// grid: (ceil(nx/8), ceil(nz/32), groups) with group = one frame (NQ = 0) or NQ quads.
// ------------------------------------------------------------------------------------------------------
constexpr int kDirectCols = 8;
constexpr int kDirectRows = 32;

template <int K, int NQ, int W>
__global__ void __launch_bounds__(256) bf_direct_kernel(const BfParams P) {
    constexpr int NF = NQ == 0 ? 1 : 4 * NQ;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int j = blockIdx.x * kDirectCols + warp;
    const int m = blockIdx.y * kDirectRows + lane;
    const float2 xj = P.xj[min(j, P.nx - 1)];
    const float4 row = P.zrow[min(m, P.nz - 1)];

    float p[NF][kAcc<K, W>];
#pragma unroll
    for (int f = 0; f < NF; ++f)
#pragma unroll
        for (int k = 0; k < kAcc<K, W>; ++k) p[f][k] = 0.0f;

    if constexpr (NQ == 0) {
        const float* chan = P.rf + (size_t)blockIdx.z * P.N * (size_t)P.Sp;
#pragma unroll 4
        for (int i = 0; i < P.N; ++i, chan += P.Sp) {
            const float2 xe = __ldg(P.xe + i);
            const float2 xs = lateral_square(xj, xe);
            const Tap t = delay_tap<false>(xs.x, xs.y, row, P.S);
            const float s0 = __ldg(chan + t.i0), s1 = __ldg(chan + t.i0 + 1);
            accumulate_w<K, W>(interp<false>(t, s0, s1), p[0]);
        }
    } else {
        const size_t quad_stride = (size_t)P.N * (size_t)P.S;      // float4 units
        const float4* chan = reinterpret_cast<const float4*>(P.rf) + (size_t)blockIdx.z * NQ * quad_stride;
#pragma unroll 2
        for (int i = 0; i < P.N; ++i, chan += P.S) {
            const float2 xe = __ldg(P.xe + i);
            const float2 xs = lateral_square(xj, xe);
            const Tap t = delay_tap<false>(xs.x, xs.y, row, P.S);
#pragma unroll
            for (int q = 0; q < NQ; ++q) {
                const float4 s0 = __ldg(chan + q * quad_stride + t.i0);
                const float4 s1 = __ldg(chan + q * quad_stride + t.i0 + 1);
                accumulate_w<K, W>(interp<false>(t, s0.x, s1.x), p[4 * q + 0]);
                accumulate_w<K, W>(interp<false>(t, s0.y, s1.y), p[4 * q + 1]);
                accumulate_w<K, W>(interp<false>(t, s0.z, s1.z), p[4 * q + 2]);
                accumulate_w<K, W>(interp<false>(t, s0.w, s1.w), p[4 * q + 3]);
            }
        }
    }

    if (j < P.nx && m < P.nz) {
        const size_t img = (size_t)P.nz * P.nx;
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            const int frame = blockIdx.z * NF + f;
            if (frame < P.n_frames) P.out[(size_t)frame * img + (size_t)m * P.nx + j] = combine_w<K, W>(p[f], P.inv_n);
        }
    }
}

// ------------------------------------------------------------------------------------------------------
// a7 + a8: axial FIR band-pass and Hilbert-FIR envelope, fused per tile of TZ rows x 32 columns.
//
//   y[m] = sum_{t<T} h[t] x[m + T/2 - t]        x = 0 outside [0, nz)      (A11, A12)
//   q[m] = sum_{t'<2L+1} g[t'] y[m + L - t']    y = 0 outside [0, nz)      (A9)
//   env  = sqrt(y^2 + q^2); per-frame max of env by atomicMax on the bit pattern (env >= 0)
//
// Both filters are "out[m] = sum_t taps[t] in[m + shift - t]" with the tap count padded to a multiple of 8
// by zeros; fir8 computes 8 consecutive rows of one column with a 15-row register window, 64 FMAs per
// 8 + 8 shared-memory loads.  Lanes own columns (coalesced image rows).
// ------------------------------------------------------------------------------------------------------
struct PostParams {
    const float* x;        // [F][nz][nx] beamformed image
    float* out;            // [F][nz][nx]: y (ENV = false) or env (ENV = true)
    unsigned int* frame_max;   // [F] bit pattern of the per-frame max of env (ENV = true), zeroed before launch
    const float* taps_bp;  // [TpB] padded
    const float* taps_h;   // [TpH] padded
    int TpB, shiftB;       // padded band-pass tap count, T/2
    int TpH, shiftH;       // padded Hilbert tap count, L
    int nx, nz;
};

// in_col: shared-memory column of this lane, row r of the image stored at in_col[(r - in_r0) * 32]
__device__ __forceinline__ void fir8(const float* in_col, int in_r0, const float* taps, int Tp, int shift, int m0,
                                     float (&acc)[8]) {
    const int c = m0 + shift;
    const float* base = in_col + (c - in_r0) * 32;
    float w[15];
#pragma unroll
    for (int e = 0; e < 7; ++e) w[8 + e] = base[(1 + e) * 32];
#pragma unroll
    for (int r = 0; r < 8; ++r) acc[r] = 0.0f;
    for (int tb = 0; tb < Tp; tb += 8) {
#pragma unroll
        for (int d = 0; d < 8; ++d) w[d] = base[(d - 7 - tb) * 32];
#pragma unroll
        for (int tt = 0; tt < 8; ++tt) {
            const float h = taps[tb + tt];
#pragma unroll
            for (int r = 0; r < 8; ++r) acc[r] = fmaf(h, w[r - tt + 7], acc[r]);
        }
#pragma unroll
        for (int d = 6; d >= 0; --d) w[d + 8] = w[d];
    }
}

template <int TZ, bool ENV>
__global__ void __launch_bounds__(256) post_fir_kernel(const PostParams P) {
    extern __shared__ float post_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int col0 = blockIdx.x * 32, r0 = blockIdx.y * TZ, f = blockIdx.z;
    const int col = col0 + lane;
    // y rows this block needs and x rows those need
    const int yr0 = ENV ? r0 + P.shiftH - P.TpH + 1 : r0;
    const int YR = ENV ? ((TZ + P.TpH - 1 + 7) & ~7) : TZ;
    const int xr0 = yr0 + P.shiftB - P.TpB + 1;
    const int XR = YR + P.TpB - 1;
    float* xs = post_smem;                    // [XR][32]
    float* ys = xs + XR * 32;            // [YR][32]   (ENV only)
    float* hb = ys + (ENV ? YR * 32 : 0);   // [TpB]
    float* hh = hb + P.TpB;              // [TpH]
    for (int t = threadIdx.x; t < P.TpB; t += 256) hb[t] = P.taps_bp[t];
    if (ENV) for (int t = threadIdx.x; t < P.TpH; t += 256) hh[t] = P.taps_h[t];
    const float* img = P.x + (size_t)f * P.nz * P.nx;
    for (int r = warp; r < XR; r += 8) {
        const int gr = xr0 + r;
        xs[r * 32 + lane] = (gr >= 0 && gr < P.nz && col < P.nx) ? img[(size_t)gr * P.nx + col] : 0.0f;
    }
    __syncthreads();
    float acc[8];
    if constexpr (!ENV) {
        for (int g = warp; g < TZ / 8; g += 8) {
            const int m0 = r0 + g * 8;
            fir8(xs + lane, xr0, hb, P.TpB, P.shiftB, m0, acc);
#pragma unroll
            for (int r = 0; r < 8; ++r)
                if (m0 + r < P.nz && col < P.nx) P.out[((size_t)f * P.nz + m0 + r) * P.nx + col] = acc[r];
        }
    } else {
    for (int g = warp; g < YR / 8; g += 8) {
        const int m0 = yr0 + g * 8;
        fir8(xs + lane, xr0, hb, P.TpB, P.shiftB, m0, acc);
#pragma unroll
        for (int r = 0; r < 8; ++r) ys[(g * 8 + r) * 32 + lane] = (m0 + r >= 0 && m0 + r < P.nz) ? acc[r] : 0.0f;
    }
    __syncthreads();
    float vmax = 0.0f;
    for (int g = warp; g < TZ / 8; g += 8) {
        const int m0 = r0 + g * 8;
        fir8(ys + lane, yr0, hh, P.TpH, P.shiftH, m0, acc);
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const float y = ys[(m0 + r - yr0) * 32 + lane];
            const float env = sqrtf(fmaf(y, y, acc[r] * acc[r]));
            if (m0 + r < P.nz && col < P.nx) {
                P.out[((size_t)f * P.nz + m0 + r) * P.nx + col] = env;
                vmax = fmaxf(vmax, env);
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) vmax = fmaxf(vmax, __shfl_xor_sync(0xffffffffu, vmax, o));
    if (lane == 0 && vmax > 0.0f) atomicMax(P.frame_max + f, __float_as_uint(vmax));
    }
}

// a9: out = max(20 log10(env / M_frame), -DR); env = 0 or M = 0 gives -DR (A10).  In place.
// grid: (ceil(npix / 1024), F), 256 threads x 4 pixels.
__global__ void __launch_bounds__(256) post_log_kernel(float* __restrict__ img, const unsigned int* __restrict__ frame_max,
                                                        int npix, float dyn_range_db) {
    const int f = blockIdx.y;
    const float M = __uint_as_float(frame_max[f]);
    const float lgM = lg2_approx(M);
    float* p = img + (size_t)f * npix;
    const float k = 6.02059991327962f;   // 20 log10(2)
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int i = (blockIdx.x * 4 + u) * 256 + threadIdx.x;
        if (i < npix) {
            const float e = p[i];
            float v = -dyn_range_db;
            if (M > 0.0f && e > 0.0f) v = fmaxf(k * (lg2_approx(e) - lgM), -dyn_range_db);
            p[i] = v;
        }
    }
}

__device__ __forceinline__ float log_db(float e, float M, float lgM, float dr) {
    const float k = 6.02059991327962f;   // 20 log10(2)
    return (M > 0.0f && e > 0.0f) ? fmaxf(k * (lg2_approx(e) - lgM), -dr) : -dr;
}

// The same for npix a multiple of 4 at a 16-byte aligned address.  grid: (ceil(npix / 4096), F), 256 threads x 4 x 128 bit.
__global__ void __launch_bounds__(256) post_log_vec_kernel(float4* __restrict__ img, const unsigned int* __restrict__ frame_max,
                                                            int npix4, float dyn_range_db) {
    const int f = blockIdx.y;
    const float M = __uint_as_float(frame_max[f]);
    const float lgM = lg2_approx(M);
    float4* p = img + (size_t)f * npix4;
    float4 e[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int i = (blockIdx.x * 4 + u) * 256 + threadIdx.x;
        e[u] = i < npix4 ? p[i] : make_float4(0.f, 0.f, 0.f, 0.f);
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const int i = (blockIdx.x * 4 + u) * 256 + threadIdx.x;
        if (i < npix4)
            __stcs(p + i, make_float4(log_db(e[u].x, M, lgM, dyn_range_db), log_db(e[u].y, M, lgM, dyn_range_db),
                                      log_db(e[u].z, M, lgM, dyn_range_db), log_db(e[u].w, M, lgM, dyn_range_db)));
    }
}

inline void launch_post_log(float* out, const unsigned int* frame_max, int npix, int F, float dr, cudaStream_t st) {
    if (npix % 4 == 0 && (reinterpret_cast<uintptr_t>(out) & 15) == 0)
        post_log_vec_kernel<<<dim3((npix / 4 + 1023) / 1024, F), 256, 0, st>>>((float4*)out, frame_max, npix / 4, dr);
    else
        post_log_kernel<<<dim3((npix + 1023) / 1024, F), 256, 0, st>>>(out, frame_max, npix, dr);
}

}  // namespace pab
