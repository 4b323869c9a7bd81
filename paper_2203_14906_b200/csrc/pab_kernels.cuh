// pab_kernels.cuh -- ingest (a1) and direct beamforming (a2..a6, a10) kernels (translation unit pab_tu_direct.cu).
// The staged (bulk-copy + mbarrier) beamforming kernel lives in pab_staged.cuh, the post chain in pab_post.cuh.
#pragma once
#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>
#include "pab_math.cuh"
#include "pab_types.h"

namespace pab {

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


// ---- host side ----
template <typename T>
inline void launch_ingest_quad(const void* rf, float* stage, int F, int N, int S, float scale, cudaStream_t st) {
    const int nq = (F + 3) / 4;
    dim3 grid((S + 1023) / 1024, N, nq);
    if constexpr (std::is_same<T, float>::value) {
        if (S % 4 == 0 && (reinterpret_cast<uintptr_t>(rf) & 15) == 0) {
            ingest_quad_vec_kernel<<<dim3((S / 4 + 255) / 256, N, nq), 256, 0, st>>>((const float4*)rf, (float4*)stage, F, N, S / 4, scale);
            return;
        }
    }
    ingest_quad_kernel<T><<<grid, 256, 0, st>>>((const T*)rf, (float4*)stage, F, N, S, scale);
}
template <typename T>
inline void launch_ingest_lin(const void* rf, float* stage, int F, int N, int S, int Sp, float scale, cudaStream_t st) {
    dim3 grid((Sp + 255) / 256, N, F);
    ingest_lin_kernel<T><<<grid, 256, 0, st>>>((const T*)rf, stage, N, S, Sp, scale);
}

template <int K, int NQ, int W>
inline void launch_direct(const BfParams& P, int groups, cudaStream_t st) {
    dim3 grid((P.nx + kDirectCols - 1) / kDirectCols, (P.nz + kDirectRows - 1) / kDirectRows, groups);
    bf_direct_kernel<K, NQ, W><<<grid, 256, 0, st>>>(P);
}

template <int NQ, int W>
inline void launch_direct_order_w(int order, const BfParams& P, int groups, cudaStream_t st) {
    switch (order) {
    case 1: launch_direct<1, NQ, W>(P, groups, st); break;
    case 2: launch_direct<2, NQ, W>(P, groups, st); break;
    case 3: launch_direct<3, NQ, W>(P, groups, st); break;
    case 4: launch_direct<4, NQ, W>(P, groups, st); break;
    case 5: launch_direct<5, NQ, W>(P, groups, st); break;
    default:
        if constexpr (NQ <= 1 && W == 0) {          // orders 6..8: at most 4 frames per thread, no weighting
            if (order == 6) launch_direct<6, NQ, W>(P, groups, st);
            else if (order == 7) launch_direct<7, NQ, W>(P, groups, st);
            else launch_direct<8, NQ, W>(P, groups, st);
        }
        break;
    }
}

// nq = 0: lin layout, one frame per thread; 1, 2, 4 quads per thread (4 only without weighting)
inline void launch_direct_nq(int order, int nq, int weight, const BfParams& P, int groups, cudaStream_t st) {
    if (weight == 0) {
        if (nq == 4) launch_direct_order_w<4, 0>(order, P, groups, st);
        else if (nq == 2) launch_direct_order_w<2, 0>(order, P, groups, st);
        else if (nq == 1) launch_direct_order_w<1, 0>(order, P, groups, st);
        else launch_direct_order_w<0, 0>(order, P, groups, st);
    } else {
        if (nq == 2) launch_direct_order_w<2, 1>(order, P, groups, st);
        else if (nq == 1) launch_direct_order_w<1, 1>(order, P, groups, st);
        else launch_direct_order_w<0, 1>(order, P, groups, st);
    }
}

}  // namespace pab
