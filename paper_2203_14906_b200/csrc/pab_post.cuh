// pab_post.cuh -- fast path of the post chain (a7 + a8) for filters of <= 64 taps: the taps travel in the
// kernel parameter block (constant bank), so after full unrolling every FFMA takes its tap as a constant
// operand and the inner loop has no tap loads; structurally zero taps (every other tap of the type-III
// Hilbert FIR, reading A9) are skipped at compile time.  Same definitions as post_fir_kernel:
//   y[m] = sum_{t<T} h[t] x[m + T/2 - t]      (A11, A12)      q[m] = sum_{t'} g[t'] y[m + L - t']   (A9)
//   env = sqrt(y^2 + q^2), per-frame max by atomicMax on the bit pattern.
#pragma once
#include <cuda_runtime.h>
#include "pab_kernels.cuh"

namespace pab {

struct PostTaps64 {
    float hb[64];   // band-pass taps, zero-padded
    float hh[64];   // Hilbert taps g[t' ] = g(t' - L), zero-padded
};

// R (8 or 16) consecutive output rows m0..m0+R-1 of one column: out[m] = sum_t taps[t] in[m + shift - t], t < 64, from
// an (R + 7)-row register window that slides 8 rows per block of 8 taps: 8 R FMAs per 8 shared loads.
// PAR = 0 / 1: only taps of that index parity are non-zero; PAR = 2: dense.
template <int R, int PAR>
__device__ __forceinline__ void fir_c64(const float* in_col, int in_r0, const float (&taps)[64], int shift, int m0,
                                        float (&acc)[R]) {
    const float* base = in_col + (m0 + shift - in_r0) * 32;
    float w[R + 7];
#pragma unroll
    for (int e = 0; e < R - 1; ++e) w[8 + e] = base[(1 + e) * 32];
#pragma unroll
    for (int r = 0; r < R; ++r) acc[r] = 0.0f;
#pragma unroll
    for (int tb = 0; tb < 64; tb += 8) {
#pragma unroll
        for (int d = 0; d < 8; ++d) w[d] = base[(d - 7 - tb) * 32];
#pragma unroll
        for (int tt = 0; tt < 8; ++tt) {
            if (PAR == 2 || ((tb + tt) & 1) == PAR) {
                const float h = taps[tb + tt];
#pragma unroll
                for (int r = 0; r < R; ++r) acc[r] = fmaf(h, w[r - tt + 7], acc[r]);
            }
        }
#pragma unroll
        for (int d = R - 2; d >= 0; --d) w[d + 8] = w[d];
    }
}

constexpr int kPostFastTZ = 256;

// grid: (ceil(nx/32), ceil(nz/TZ), F), 256 threads; lanes own columns.
template <int TZ, bool ENV, int HPAR>
__global__ void __launch_bounds__(256) post_fir64_kernel(const PostParams P, const __grid_constant__ PostTaps64 T) {
    extern __shared__ float post64_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int col0 = blockIdx.x * 32, r0 = blockIdx.y * TZ, f = blockIdx.z;
    const int col = col0 + lane;
    const int yr0 = ENV ? r0 + P.shiftH - 63 : r0;           // first y row this block needs
    constexpr int YR = ENV ? ((TZ + 63 + 7) & ~7) : TZ;
    const int xr0 = yr0 + P.shiftB - 63;                     // first x row those need
    constexpr int XR = YR + 63;
    float* xs = post64_smem;            // [XR][32]
    float* ys = xs + XR * 32;           // [YR][32]   (ENV only)
    const float* img = P.x + (size_t)f * P.nz * P.nx;
    // tile load: 16 rows per warp in flight at a time (the loop is latency-bound otherwise)
    constexpr int kRowsPerWarp = (XR + 7) / 8;
#pragma unroll 1
    for (int k0 = 0; k0 < kRowsPerWarp; k0 += 16) {
        float v[16];
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const int r = warp + 8 * (k0 + k), gr = xr0 + r;
            v[k] = (r < XR && gr >= 0 && gr < P.nz && col < P.nx) ? __ldg(img + (size_t)gr * P.nx + col) : 0.0f;
        }
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const int r = warp + 8 * (k0 + k);
            if (r < XR) xs[r * 32 + lane] = v[k];
        }
    }
    __syncthreads();
    // every warp owns a slab of consecutive rows: 32 output rows (two 16-row groups), and with the envelope 40 rows of
    // the band-pass intermediate (16 + 16 + 8): the same work for all 8 warps
    static_assert(TZ == 256, "the row slabs below assume 256-row tiles and 8 warps");
    float a16[16], a8[8];
    if constexpr (!ENV) {
#pragma unroll 1
        for (int g = 0; g < 2; ++g) {
            const int m0 = r0 + warp * 32 + g * 16;
            fir_c64<16, 2>(xs + lane, xr0, T.hb, P.shiftB, m0, a16);
#pragma unroll
            for (int r = 0; r < 16; ++r)
                if (m0 + r < P.nz && col < P.nx) P.out[((size_t)f * P.nz + m0 + r) * P.nx + col] = a16[r];
        }
    } else {
        static_assert(!ENV || YR == 320, "band-pass intermediate: 8 slabs of 40 rows");
        const int y0 = warp * 40;                                  // first row of this warp's slab, relative to yr0
#pragma unroll 1
        for (int g = 0; g < 2; ++g) {
            const int m0 = yr0 + y0 + g * 16;
            fir_c64<16, 2>(xs + lane, xr0, T.hb, P.shiftB, m0, a16);
#pragma unroll
            for (int r = 0; r < 16; ++r) ys[(y0 + g * 16 + r) * 32 + lane] = (m0 + r >= 0 && m0 + r < P.nz) ? a16[r] : 0.0f;
        }
        {
            const int m0 = yr0 + y0 + 32;
            fir_c64<8, 2>(xs + lane, xr0, T.hb, P.shiftB, m0, a8);
#pragma unroll
            for (int r = 0; r < 8; ++r) ys[(y0 + 32 + r) * 32 + lane] = (m0 + r >= 0 && m0 + r < P.nz) ? a8[r] : 0.0f;
        }
        __syncthreads();
        float vmax = 0.0f;
#pragma unroll 1
        for (int g = 0; g < 2; ++g) {
            const int m0 = r0 + warp * 32 + g * 16;
            fir_c64<16, HPAR>(ys + lane, yr0, T.hh, P.shiftH, m0, a16);
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const float y = ys[(m0 + r - yr0) * 32 + lane];
                const float env = sqrtf(fmaf(y, y, a16[r] * a16[r]));
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

inline size_t post64_smem_bytes(bool env) {
    const int YR = env ? ((kPostFastTZ + 63 + 7) & ~7) : kPostFastTZ;
    return ((size_t)(YR + 63) * 32 + (env ? (size_t)YR * 32 : 0)) * 4;
}

inline cudaError_t post64_configure(int smem_optin) {
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(post_fir64_kernel<kPostFastTZ, false, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(post_fir64_kernel<kPostFastTZ, true, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(post_fir64_kernel<kPostFastTZ, true, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(post_fir64_kernel<kPostFastTZ, true, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
}

inline void launch_post64(const PostParams& Q, const PostTaps64& T, bool env, int hpar, int F, cudaStream_t st) {
    dim3 grid((Q.nx + 31) / 32, (Q.nz + kPostFastTZ - 1) / kPostFastTZ, F);
    const size_t sm = post64_smem_bytes(env);
    if (!env) post_fir64_kernel<kPostFastTZ, false, 2><<<grid, 256, sm, st>>>(Q, T);
    else if (hpar == 0) post_fir64_kernel<kPostFastTZ, true, 0><<<grid, 256, sm, st>>>(Q, T);
    else if (hpar == 1) post_fir64_kernel<kPostFastTZ, true, 1><<<grid, 256, sm, st>>>(Q, T);
    else post_fir64_kernel<kPostFastTZ, true, 2><<<grid, 256, sm, st>>>(Q, T);
}

}  // namespace pab
