// pab_post.cuh -- fast path of the post chain (a7 + a8) for filters of <= 64 taps: the taps travel in the
// kernel parameter block (constant bank), so after full unrolling every FFMA takes its tap as a constant
// operand and the inner loop has no tap loads; structurally zero taps (every other tap of the type-III
// Hilbert FIR, reading A9) are skipped at compile time.  Same definitions as post_fir_kernel:
//   y[m] = sum_{t<T} h[t] x[m + T/2 - t]      (A11, A12)      q[m] = sum_{t'} g[t'] y[m + L - t']   (A9)
//   env = sqrt(y^2 + q^2), per-frame max by atomicMax on the bit pattern.
#pragma once
#include <cuda.h>            // CUtensorMap (the encode function itself is fetched through the runtime, no libcuda link)
#include <cuda_runtime.h>
#include "pab_math.cuh"
#include "pab_pipe.cuh"   // mbarrier / bulk-copy helpers

namespace pab {

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


// Blackwell packed fp32 FMA (FFMA2): two independent fp32 FMAs, each rounded as fmaf, in one issue slot.
__device__ __forceinline__ float2 ffma2(float2 a, float2 b, float2 c) {
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;"
        : "=l"(r)
        : "l"(reinterpret_cast<unsigned long long&>(a)), "l"(reinterpret_cast<unsigned long long&>(b)),
          "l"(reinterpret_cast<unsigned long long&>(c)));
    return reinterpret_cast<float2&>(r);
}

// R consecutive output rows of one column, dense taps; base = in_col + (m0 + shift - 63 - in_r0) * 32 is window row 0.
// The two FMAs of an FFMA2 take neighbouring taps and neighbouring window rows (an aligned register pair), so even
// output rows pair taps (0,1),(2,3).. and odd rows (1,2),(3,4).. from the shifted copy, with taps 0 and 63 on their
// own; the two partial sums of a row are added at the end: 33.5 instructions per row for 64 taps.
template <int R>
__device__ __forceinline__ void fir_dense64(const float* base, const float (&hr)[64], const float (&hs)[64],
                                            float (&out)[R]) {
    static_assert(R % 2 == 0, "rows are produced in pairs");
    float w[R + 63];
#pragma unroll
    for (int a = 0; a < R + 63; ++a) w[a] = base[a * 32];
#pragma unroll
    for (int r = 0; r < R; r += 2) {
        float2 e = make_float2(0.0f, 0.0f);
        float2 o = make_float2(hr[0] * w[r + 1], hr[63] * w[r + 64]);
#pragma unroll
        for (int j = 0; j < 64; j += 2) {
            const float2 x = make_float2(w[r + j], w[r + j + 1]);
            e = ffma2(make_float2(hr[j], hr[j + 1]), x, e);
            if (j >= 2) o = ffma2(make_float2(hs[j], hs[j + 1]), x, o);
        }
        out[r] = e.x + e.y;
        out[r + 1] = o.x + o.y;
    }
}

// The same for taps that are non-zero only at reversed index parity Q (type-III Hilbert FIR, reading A9): every tap
// serves two neighbouring output rows in one FFMA2 (tap stored twice in hd), the window pairs all start at parity Q:
// 16 instructions per row for the 32 taps.
template <int R, int Q>
__device__ __forceinline__ void fir_parity64(const float* base, const float (&hd)[64], float (&out)[R]) {
    static_assert(R % 2 == 0, "rows are produced in pairs");
    float w[R + 63];
#pragma unroll
    for (int a = Q; a < R + 62 + Q; ++a) w[a] = base[a * 32];
    float2 acc[R / 2];
#pragma unroll
    for (int r = 0; r < R / 2; ++r) acc[r] = make_float2(0.0f, 0.0f);
#pragma unroll
    for (int i = 0; i < 32; ++i) {
        const float2 h = make_float2(hd[2 * i], hd[2 * i + 1]);
#pragma unroll
        for (int r = 0; r < R; r += 2) acc[r / 2] = ffma2(h, make_float2(w[r + Q + 2 * i], w[r + Q + 2 * i + 1]), acc[r / 2]);
    }
#pragma unroll
    for (int r = 0; r < R; r += 2) { out[r] = acc[r / 2].x; out[r + 1] = acc[r / 2].y; }
}

// HPAR = parity of the non-zero ORIGINAL Hilbert taps (0 / 1), 2 = dense
template <int R, int HPAR>
__device__ __forceinline__ void fir_hilbert64(const float* base, const PostTaps64& T, float (&out)[R]) {
    if constexpr (HPAR == 2) fir_dense64<R>(base, T.hhr, T.hhs, out);
    else fir_parity64<R, 1 - HPAR>(base, T.hhd, out);
}

constexpr int kPostFastTZ = 256;

// 3-D tiled TMA load of a box of rows x 32 columns of frame f, first row r (may be negative), first column c; rows and
// columns outside the image arrive as zeros.
__device__ __forceinline__ void tma_box(uint32_t dst, const CUtensorMap* tm, int c, int r, int f, uint32_t bar) {
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
                 ::"r"(dst), "l"(tm), "r"(c), "r"(r), "r"(f), "r"(bar) : "memory");
}

// grid: (ceil(nx/32), ceil(nz/TZ), F), 256 threads; lanes own columns.
// LD = 2 (rows of a multiple of 16 bytes at a 16-byte aligned address): the tile comes in as two boxes of a tiled TMA
// tensor copy over the [F][nz][nx] image (one thread issues both; the halo outside the image is zero-filled by the copy
// engine).  LD = 1 (nx a multiple of 32, no tensor map): one 1-D bulk copy per 128-byte tile row -- 350 copies issued lane
// by lane, a fifth of the CTA's time.  LD = 0: plain predicated loads.
template <int TZ, bool ENV, int HPAR, int LD>
__global__ void __launch_bounds__(256) post_fir64_kernel(const PostParams P, const __grid_constant__ PostTaps64 T,
                                                          const __grid_constant__ CUtensorMap TM) {
    extern __shared__ __align__(128) float post64_smem[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int col0 = blockIdx.x * 32, r0 = blockIdx.y * TZ, f = blockIdx.z;
    const int col = col0 + lane;
    const int yr0 = ENV ? r0 + P.shiftH - 63 : r0;           // first y row this block needs
    constexpr int YR = ENV ? ((TZ + 63 + 7) & ~7) : TZ;
    const int xr0 = yr0 + P.shiftB - 63;                     // first x row those need
    constexpr int XR = YR + 63;
    constexpr int XRA = XR + 1;         // two TMA boxes of XRA / 2 rows
    float* xs = post64_smem;            // [XRA][32]
    float* ys = xs + XRA * 32;          // [YR][32]   (ENV only)
    const float* img = P.x + (size_t)f * P.nz * P.nx;
    if constexpr (LD == 2) {
        __shared__ __align__(8) unsigned long long bar;
        const uint32_t barA = smem_u32(&bar);
        if (threadIdx.x == 0) {
            mbar_init(barA, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            mbar_arrive_expect_tx(barA, (uint32_t)XRA * 128u);
            tma_box(smem_u32(xs), &TM, col0, xr0, f, barA);
            tma_box(smem_u32(xs) + (XRA / 2) * 128, &TM, col0, xr0 + XRA / 2, f, barA);
        }
        __syncthreads();
        mbar_wait(barA, 0);
    } else if constexpr (LD == 1) {
        __shared__ __align__(8) unsigned long long bar;
        const uint32_t barA = smem_u32(&bar);
        const int lo = max(0, -xr0), hi = min(XR, P.nz - xr0);           // tile rows [lo, hi) lie inside the image
        if (threadIdx.x == 0) {
            mbar_init(barA, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            mbar_arrive_expect_tx(barA, (uint32_t)(hi - lo) * 128u);
        }
        __syncthreads();
        const uint32_t xsA = smem_u32(xs);
        for (int r = threadIdx.x; r < XR; r += 256) {
            if (r >= lo && r < hi) bulk_g2s(xsA + r * 128, img + (size_t)(xr0 + r) * P.nx + col0, 128u, barA);
            else {
#pragma unroll
                for (int c = 0; c < 32; c += 4) *reinterpret_cast<float4*>(xs + r * 32 + c) = make_float4(0.f, 0.f, 0.f, 0.f);
            }
        }
        mbar_wait(barA, 0);
    } else {
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
            fir_dense64<16>(xs + lane + (m0 + P.shiftB - 63 - xr0) * 32, T.hbr, T.hbs, a16);
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
            fir_dense64<16>(xs + lane + (m0 + P.shiftB - 63 - xr0) * 32, T.hbr, T.hbs, a16);
#pragma unroll
            for (int r = 0; r < 16; ++r) ys[(y0 + g * 16 + r) * 32 + lane] = (m0 + r >= 0 && m0 + r < P.nz) ? a16[r] : 0.0f;
        }
        {
            const int m0 = yr0 + y0 + 32;
            fir_dense64<8>(xs + lane + (m0 + P.shiftB - 63 - xr0) * 32, T.hbr, T.hbs, a8);
#pragma unroll
            for (int r = 0; r < 8; ++r) ys[(y0 + 32 + r) * 32 + lane] = (m0 + r >= 0 && m0 + r < P.nz) ? a8[r] : 0.0f;
        }
        __syncthreads();
        float vmax = 0.0f;
#pragma unroll 1
        for (int g = 0; g < 2; ++g) {
            const int m0 = r0 + warp * 32 + g * 16;
            fir_hilbert64<16, HPAR>(ys + lane + (m0 + P.shiftH - 63 - yr0) * 32, T, a16);
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const float y = ys[(m0 + r - yr0) * 32 + lane];
                const float env = sqrt_approx(fmaf(y, y, a16[r] * a16[r]));
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

inline int post64_box_rows(bool env) {
    const int YR = env ? ((kPostFastTZ + 63 + 7) & ~7) : kPostFastTZ;
    return (YR + 64) / 2;
}
inline size_t post64_smem_bytes(bool env) {
    const int YR = env ? ((kPostFastTZ + 63 + 7) & ~7) : kPostFastTZ;
    return ((size_t)(YR + 64) * 32 + (env ? (size_t)YR * 32 : 0)) * 4;
}

template <int BULK>
inline cudaError_t post64_configure_b(int smem_optin) {
    cudaError_t e;
    smem_optin = (int)post64_smem_bytes(true);   // what the kernels use (the bulk variant adds a static mbarrier)
    if ((e = cudaFuncSetAttribute(post_fir64_kernel<kPostFastTZ, false, 2, BULK>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(post_fir64_kernel<kPostFastTZ, true, 0, BULK>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(post_fir64_kernel<kPostFastTZ, true, 1, BULK>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(post_fir64_kernel<kPostFastTZ, true, 2, BULK>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
}

inline cudaError_t post64_configure(int smem_optin) {
    cudaError_t e = post64_configure_b<0>(smem_optin);
    if (e == cudaSuccess) e = post64_configure_b<1>(smem_optin);
    return e != cudaSuccess ? e : post64_configure_b<2>(smem_optin);
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (libpab.so does not link libcuda); nullptr: unavailable
using TensorMapEncodeFn = CUresult (*)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                       const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                       CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
inline TensorMapEncodeFn tensor_map_encode_fn() {
    static const TensorMapEncodeFn fn = [] {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess || q != cudaDriverEntryPointSuccess)
            p = nullptr;
        return reinterpret_cast<TensorMapEncodeFn>(p);
    }();
    return fn;
}
// tensor map of the [F][nz][nx] fp32 image with boxes of box_rows x 32 columns; false: not expressible / no driver support
inline bool post64_tensor_map(const float* x, int nx, int nz, int F, int box_rows, CUtensorMap* tm) {
    const TensorMapEncodeFn enc = tensor_map_encode_fn();
    if (!enc || nx % 4 != 0 || (reinterpret_cast<uintptr_t>(x) & 15) != 0) return false;
    const cuuint64_t dims[3] = {(cuuint64_t)nx, (cuuint64_t)nz, (cuuint64_t)F};
    const cuuint64_t strides[2] = {(cuuint64_t)nx * 4, (cuuint64_t)nx * nz * 4};
    const cuuint32_t box[3] = {32, (cuuint32_t)box_rows, 1}, estr[3] = {1, 1, 1};
    return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(x), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int LD>
inline void launch_post64_b(const PostParams& Q, const PostTaps64& T, const CUtensorMap& tm, bool env, int hpar, int F, cudaStream_t st) {
    dim3 grid((Q.nx + 31) / 32, (Q.nz + kPostFastTZ - 1) / kPostFastTZ, F);
    const size_t sm = post64_smem_bytes(env);
    if (!env) post_fir64_kernel<kPostFastTZ, false, 2, LD><<<grid, 256, sm, st>>>(Q, T, tm);
    else if (hpar == 0) post_fir64_kernel<kPostFastTZ, true, 0, LD><<<grid, 256, sm, st>>>(Q, T, tm);
    else if (hpar == 1) post_fir64_kernel<kPostFastTZ, true, 1, LD><<<grid, 256, sm, st>>>(Q, T, tm);
    else post_fir64_kernel<kPostFastTZ, true, 2, LD><<<grid, 256, sm, st>>>(Q, T, tm);
}

inline void launch_post64(const PostParams& Q, const PostTaps64& T, bool env, int hpar, int F, cudaStream_t st) {
    alignas(64) CUtensorMap tm{};
    if (post64_tensor_map(Q.x, Q.nx, Q.nz, F, post64_box_rows(env), &tm)) launch_post64_b<2>(Q, T, tm, env, hpar, F, st);
    // bulk row copies need 128-byte rows of whole tiles at 16-byte aligned addresses
    else if (Q.nx % 32 == 0 && (reinterpret_cast<uintptr_t>(Q.x) & 15) == 0) launch_post64_b<1>(Q, T, tm, env, hpar, F, st);
    else launch_post64_b<0>(Q, T, tm, env, hpar, F, st);
}

}  // namespace pab
