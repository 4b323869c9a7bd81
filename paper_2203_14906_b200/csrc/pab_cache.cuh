// pab_cache.cuh -- the cached-delay variant of the fused beamforming kernel (BASELINE.json north_star: "Per-pixel
// delays are computed in-kernel, with no delay table, or from a cached ... table where ncu shows it wins").
//
// The delay of a (pixel, element) pair does not depend on the frame.  With many frames per thread its cost is
// amortised (bf_staged_kernel); with one frame per thread (calls of 1..3 frames) the ~35 instructions of
// delay_tap dominate the ~9 of the rest.  Here the interpolation tap of every (pixel, element) is computed ONCE
// per geometry, in fp64, and kept in device memory as one 32-bit word: 12 bits of integer sample offset from
// the staged window's start and 20 bits of fraction (2^-21 samples worst-case rounding).  It is the paper's own
// arrangement (delays "calculated and stored in the GPU (global) memory") with the table laid out
// tile-major, [tile row][tile col][element][8 cols][64 rows], so the 2 KB block of one (tile, element) is
// contiguous and the producer warp stages it by one bulk copy beside that element's RF window.  In-range
// geometries only (no out-of-record pixels); the window start of every (tile, element) is stored beside it so
// that the table and the staged window agree exactly.
#pragma once
#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>
#include "pab_math.cuh"
#include "pab_pipe.cuh"

namespace pab {

// grid: (tiles_x, tiles_z, N), 512 threads = one tile.  taps[((tile * N + i) * 8 + col) * 64 + row], w0s[tile * N + i]
__global__ void __launch_bounds__(kStgRows * kStgCols) delay_cache_kernel(const CacheGeom G, uint32_t* __restrict__ taps,
                                                                           int* __restrict__ w0s) {
    __shared__ int s_min;
    const int col = threadIdx.x / kStgRows, row = threadIdx.x % kStgRows;
    const int j = min((int)blockIdx.x * kStgCols + col, G.nx - 1), m = min((int)blockIdx.y * G.tile_rows + min(row, G.tile_rows - 1), G.nz - 1);
    const int i = blockIdx.z;
    // the definition, every operation individually rounded in fp64 (readings A5)
    const double x = __dadd_rn(G.x0, __dmul_rn((double)j, G.dx));
    const double z = __dadd_rn(G.z0, __dmul_rn((double)m, G.dz));
    const double xe = __dmul_rn(__dsub_rn((double)i, __ddiv_rn(__dsub_rn((double)G.N, 1.0), 2.0)), G.pitch);
    const double ddx = __dsub_rn(x, xe);
    const double idx = __ddiv_rn(__dmul_rn(G.fs, __dsqrt_rn(__dadd_rn(__dmul_rn(ddx, ddx), __dmul_rn(z, z)))), G.c);
    if (threadIdx.x == 0) s_min = 0x7fffffff;
    __syncthreads();
    atomicMin(&s_min, (int)floor(idx));
    __syncthreads();
    const int w0 = max(s_min - 1, 0) & ~3;
    const size_t blk = ((size_t)blockIdx.y * G.tiles_x + blockIdx.x) * G.N + i;
    if (threadIdx.x == 0) w0s[blk] = w0;
    const double rel = idx - (double)w0;                                 // >= 0, < window
    if (taps) taps[blk * (kStgRows * kStgCols) + threadIdx.x] = (uint32_t)llrint(rel * (double)(1u << kCacheFracBits));
}

// Compact table for translation-invariant geometries (pitch = q dx with an integer q, exactly): the lateral offset
// of (column j, element i) is x0 + (d - q (N-1)/2) dx with d = j - q i + q (N-1), so the tap depends on (d, row)
// only: nd = nx + q (N-1) columns instead of nx N -- 2 MB instead of 134 MB at C2, resident in L2/L1.
// compact[d * nz + m] = (floor(idx), fraction as float bits).  grid: (ceil(nz/256), nd)
__global__ void __launch_bounds__(256) delay_compact_kernel(const CacheGeom G, int q, uint2* __restrict__ compact) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x, d = blockIdx.y;
    if (m >= G.nz) return;
    const double z = __dadd_rn(G.z0, __dmul_rn((double)m, G.dz));
    const double ddx = __dadd_rn(G.x0, __dmul_rn(__dsub_rn((double)d, __dmul_rn((double)q, __ddiv_rn(__dsub_rn((double)G.N, 1.0), 2.0))), G.dx));
    const double idx = __ddiv_rn(__dmul_rn(G.fs, __dsqrt_rn(__dadd_rn(__dmul_rn(ddx, ddx), __dmul_rn(z, z)))), G.c);
    const double fl = floor(idx);
    compact[(size_t)d * G.nz + m] = make_uint2((unsigned)(int)fl, __float_as_uint((float)(idx - fl)));
}

__device__ __forceinline__ uint32_t lds32u(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}

// NQ = 0: lin layout, one frame per thread; NQ = 4 (orders 1..3) / NQ = 2 (orders 4, 5): quad layout, 16 / 8 frames
// per thread.  In-range geometries.
// COMPACT: taps come from the (d, row) table through L1/L2 (q = pitch / dx), only the window starts are staged.
// W = 1: coherence-factor weighting (row f1), frame groups with the tile-major table only (NQ = 1, 2; orders 4, 5: NQ = 1).
// RM (root mix, order 3, 16 frames per thread): how many of a thread's 8 frame pairs take their cube root on the FMA
// pipe (cbrt_fma2) instead of the XU pipe: 0, 1 (pair 7) or 2 (pairs 3 and 7).
// R7: 56-row tiles (pab_pipe.cuh tile_row; orders 1, 2 with their own table set).
template <int K, int NQ, bool COMPACT, int W = 0, int RM = 0, bool R7 = false>
__global__ void __launch_bounds__(kStgThreads, 1) bf_cached_kernel(const BfParams P, const StagedCfg C,
                                                                    const uint32_t* __restrict__ taps,
                                                                    const int* __restrict__ w0s,
                                                                    const uint2* __restrict__ compact, int q) {
    constexpr int NF = NQ == 0 ? 1 : 4 * NQ;
    constexpr int BPS = NQ == 0 ? 4 : 16;
    constexpr int NCOPY = NQ == 0 ? 1 : NQ;
    extern __shared__ __align__(128) unsigned char stg_smem[];
    unsigned char* smem = stg_smem;
    const uint32_t bar0 = smem_u32(smem);
    // [stages][chunk] blocks of 512 uint32 taps, or (COMPACT) [stages][chunk] window starts
    constexpr int kBlk = COMPACT ? 4 : kCacheBlockBytes;
    const uint32_t ctab0 = bar0 + 64;
    const uint32_t data0 = ctab0 + ((C.stages * C.chunk * kBlk + 127) & ~127);
    const int quad_bytes = C.window * BPS;
    const int slot_bytes = quad_bytes * NCOPY;
    const int stage_bytes = C.chunk * slot_bytes;
    const uint32_t ebuf = data0 + C.stages * stage_bytes;          // epilogue transpose buffer (C.epi)
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_chunks = (P.N + C.chunk - 1) / C.chunk;
    const int n_tiles = C.tiles_x * C.tiles_z * C.groups;

    if (threadIdx.x == 0) {
        for (int s = 0; s < C.stages; ++s) {
            mbar_init(bar0 + 8 * s, C.chunk);
            mbar_init(bar0 + 8 * (C.stages + s), kStgConsumerWarps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == kStgConsumerWarps) {
        if (lane >= C.chunk) return;
        const size_t chan_stride = NQ == 0 ? (size_t)P.Sp * 4 : (size_t)P.S * 16;
        const size_t grp_stride = (size_t)P.N * chan_stride;
        const int row_len = NQ == 0 ? P.Sp : P.S;
        int s = 0;
        uint32_t ph = 1;
        for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            const int bz = tile % C.groups, txy = tile / C.groups;       // frame groups innermost: table blocks reused from L2
            const char* grp = reinterpret_cast<const char*>(P.rf) + (size_t)bz * (NQ == 0 ? 1 : NQ) * grp_stride;
            const size_t blk0 = (size_t)txy * P.N;
            for (int ck = 0; ck < n_chunks; ++ck) {
                const uint32_t full = bar0 + 8 * s, empty = bar0 + 8 * (C.stages + s);
                mbar_wait_relaxed(empty, ph);
                const int ch = ck * C.chunk + lane;
                if (ch < P.N) {
                    const int w0 = __ldg(w0s + blk0 + ch);
                    const int len = min(C.window, row_len - w0);
                    const uint32_t bytes = (uint32_t)len * BPS;
                    const int slot = s * stage_bytes + lane * slot_bytes;
                    if constexpr (COMPACT) {          // the shared address sample 0 of this channel would have
                        asm volatile("st.shared.u32 [%0], %1;" ::"r"(ctab0 + (s * C.chunk + lane) * 4),
                                     "r"(data0 + slot - (uint32_t)w0 * BPS) : "memory");
                        mbar_arrive_expect_tx(full, bytes * NCOPY);
                    } else {
                        mbar_arrive_expect_tx(full, bytes * NCOPY + kCacheBlockBytes);
                        bulk_g2s(ctab0 + (s * C.chunk + lane) * kCacheBlockBytes,
                                 taps + (blk0 + ch) * (size_t)(kStgRows * kStgCols), kCacheBlockBytes, full);
                    }
                    const char* src = grp + (size_t)ch * chan_stride + (size_t)w0 * BPS;
#pragma unroll
                    for (int c = 0; c < NCOPY; ++c)
                        bulk_g2s(data0 + slot + c * quad_bytes, src + c * grp_stride, bytes, full);
                } else {
                    mbar_arrive(full);
                }
                if (++s == C.stages) { s = 0; ph ^= 1; }
            }
        }
        return;
    }

    const int col = warp & 7;
    bool live;
    constexpr int TR = R7 ? 56 : kStgRows;
    const int trow = tile_row(TR, warp, lane, &live);                // this thread's row inside the tile
    const uint32_t my = (uint32_t)((col * kStgRows + trow) * 4);
    int s = 0;
    uint32_t ph = 0;
    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const int bz = tile % C.groups, txy = tile / C.groups;
        const int bx = txy % C.tiles_x, by = txy / C.tiles_x;
        const int j = bx * kStgCols + col;
        const int m = by * TR + trow;
        // one frame per thread: scalar accumulators; frame groups: the frames in pairs, packed f32x2 arithmetic
        float p[1][kAcc<K, W>];
        float2 pp[NQ == 0 ? 1 : NF / 2][kAcc<K, W>];
#pragma unroll
        for (int k = 0; k < kAcc<K, W>; ++k) p[0][k] = 0.0f;
#pragma unroll
        for (int f = 0; f < (NQ == 0 ? 1 : NF / 2); ++f)
#pragma unroll
            for (int k = 0; k < kAcc<K, W>; ++k) pp[f][k] = make_float2(0.0f, 0.0f);
        // COMPACT: this pixel's row of the (d, row) table; d = j - q i + q (N - 1) falls by q per element
        // (32-bit entry index: pab_set_delay_cache builds the compact table only below 2^31 entries)
        const uint32_t ci0 = (uint32_t)(min(j, P.nx - 1) + q * (P.N - 1)) * (uint32_t)P.nz + (uint32_t)min(m, P.nz - 1);
        const uint32_t cstep = (uint32_t)q * (uint32_t)P.nz;

        for (int ck = 0; ck < n_chunks; ++ck) {
            const int nch = min(C.chunk, P.N - ck * C.chunk);
            const uint32_t cik = ci0 - (uint32_t)(ck * C.chunk) * cstep;
            mbar_wait(bar0 + 8 * s, ph);
            const uint32_t ctab_s = ctab0 + s * C.chunk * kBlk + (COMPACT ? 0u : my);
            const uint32_t data_s = data0 + s * stage_bytes;
            constexpr int kElemUnroll = NQ >= 4 ? 2 : 4;
#pragma unroll (kElemUnroll)
            for (int l = 0; l < nch; ++l) {
                float a;
                uint32_t addr;
                if constexpr (COMPACT) {
                    const uint2 e = __ldg(compact + (cik - (uint32_t)l * cstep));
                    a = __uint_as_float(e.y);
                    addr = lds32u(ctab_s + l * 4) + e.x * BPS;
                } else {
                    const uint32_t e = lds32u(ctab_s + l * kCacheBlockBytes);
                    a = __uint_as_float(0x3F800000u | ((e << (32 - kCacheFracBits)) >> 9)) - 1.0f;          // fraction, exact
                    addr = data_s + l * slot_bytes + (e >> kCacheFracBits) * BPS;
                }
                if constexpr (NQ == 0) {
                    const float s0 = lds32(addr), s1 = lds32(addr + 4);
                    accumulate_w<K, W>(fmaf(a, s1 - s0, s0), p[0]);
                } else {
                    // quad c of the group (compile-time c: which of its two frame pairs takes the FMA-pipe root)
                    auto quad = [&](auto qc) {
                        constexpr int c = decltype(qc)::value;
                        const float4 s0 = lds128(addr + c * quad_bytes);
                        const float4 s1 = lds128(addr + c * quad_bytes + 16);
                        constexpr bool fma_root = K == 3 && NQ == 4 && W == 0 && ((RM == 2 && (c & 1)) || (RM == 1 && c == 3));
                        accumulate2_w<K, W>(interp2(a, make_float2(s0.x, s0.y), make_float2(s1.x, s1.y)), pp[2 * c + 0]);
                        accumulate2_w<K, W, fma_root>(interp2(a, make_float2(s0.z, s0.w), make_float2(s1.z, s1.w)), pp[2 * c + 1]);
                    };
                    quad(std::integral_constant<int, 0>{});
                    if constexpr (NQ >= 2) quad(std::integral_constant<int, 1>{});
                    if constexpr (NQ >= 4) { quad(std::integral_constant<int, 2>{}); quad(std::integral_constant<int, 3>{}); }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar0 + 8 * (C.stages + s));
            if (++s == C.stages) { s = 0; ph ^= 1; }
        }

        const size_t img = (size_t)P.nz * P.nx;
        if constexpr (NQ == 0) {
            if (live && j < P.nx && m < P.nz && bz < P.n_frames) P.out[(size_t)bz * img + (size_t)m * P.nx + j] = combine_w<K, W>(p[0], P.inv_n);
        } else if (C.epi) {
#pragma unroll
            for (int c = 0; c < NQ; ++c) {
                const float v[4] = {combine2_w<K, W>(pp[2 * c], 0, P.inv_n), combine2_w<K, W>(pp[2 * c], 1, P.inv_n),
                                    combine2_w<K, W>(pp[2 * c + 1], 0, P.inv_n), combine2_w<K, W>(pp[2 * c + 1], 1, P.inv_n)};
                const int frame0 = bz * NF + 4 * c;
                store_quad_transposed(ebuf, v, warp, lane, trow, col, P.out + (size_t)frame0 * img, img,
                                      min(4, P.n_frames - frame0), by * TR, bx * kStgCols, P.nz, P.nx, TR);
            }
        } else if (live && j < P.nx && m < P.nz) {
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                const int frame = bz * NF + f;
                if (frame < P.n_frames) P.out[(size_t)frame * img + (size_t)m * P.nx + j] = combine2_w<K, W>(pp[f / 2], f & 1, P.inv_n);
            }
        }
    }
}

// ---- host side ----
inline size_t cached_smem_bytes(const StagedCfg& c, int nq, bool compact) {
    const int bps = nq == 0 ? 4 : 16, ncopy = nq == 0 ? 1 : nq;
    const size_t blk = compact ? 4 : kCacheBlockBytes;
    return 64 + (((size_t)c.stages * c.chunk * blk + 127) & ~(size_t)127) + (size_t)c.stages * c.chunk * (size_t)c.window * bps * ncopy +
           (c.epi ? kEpiBytes : 0);
}
template <int K, int NQ>
inline cudaError_t cached_set_attr(int smem_optin) {
    cudaError_t e = cudaFuncSetAttribute(bf_cached_kernel<K, NQ, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(bf_cached_kernel<K, NQ, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
}
// instantiated: NQ = 0 for orders 1..5; NQ = 1, 2 for orders 1..5; NQ = 4 for orders 1..3
template <int K>
inline cudaError_t cached_set_attr_k(int smem_optin) {
    cudaError_t e;
    if ((e = cached_set_attr<K, 0>(smem_optin)) != cudaSuccess) return e;
    if ((e = cached_set_attr<K, 1>(smem_optin)) != cudaSuccess) return e;
    if ((e = cached_set_attr<K, 2>(smem_optin)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(bf_cached_kernel<K, 1, false, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    if constexpr (K <= 3) {
        if ((e = cudaFuncSetAttribute(bf_cached_kernel<K, 2, false, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
        return cached_set_attr<K, 4>(smem_optin);
    } else return cudaSuccess;
}
constexpr int kRootMix = 1;          // order 3, 16 frames per thread: frame pairs rooted on the FMA pipe (0 / 1 / 2 pairs measured
                                     // 1.037 / 0.981 / 1.006 ms at C2b: DESIGN.md section 6.1)
inline cudaError_t cached_configure(int smem_optin) {
    cudaError_t e;
    if ((e = cached_set_attr_k<1>(smem_optin)) != cudaSuccess) return e;
    if ((e = cached_set_attr_k<2>(smem_optin)) != cudaSuccess) return e;
    if ((e = cached_set_attr_k<3>(smem_optin)) != cudaSuccess) return e;
    if ((e = cached_set_attr_k<4>(smem_optin)) != cudaSuccess) return e;
    if ((e = cached_set_attr_k<5>(smem_optin)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(bf_cached_kernel<3, 4, false, 0, kRootMix>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(bf_cached_kernel<1, 2, false, 0, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(bf_cached_kernel<1, 4, false, 0, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(bf_cached_kernel<2, 2, false, 0, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(bf_cached_kernel<2, 4, false, 0, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    // orders 6..8 (row f2): 4-frame groups with the tile-major table only
    if ((e = cudaFuncSetAttribute(bf_cached_kernel<6, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(bf_cached_kernel<7, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(bf_cached_kernel<8, 1, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
}
template <int K, int NQ, bool COMPACT, int W = 0, int RM = 0>
inline void launch_cached_rm(const BfParams& P, const StagedCfg& c, const CacheTables& T, int sm_count, cudaStream_t st) {
    const size_t smem = cached_smem_bytes(c, NQ, COMPACT);
    const int per_sm = resident_per_sm(bf_cached_kernel<K, NQ, COMPACT, W, RM>, kStgThreads, smem);
    const long long tiles = (long long)c.tiles_x * c.tiles_z * c.groups, resident = (long long)sm_count * per_sm;
    bf_cached_kernel<K, NQ, COMPACT, W, RM><<<(unsigned)(tiles < resident ? tiles : resident), kStgThreads, smem, st>>>(
        P, c, T.taps, T.w0s, T.compact, T.q);
}
template <int K, int NQ>
inline void launch_cached_r7(const BfParams& P, const StagedCfg& c, const CacheTables& T, int sm_count, cudaStream_t st) {
    const size_t smem = cached_smem_bytes(c, NQ, false);
    const int per_sm = resident_per_sm(bf_cached_kernel<K, NQ, false, 0, 0, true>, kStgThreads, smem);
    const long long tiles = (long long)c.tiles_x * c.tiles_z * c.groups, resident = (long long)sm_count * per_sm;
    bf_cached_kernel<K, NQ, false, 0, 0, true><<<(unsigned)(tiles < resident ? tiles : resident), kStgThreads, smem, st>>>(
        P, c, T.taps, T.w0s, T.compact, T.q);
}
template <int K, int NQ, bool COMPACT, int W = 0>
inline void launch_cached_kc(const BfParams& P, const StagedCfg& c, const CacheTables& T, int sm_count, cudaStream_t st) {
    if constexpr (K <= 2 && (NQ == 2 || NQ == 4) && !COMPACT && W == 0) {
        if (c.tile_rows == 56) { launch_cached_r7<K, NQ>(P, c, T, sm_count, st); return; }
    }
    if constexpr (K == 3 && NQ == 4 && !COMPACT && W == 0) {
        launch_cached_rm<K, NQ, COMPACT, W, kRootMix>(P, c, T, sm_count, st);
        return;
    }
    launch_cached_rm<K, NQ, COMPACT, W, 0>(P, c, T, sm_count, st);
}
template <int K, int NQ>
inline void launch_cached_k(const BfParams& P, const StagedCfg& c, const CacheTables& T, int sm_count, cudaStream_t st) {
    if (T.compact) launch_cached_kc<K, NQ, true>(P, c, T, sm_count, st);
    else launch_cached_kc<K, NQ, false>(P, c, T, sm_count, st);
}
// does at least one channel per stage fit in shared memory for this group size?  (the tap block makes the slot larger
// than the plain staged kernel's, so a geometry whose plan has chunk 1 may not fit here: the caller falls back)
inline bool cached_fits(const pab_plan_info& plan, int nq, bool compact, int smem_limit) {
    const long long slot = (long long)plan.window_samples * (nq == 0 ? 4 : 16 * nq) + (compact ? 4 : kCacheBlockBytes);
    return plan.stages > 0 && (long long)(smem_limit - 64 - 128) / (plan.stages * slot) >= 1;
}

template <int K>
inline void launch_cached_nq(int nq, int weight, const BfParams& P, const StagedCfg& c, const CacheTables& T, int sm_count, cudaStream_t st) {
    if (weight != 0) {          // cached_weight_ok(order, nq, compact) held
        if (nq == 1) launch_cached_kc<K, 1, false, 1>(P, c, T, sm_count, st);
        else if constexpr (K <= 3) launch_cached_kc<K, 2, false, 1>(P, c, T, sm_count, st);
        return;
    }
    if (nq == 0) launch_cached_k<K, 0>(P, c, T, sm_count, st);
    else if (nq == 1) launch_cached_k<K, 1>(P, c, T, sm_count, st);
    else if (nq == 2) launch_cached_k<K, 2>(P, c, T, sm_count, st);
    else if constexpr (K <= 3) launch_cached_k<K, 4>(P, c, T, sm_count, st);
}
// which (order, frame group, table) combinations have a coherence-factor instantiation
inline bool cached_weight_ok(int order, int nq, bool compact) {
    return !compact && (nq == 1 || (nq == 2 && order <= 3));
}
// nq = 0, 1, 2 (orders 1..5), 4 (orders 1..3) or 1 (orders 6..8, tile-major table); weight != 0 only where cached_weight_ok
inline void launch_cached(int order, int nq, int weight, const BfParams& P, int groups, const pab_plan_info& plan, int chunk_cap,
                          int smem_limit, int sm_count, const CacheTables& T, cudaStream_t st) {
    const long long slot = (long long)plan.window_samples * (nq == 0 ? 4 : 16 * nq) + (T.compact ? 4 : kCacheBlockBytes);
    const StagedCfg c = make_cfg(slot, plan.stages, plan.window_samples, nq, chunk_cap, smem_limit, P, groups, T.tile_rows);
    switch (order) {
    case 1: launch_cached_nq<1>(nq, weight, P, c, T, sm_count, st); break;
    case 2: launch_cached_nq<2>(nq, weight, P, c, T, sm_count, st); break;
    case 3: launch_cached_nq<3>(nq, weight, P, c, T, sm_count, st); break;
    case 4: launch_cached_nq<4>(nq, weight, P, c, T, sm_count, st); break;
    case 5: launch_cached_nq<5>(nq, weight, P, c, T, sm_count, st); break;
    case 6: launch_cached_kc<6, 1, false>(P, c, T, sm_count, st); break;          // orders 6..8: nq == 1, no weighting
    case 7: launch_cached_kc<7, 1, false>(P, c, T, sm_count, st); break;
    default: launch_cached_kc<8, 1, false>(P, c, T, sm_count, st); break;
    }
}

}  // namespace pab
