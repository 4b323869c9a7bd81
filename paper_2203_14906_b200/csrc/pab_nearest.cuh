// pab_nearest.cuh -- SURVEY.md section 8(f) row f4: the literal eq. (1) of the paper, integer
// delays: s_i = rf_i[n_i], n_i = floor(idx_i + 1/2) (reading A21), zero outside the record (A6).
//
// With integer delays the signed k-th root commutes with the gather, so it is taken ONCE PER RF SAMPLE while the
// frames are staged (N S roots per frame instead of nz nx N), and the hot loop has no transcendental at all:
// it turns from XU-bound into shared-memory / FP32-bound.  The integer decision n_i must be the oracle's, so it
// is not taken in fp32: the paper's own data structure, a delay table in global memory ("all the
// delays ... were calculated and stored in the GPU (global) memory"), is built once per geometry by an fp64
// kernel that evaluates fs sqrt((x - xe)^2 + z^2) / c with individually rounded IEEE operations, and holds
// n_i as uint16 (0xFFFF = outside the record), laid out tile-major, [tile row][tile column][element][8 columns][64
// rows], so the 1 KB block one element contributes to one 64 x 8 pixel tile is contiguous: the producer warp brings
// it into shared memory with one bulk copy next to that element's RF window.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "pab_math.cuh"
#include "pab_pipe.cuh"

namespace pab {

// table[nearest_index(...)] = floor(idx + 1/2) or 0xFFFF.
// grid: (ceil(nz_pad/256), nx_pad, N) with nz_pad, nx_pad the grid rounded up to whole tiles.
__host__ __device__ __forceinline__ size_t nearest_index(int i, int j, int m, int N, int tiles_x) {
    return ((((size_t)(m / kStgRows) * tiles_x + (size_t)(j / kStgCols)) * N + i) * kStgCols + (j % kStgCols)) * kStgRows + (m % kStgRows);
}
__global__ void __launch_bounds__(256) nearest_table_kernel(const NearestGeom G, unsigned short* __restrict__ table) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x, j = blockIdx.y, i = blockIdx.z;
    const int tiles_x = (G.nx + kStgCols - 1) / kStgCols, tiles_z = (G.nz + kStgRows - 1) / kStgRows;
    if (m >= tiles_z * kStgRows) return;
    // every operation individually rounded (no fused multiply-add), in the order the definition is written
    // padding pixels of edge tiles repeat the last real column / row, so their entries stay inside the tile's window
    const int jc = min(j, G.nx - 1), mc = min(m, G.nz - 1);
    const double x = __dadd_rn(G.x0, __dmul_rn((double)jc, G.dx));
    const double z = __dadd_rn(G.z0, __dmul_rn((double)mc, G.dz));
    const double xe = __dmul_rn(__dsub_rn((double)i, __ddiv_rn(__dsub_rn((double)G.N, 1.0), 2.0)), G.pitch);
    const double ddx = __dsub_rn(x, xe);
    const double d = __dsqrt_rn(__dadd_rn(__dmul_rn(ddx, ddx), __dmul_rn(z, z)));
    const double idx = __ddiv_rn(__dmul_rn(G.fs, d), G.c);
    const double n = floor(__dadd_rn(idx, 0.5));
    const bool ok = n >= 0.0 && n <= (double)(G.S - 1);
    table[nearest_index(i, j, m, G.N, tiles_x)] = ok ? (unsigned short)n : kNearestInvalid;
}

__device__ __forceinline__ int lds_u16(uint32_t addr) {
    unsigned short v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(addr));
    return (int)v;
}

// signed k-th root of one RF sample, taken once while staging (accurate library roots: cost is per sample)
template <int K>
__device__ __forceinline__ float sroot_sample(float s) {
    if constexpr (K == 1) return s;
    else {
        const float a = fabsf(s);
        float r;
        if constexpr (K == 2) r = sqrtf(a);
        else if constexpr (K == 3) r = cbrtf(a);
        else if constexpr (K == 4) r = sqrtf(sqrtf(a));
        else r = powf(a, 0.2f);
        return copysignf(r, s);
    }
}

// rf[F][N][S] -> quad[ceil(F/4)][N][S][4] of u = sroot_K(scale * stored); frames beyond F are zeros.
template <typename T, int K>
__global__ void __launch_bounds__(256) ingest_root_quad_kernel(const T* __restrict__ rf, float4* __restrict__ quad,
                                                                int F, int N, int S, float scale) {
    const int n = blockIdx.y, q = blockIdx.z;
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= S) return;
    float v[4];
#pragma unroll
    for (int fr = 0; fr < 4; ++fr) {
        const int f = q * 4 + fr;
        v[fr] = f < F ? sroot_sample<K>(scale * (float)rf[((size_t)f * N + n) * (size_t)S + s]) : 0.0f;
    }
    quad[((size_t)q * N + n) * (size_t)S + s] = make_float4(v[0], v[1], v[2], v[3]);
}

// power sums from an already rooted sample u: p_m += u^m, m = 1..K  (p_K = sum u^K = sum s or sum |s|)
template <int K>
__device__ __forceinline__ void accumulate_rooted(float u, float (&p)[K]) {
    p[0] += u;
    if constexpr (K >= 2) {
        const float u2 = u * u;
        p[1] += u2;
        if constexpr (K >= 3) p[2] = fmaf(u2, u, p[2]);
        if constexpr (K >= 4) p[3] = fmaf(u2, u2, p[3]);
        if constexpr (K >= 5) p[4] = fmaf(u2 * u2, u, p[4]);
    }
}

// the same on two frames (packed f32x2, pab_math.cuh)
template <int K>
__device__ __forceinline__ void accumulate_rooted2(float2 u, float2 (&p)[K]) {
    p[0] = add2(p[0], u);
    if constexpr (K >= 2) {
        const float2 u2 = mul2(u, u);
        p[1] = add2(p[1], u2);
        if constexpr (K >= 3) p[2] = fma2(u2, u, p[2]);
        if constexpr (K >= 4) p[3] = fma2(u2, u2, p[3]);
        if constexpr (K >= 5) p[4] = fma2(mul2(u2, u2), u, p[4]);
    }
}
template <int K>
__device__ __forceinline__ float combine_half(const float2 (&p)[K], int h) {
    float q[K];
#pragma unroll
    for (int k = 0; k < K; ++k) q[k] = h == 0 ? p[k].x : p[k].y;
    return combine<K>(q);
}

// ------------------------------------------------------------------------------------------------------
// Staged kernel: same tile, producer warp, bulk-copy ring and persistent tile loop as bf_staged_kernel; the
// consumer's per-(pixel, element) work is one 16-bit table load, one address, and NQ 128-bit shared loads.
// ------------------------------------------------------------------------------------------------------
template <int K, int NQ, bool INR>
__global__ void __launch_bounds__(kStgThreads, 1) bf_nearest_staged_kernel(const BfParams P, const StagedCfg C,
                                                                            const unsigned short* __restrict__ table) {
    constexpr int NF = 4 * NQ;
    constexpr int BPS = 16;
    extern __shared__ __align__(128) unsigned char stg_smem[];
    unsigned char* smem = stg_smem;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);
    ChanEntry* tab = reinterpret_cast<ChanEntry*>(smem + 64);
    const int tab_bytes = (C.stages * C.chunk * (int)sizeof(ChanEntry) + 127) & ~127;
    const uint32_t ntab0 = smem_u32(smem + 64 + tab_bytes);             // [stages][chunk][8 cols][64 rows] uint16
    const uint32_t data0 = ntab0 + C.stages * C.chunk * kNearBlockBytes;
    const int quad_bytes = C.window * BPS;
    const int slot_bytes = quad_bytes * NQ;
    const int stage_bytes = C.chunk * slot_bytes;
    const uint32_t bar0 = smem_u32(bars);
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
        const size_t chan_stride = (size_t)P.S * 16;
        const size_t grp_stride = (size_t)P.N * chan_stride;
        int s = 0;
        uint32_t ph = 1;
        for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            const int bx = tile % C.tiles_x, by = (tile / C.tiles_x) % C.tiles_z, bz = tile / (C.tiles_x * C.tiles_z);
            const int c0 = bx * kStgCols, r0 = by * kStgRows;
            const int rl = min(r0 + kStgRows - 1, P.nz - 1);
            const float4 zf = P.zrow[r0], zl = P.zrow[rl];
            const float2 xa = P.xj[c0], xb = P.xj[min(c0 + kStgCols - 1, P.nx - 1)];
            const char* grp = reinterpret_cast<const char*>(P.rf) + (size_t)bz * NQ * grp_stride;
            const char* tblk = reinterpret_cast<const char*>(table) + ((size_t)by * C.tiles_x + bx) * (size_t)P.N * kNearBlockBytes;
            for (int ck = 0; ck < n_chunks; ++ck) {
                const uint32_t full = bar0 + 8 * s, empty = bar0 + 8 * (C.stages + s);
                mbar_wait_relaxed(empty, ph);
                const int ch = ck * C.chunk + lane;
                if (ch < P.N) {
                    const float2 xe = __ldg(P.xe + ch);
                    const float xlo = (xa.x - xe.x) + (xa.y - xe.y), xhi = (xb.x - xe.x) + (xb.y - xe.y);
                    const float amax = fmaxf(fabsf(xlo), fabsf(xhi));
                    const float amin = (xlo <= 0.0f && xhi >= 0.0f) ? 0.0f : fminf(fabsf(xlo), fabsf(xhi));
                    const float imin = fminf(sqrtf(fmaf(amin, amin, zf.x * zf.x)), 2.0e6f);
                    const float imax = fminf(sqrtf(fmaf(amax, amax, zl.x * zl.x)), 2.0e6f);
                    int w0 = max((int)floorf(imin) - 1, 0) & ~3;
                    int w1 = (int)floorf(imax) + 3;
                    w0 = min(w0, (P.S - 2) & ~3);
                    w1 = min(max(w1, w0 + 2), P.S);
                    w1 = min(w1, w0 + C.window);
                    const int len = w1 - w0;
                    const int slot = s * stage_bytes + lane * slot_bytes;
                    ChanEntry e;
#pragma unroll
                    for (int c = 0; c < kStgCols; ++c) e.xs[c] = make_float2(0.0f, 0.0f);
                    e.base = (int)data0 + slot - w0 * BPS; e.w0 = w0; e.w1m2 = w1 - 2; e.pad = 0;
                    tab[s * C.chunk + lane] = e;
                    const uint32_t bytes = (uint32_t)len * BPS;
                    mbar_arrive_expect_tx(full, bytes * NQ + kNearBlockBytes);
                    bulk_g2s(ntab0 + (s * C.chunk + lane) * kNearBlockBytes, tblk + (size_t)ch * kNearBlockBytes, kNearBlockBytes, full);
                    const char* src = grp + (size_t)ch * chan_stride + (size_t)w0 * BPS;
#pragma unroll
                    for (int q = 0; q < NQ; ++q)
                        bulk_g2s(data0 + slot + q * quad_bytes, src + q * grp_stride, bytes, full);
                } else {
                    mbar_arrive(full);
                }
                if (++s == C.stages) { s = 0; ph ^= 1; }
            }
        }
        return;
    }

    const int col = warp & 7;
    const uint32_t my = (uint32_t)((col * kStgRows + (warp >> 3) * 32 + lane) * 2);   // this pixel inside a table block
    int s = 0;
    uint32_t ph = 0;
    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const int bx = tile % C.tiles_x, by = (tile / C.tiles_x) % C.tiles_z, bz = tile / (C.tiles_x * C.tiles_z);
        const int j = bx * kStgCols + col;
        const int m = by * kStgRows + (warp >> 3) * 32 + lane;
        float2 p[NF / 2][K];
#pragma unroll
        for (int f = 0; f < NF / 2; ++f)
#pragma unroll
            for (int k = 0; k < K; ++k) p[f][k] = make_float2(0.0f, 0.0f);

        for (int ck = 0; ck < n_chunks; ++ck) {
            const int nch = min(C.chunk, P.N - ck * C.chunk);
            mbar_wait(bar0 + 8 * s, ph);
            const uint32_t tab_s = smem_u32(tab + s * C.chunk);
            const uint32_t ntab_s = ntab0 + s * C.chunk * kNearBlockBytes + my;
#pragma unroll 4
            for (int l = 0; l < nch; ++l) {
                int n = lds_u16(ntab_s + l * kNearBlockBytes);
                const int base = __float_as_int(lds32(tab_s + l * kCE + 64));
                bool ok = true;
                if constexpr (!INR) {
                    ok = n != (int)kNearestInvalid;
                    const int w0 = __float_as_int(lds32(tab_s + l * kCE + 68));
                    const int w1m1 = __float_as_int(lds32(tab_s + l * kCE + 72)) + 1;
                    n = min(max(n, w0), w1m1);
                }
                const uint32_t a = (uint32_t)base + n * BPS;
#pragma unroll
                for (int q = 0; q < NQ; ++q) {
                    float4 u = lds128(a + q * quad_bytes);
                    if constexpr (!INR) { if (!ok) u = make_float4(0.0f, 0.0f, 0.0f, 0.0f); }
                    accumulate_rooted2<K>(make_float2(u.x, u.y), p[2 * q + 0]);
                    accumulate_rooted2<K>(make_float2(u.z, u.w), p[2 * q + 1]);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar0 + 8 * (C.stages + s));
            if (++s == C.stages) { s = 0; ph ^= 1; }
        }

        const size_t img = (size_t)P.nz * P.nx;
        if (C.epi) {
#pragma unroll
            for (int c = 0; c < NQ; ++c) {
                const float v[4] = {combine_half<K>(p[2 * c], 0), combine_half<K>(p[2 * c], 1), combine_half<K>(p[2 * c + 1], 0),
                                    combine_half<K>(p[2 * c + 1], 1)};
                const int frame0 = bz * NF + 4 * c;
                store_quad_transposed(ebuf, v, warp, lane, (warp >> 3) * 32 + lane, col, P.out + (size_t)frame0 * img, img,
                                      min(4, P.n_frames - frame0), by * kStgRows, bx * kStgCols, P.nz, P.nx);
            }
        } else if (j < P.nx && m < P.nz) {
#pragma unroll
            for (int f = 0; f < NF; ++f) {
                const int frame = bz * NF + f;
                if (frame < P.n_frames) P.out[(size_t)frame * img + (size_t)m * P.nx + j] = combine_half<K>(p[f / 2], f & 1);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------------
// Direct kernel (no shared memory, any geometry): gathers the rooted quads through L1/L2.
// grid: (ceil(nx/8), ceil(nz/32), groups), 256 threads, lanes along depth.
// ------------------------------------------------------------------------------------------------------
template <int K, int NQ>
__global__ void __launch_bounds__(256) bf_nearest_direct_kernel(const BfParams P, const unsigned short* __restrict__ table) {
    constexpr int NF = 4 * NQ;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int j = blockIdx.x * kDirectCols + warp;
    const int m = blockIdx.y * kDirectRows + lane;
    const int tiles_x = (P.nx + kStgCols - 1) / kStgCols;
    const size_t tstride = (size_t)kStgCols * kStgRows;        // table entries between consecutive elements of a tile
    const unsigned short* tp = table + nearest_index(0, min(j, P.nx - 1), min(m, P.nz - 1), P.N, tiles_x);
    float p[NF][K];
#pragma unroll
    for (int f = 0; f < NF; ++f)
#pragma unroll
        for (int k = 0; k < K; ++k) p[f][k] = 0.0f;
    const size_t quad_stride = (size_t)P.N * (size_t)P.S;
    const float4* chan = reinterpret_cast<const float4*>(P.rf) + (size_t)blockIdx.z * NQ * quad_stride;
#pragma unroll 4
    for (int i = 0; i < P.N; ++i, chan += P.S, tp += tstride) {
        const int n = __ldg(tp);
        const bool ok = n != (int)kNearestInvalid;
        const int nn = ok ? n : 0;
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            float4 u = __ldg(chan + q * quad_stride + nn);
            if (!ok) u = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            accumulate_rooted<K>(u.x, p[4 * q + 0]);
            accumulate_rooted<K>(u.y, p[4 * q + 1]);
            accumulate_rooted<K>(u.z, p[4 * q + 2]);
            accumulate_rooted<K>(u.w, p[4 * q + 3]);
        }
    }
    if (j < P.nx && m < P.nz) {
        const size_t img = (size_t)P.nz * P.nx;
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            const int frame = blockIdx.z * NF + f;
            if (frame < P.n_frames) P.out[(size_t)frame * img + (size_t)m * P.nx + j] = combine<K>(p[f]);
        }
    }
}

// ---- host side ----
template <int K, int NQ, bool INR>
inline void launch_nearest_staged_k(const BfParams& P, const StagedCfg& c, const unsigned short* table, int sm_count,
                                    int smem_optin, cudaStream_t st) {
    const size_t smem = staged_smem_bytes(c, NQ) + (size_t)c.stages * c.chunk * kNearBlockBytes;      // includes the epilogue buffer
    (void)smem_optin;
    const long long tiles = (long long)c.tiles_x * c.tiles_z * c.groups;
    bf_nearest_staged_kernel<K, NQ, INR><<<(unsigned)(tiles < sm_count ? tiles : sm_count), kStgThreads, smem, st>>>(P, c, table);
}
// opt in to the large dynamic shared memory for every instantiation on the current device (pab_set_interp)
template <int K, bool INR>
inline cudaError_t nearest_set_attr_k(int smem_optin) {
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(bf_nearest_staged_kernel<K, 1, INR>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(bf_nearest_staged_kernel<K, 2, INR>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    if constexpr (K <= 3)
        if ((e = cudaFuncSetAttribute(bf_nearest_staged_kernel<K, 4, INR>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    return cudaSuccess;
}
template <bool INR>
inline cudaError_t nearest_set_attr_inr(int smem_optin) {
    cudaError_t e;
    if ((e = nearest_set_attr_k<1, INR>(smem_optin)) != cudaSuccess) return e;
    if ((e = nearest_set_attr_k<2, INR>(smem_optin)) != cudaSuccess) return e;
    if ((e = nearest_set_attr_k<3, INR>(smem_optin)) != cudaSuccess) return e;
    if ((e = nearest_set_attr_k<4, INR>(smem_optin)) != cudaSuccess) return e;
    return nearest_set_attr_k<5, INR>(smem_optin);
}
inline cudaError_t nearest_configure(int smem_optin) {
    cudaError_t e = nearest_set_attr_inr<true>(smem_optin);
    return e != cudaSuccess ? e : nearest_set_attr_inr<false>(smem_optin);
}

template <int K, bool INR>
inline void launch_nearest_staged_nq(int nq, const BfParams& P, const StagedCfg& c, const unsigned short* table,
                                     int sm_count, int smem_optin, cudaStream_t st) {
    if (nq == 1) launch_nearest_staged_k<K, 1, INR>(P, c, table, sm_count, smem_optin, st);
    else if (nq == 2) launch_nearest_staged_k<K, 2, INR>(P, c, table, sm_count, smem_optin, st);
    else if constexpr (K <= 3) launch_nearest_staged_k<K, 4, INR>(P, c, table, sm_count, smem_optin, st);
}
template <bool INR>
inline void launch_nearest_staged_inr(int order, int nq, const BfParams& P, const StagedCfg& c, const unsigned short* table,
                                      int sm_count, int smem_optin, cudaStream_t st) {
    switch (order) {
    case 1: launch_nearest_staged_nq<1, INR>(nq, P, c, table, sm_count, smem_optin, st); break;
    case 2: launch_nearest_staged_nq<2, INR>(nq, P, c, table, sm_count, smem_optin, st); break;
    case 3: launch_nearest_staged_nq<3, INR>(nq, P, c, table, sm_count, smem_optin, st); break;
    case 4: launch_nearest_staged_nq<4, INR>(nq, P, c, table, sm_count, smem_optin, st); break;
    default: launch_nearest_staged_nq<5, INR>(nq, P, c, table, sm_count, smem_optin, st); break;
    }
}
inline bool nearest_staged_fits(const pab_plan_info& plan, int nq, int stages, int smem_limit) {
    if (stages <= 0) stages = 2;
    const long long slot = (long long)plan.window_samples * 16 * nq + (long long)sizeof(ChanEntry) + kNearBlockBytes;
    return (long long)(smem_limit - 64 - 128) / (stages * slot) >= 1;
}

// nq = 1, 2 or 4 quads per thread (4 only for orders <= 3)
inline void launch_nearest_staged(int order, int nq, bool in_range, const BfParams& P, int groups, const pab_plan_info& plan,
                                  int stages, int chunk_cap, int smem_limit, int sm_count, const unsigned short* table,
                                  cudaStream_t st) {
    // this kernel is bound by the latency of the staging pipeline, not by arithmetic: two deep stages of many
    // channels measured 4 % faster than three shallower ones (stages = 0: that default)
    if (stages <= 0) stages = 2;
    const long long slot = (long long)plan.window_samples * 16 * nq + (long long)sizeof(ChanEntry) + kNearBlockBytes;
    const StagedCfg c = make_cfg(slot, stages, plan.window_samples, nq, chunk_cap, smem_limit, P, groups);
    if (in_range) launch_nearest_staged_inr<true>(order, nq, P, c, table, sm_count, smem_limit, st);
    else launch_nearest_staged_inr<false>(order, nq, P, c, table, sm_count, smem_limit, st);
}

template <int K>
inline void launch_nearest_direct_k(int nq, const BfParams& P, int groups, const unsigned short* table, cudaStream_t st) {
    dim3 grid((P.nx + kDirectCols - 1) / kDirectCols, (P.nz + kDirectRows - 1) / kDirectRows, groups);
    if (nq == 1) bf_nearest_direct_kernel<K, 1><<<grid, 256, 0, st>>>(P, table);
    else if (nq == 2) bf_nearest_direct_kernel<K, 2><<<grid, 256, 0, st>>>(P, table);
    else if constexpr (K <= 3) bf_nearest_direct_kernel<K, 4><<<grid, 256, 0, st>>>(P, table);
}
inline void launch_nearest_direct(int order, int nq, const BfParams& P, int groups, const unsigned short* table, cudaStream_t st) {
    switch (order) {
    case 1: launch_nearest_direct_k<1>(nq, P, groups, table, st); break;
    case 2: launch_nearest_direct_k<2>(nq, P, groups, table, st); break;
    case 3: launch_nearest_direct_k<3>(nq, P, groups, table, st); break;
    case 4: launch_nearest_direct_k<4>(nq, P, groups, table, st); break;
    default: launch_nearest_direct_k<5>(nq, P, groups, table, st); break;
    }
}

template <typename T>
inline void launch_ingest_root_quad(int order, const void* rf, float* stage, int F, int N, int S, float scale, cudaStream_t st) {
    dim3 grid((S + 255) / 256, N, (F + 3) / 4);
    switch (order) {
    case 1: ingest_root_quad_kernel<T, 1><<<grid, 256, 0, st>>>((const T*)rf, (float4*)stage, F, N, S, scale); break;
    case 2: ingest_root_quad_kernel<T, 2><<<grid, 256, 0, st>>>((const T*)rf, (float4*)stage, F, N, S, scale); break;
    case 3: ingest_root_quad_kernel<T, 3><<<grid, 256, 0, st>>>((const T*)rf, (float4*)stage, F, N, S, scale); break;
    case 4: ingest_root_quad_kernel<T, 4><<<grid, 256, 0, st>>>((const T*)rf, (float4*)stage, F, N, S, scale); break;
    default: ingest_root_quad_kernel<T, 5><<<grid, 256, 0, st>>>((const T*)rf, (float4*)stage, F, N, S, scale); break;
    }
}

}  // namespace pab
