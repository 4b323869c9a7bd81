// pab_staged.cuh -- the staged beamforming kernel: per pixel tile, the RF window every channel contributes
// is brought into shared memory once by 1-D bulk async copies (TMA engine, cp.async.bulk, SASS UBLKCP)
// issued by a producer warp, signalled through an mbarrier full/empty ring, and gathered from there by the
// consumer warps (steps a1..a6 + a10 of DESIGN.md).
//
// Tile = 64 rows x 8 columns, 16 consumer warps (one column and 32 consecutive rows each: lanes along
// depth, so a warp's gathers from one channel are <= ~1 sample apart per lane, bank-conflict free in the
// quad layout) + 1 producer warp whose lanes each own one channel of the current chunk.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "pab_math.cuh"
#include "pab_pipe.cuh"

namespace pab {

// NQ = 0: lin layout, one frame per thread; NQ = 1, 2, 4: quad layout, 4 NQ frames per thread.
// INR: every delay index of the geometry lies inside the record (checked on the host): no masks, no clamps.
// Persistent: grid = min(#tiles, resident CTAs); CTA b takes tiles b, b + gridDim.x, ...  The full/empty ring
// runs on across tiles, so the producer warp is already copying the next tile's first chunks while the
// consumer warps finish the current tile and store its images.
template <int K, int NQ, bool INR, int W>
__global__ void __launch_bounds__(kStgThreads, 1) bf_staged_kernel(const BfParams P, const StagedCfg C) {
    constexpr int NF = NQ == 0 ? 1 : 4 * NQ;
    constexpr int BPS = NQ == 0 ? 4 : 16;              // bytes per staged sample
    constexpr int NCOPY = NQ == 0 ? 1 : NQ;            // bulk copies per channel
    extern __shared__ __align__(128) unsigned char stg_smem[];
    unsigned char* smem = stg_smem;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem);                 // full[stages], empty[stages]
    ChanEntry* tab = reinterpret_cast<ChanEntry*>(smem + 64);           // [stages][chunk]
    const int tab_bytes = (C.stages * C.chunk * (int)sizeof(ChanEntry) + 127) & ~127;
    const uint32_t data0 = smem_u32(smem + 64 + tab_bytes);
    const int quad_bytes = C.window * BPS;
    const int slot_bytes = quad_bytes * NCOPY;
    const int stage_bytes = C.chunk * slot_bytes;
    const uint32_t bar0 = smem_u32(bars);
    const uint32_t ebuf = data0 + C.stages * stage_bytes;          // epilogue transpose buffer (C.epi)

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_chunks = (P.N + C.chunk - 1) / C.chunk;
    const int n_tiles = C.tiles_x * C.tiles_z * C.groups;

    if (threadIdx.x == 0) {
        for (int s = 0; s < C.stages; ++s) {
            mbar_init(bar0 + 8 * s, C.chunk);                               // full: one arrival per producer lane
            mbar_init(bar0 + 8 * (C.stages + s), kStgConsumerWarps);        // empty: one arrival per consumer warp
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == kStgConsumerWarps) {
        // ---------------- producer warp: lane l stages channel (chunk * C.chunk + l) ----------------
        if (lane >= C.chunk) return;
        const size_t chan_stride = NQ == 0 ? (size_t)P.Sp * 4 : (size_t)P.S * 16;        // bytes
        const size_t grp_stride = (size_t)P.N * chan_stride;                              // one frame / one quad
        const int row_len = NQ == 0 ? P.Sp : P.S;
        int s = 0;
        uint32_t ph = 1;                                     // parity to wait for on empty[s]
        for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
            const int bx = tile % C.tiles_x, by = (tile / C.tiles_x) % C.tiles_z, bz = tile / (C.tiles_x * C.tiles_z);
            const int c0 = bx * kStgCols, r0 = by * C.tile_rows;
            const int rl = min(r0 + C.tile_rows - 1, P.nz - 1);
            const float4 zf = P.zrow[r0], zl = P.zrow[rl];
            float2 xj[kStgCols];
#pragma unroll
            for (int c = 0; c < kStgCols; ++c) xj[c] = P.xj[min(c0 + c, P.nx - 1)];
            const char* grp = reinterpret_cast<const char*>(P.rf) + (size_t)bz * (NQ == 0 ? 1 : NQ) * grp_stride;
            for (int ck = 0; ck < n_chunks; ++ck) {
                const uint32_t full = bar0 + 8 * s, empty = bar0 + 8 * (C.stages + s);
                mbar_wait_relaxed(empty, ph);
                const int ch = ck * C.chunk + lane;
                if (ch < P.N) {
                    const float2 xe = __ldg(P.xe + ch);
                    ChanEntry e;
                    float xlo = 0.0f, xhi = 0.0f;
#pragma unroll
                    for (int c = 0; c < kStgCols; ++c) {            // fp64: the exact table difference and its square
                        const double d = ((double)xj[c].x + (double)xj[c].y) - ((double)xe.x + (double)xe.y);
                        const float hi = (float)d;
                        const float xs2 = hi * hi;
                        if constexpr (INR) {        // in-range: the square itself, as a double in the entry's 8 bytes (delay_tap_f64)
                            const double dd = d * d;
                            e.xs[c] = make_float2(__int_as_float(__double2loint(dd)), __int_as_float(__double2hiint(dd)));
                        } else {
                            e.xs[c] = make_float2(xs2, (float)((double)xs2 - d * d));
                        }
                        if (c == 0) xlo = hi;
                        if (c == kStgCols - 1) xhi = hi;
                    }
                    const float amax = fmaxf(fabsf(xlo), fabsf(xhi));
                    const float amin = (xlo <= 0.0f && xhi >= 0.0f) ? 0.0f : fminf(fabsf(xlo), fabsf(xhi));
                    const float imin = fminf(sqrtf(fmaf(amin, amin, zf.x * zf.x)), 2.0e6f);
                    const float imax = fminf(sqrtf(fmaf(amax, amax, zl.x * zl.x)), 2.0e6f);
                    int w0 = max((int)floorf(imin) - 1, 0) & ~3;
                    int w1 = (int)floorf(imax) + 3;
                    if (NQ == 0) {
                        w1 = (w1 + 3) & ~3;
                        w0 = min(w0, row_len - 4);
                        w1 = min(max(w1, w0 + 4), row_len);
                    } else {
                        w0 = min(w0, (row_len - 2) & ~3);
                        w1 = min(max(w1, w0 + 2), row_len);
                    }
                    w1 = min(w1, w0 + C.window);
                    const int len = w1 - w0;
                    const int slot = s * stage_bytes + lane * slot_bytes;
                    e.base = (int)data0 + slot - w0 * BPS; e.w0 = w0; e.w1m2 = w1 - 2; e.pad = 0;
                    tab[s * C.chunk + lane] = e;
                    const uint32_t bytes = (uint32_t)len * BPS;
                    mbar_arrive_expect_tx(full, bytes * NCOPY);
                    const char* src = grp + (size_t)ch * chan_stride + (size_t)w0 * BPS;
#pragma unroll
                    for (int q = 0; q < NCOPY; ++q)
                        bulk_g2s(data0 + slot + q * quad_bytes, src + q * grp_stride, bytes, full);
                } else {
                    mbar_arrive(full);
                }
                if (++s == C.stages) { s = 0; ph ^= 1; }
            }
        }
        return;
    }

    // ---------------- consumer warps ----------------
    const int col = warp & 7;
    int s = 0;
    uint32_t ph = 0;                                         // parity to wait for on full[s]
    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const int bx = tile % C.tiles_x, by = (tile / C.tiles_x) % C.tiles_z, bz = tile / (C.tiles_x * C.tiles_z);
        const int j = bx * kStgCols + col;
        bool live;
        const int trow = tile_row(C.tile_rows, warp, lane, &live);
        const int m = by * C.tile_rows + trow;
        const float4 row = P.zrow[min(m, P.nz - 1)];
        const double zs64 = fma(0.5, (double)row.y, (double)row.x);          // zs = zs_hi + zs_lo (used by the in-range variant)
        // one frame per thread: scalar accumulators; frame groups: the frames in pairs, packed f32x2 arithmetic
        float p[1][kAcc<K, W>];
        float2 pp[NQ == 0 ? 1 : NF / 2][kAcc<K, W>];
#pragma unroll
        for (int k = 0; k < kAcc<K, W>; ++k) p[0][k] = 0.0f;
#pragma unroll
        for (int f = 0; f < (NQ == 0 ? 1 : NF / 2); ++f)
#pragma unroll
            for (int k = 0; k < kAcc<K, W>; ++k) pp[f][k] = make_float2(0.0f, 0.0f);

        for (int ck = 0; ck < n_chunks; ++ck) {
            mbar_wait(bar0 + 8 * s, ph);
            const int nch = min(C.chunk, P.N - ck * C.chunk);
            const uint32_t tab_s = smem_u32(tab + s * C.chunk);
            // elements in flight per thread: measured best 3 with 16 frames per thread, 2 otherwise
            constexpr int kElemUnroll = NQ >= 4 ? 3 : 2;
#pragma unroll (kElemUnroll)
            for (int l = 0; l < nch; ++l) {
                const float2 xs = lds64(tab_s + l * kCE + col * 8);
                const int base = __float_as_int(lds32(tab_s + l * kCE + 64));
                Tap t;
                if constexpr (INR) t = delay_tap_f64(__hiloint2double(__float_as_int(xs.y), __float_as_int(xs.x)), zs64);
                else t = delay_tap<INR>(xs.x, xs.y, row, P.S);
                int i0 = t.i0;
                if constexpr (!INR) {
                    const int w0 = __float_as_int(lds32(tab_s + l * kCE + 68));
                    const int w1m2 = __float_as_int(lds32(tab_s + l * kCE + 72));
                    i0 = min(max(i0, w0), w1m2);
                }
                const uint32_t a = (uint32_t)base + i0 * BPS;
                if constexpr (NQ == 0) {
                    const float s0 = lds32(a), s1 = lds32(a + 4);
                    accumulate_w<K, W>(interp<INR>(t, s0, s1), p[0]);
                } else {
#pragma unroll
                    for (int q = 0; q < NQ; ++q) {
                        const float4 s0 = lds128(a + q * quad_bytes);
                        const float4 s1 = lds128(a + q * quad_bytes + 16);
                        accumulate2_w<K, W>(interp2<INR>(t, make_float2(s0.x, s0.y), make_float2(s1.x, s1.y)), pp[2 * q + 0]);
                        // order 3, 16 frames per thread: the last frame pair takes its cube root on the FMA pipe (cbrt_fma2),
                        // which relieves the XU pipe (measured: pab_cache.cuh, kRootMix)
                        if (K == 3 && NQ == 4 && W == 0 && q == 3)
                            accumulate2_w<K, W, K == 3 && NQ == 4 && W == 0>(interp2<INR>(t, make_float2(s0.z, s0.w), make_float2(s1.z, s1.w)), pp[2 * q + 1]);
                        else
                            accumulate2_w<K, W>(interp2<INR>(t, make_float2(s0.z, s0.w), make_float2(s1.z, s1.w)), pp[2 * q + 1]);
                    }
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
                                      min(4, P.n_frames - frame0), by * C.tile_rows, bx * kStgCols, P.nz, P.nx, C.tile_rows);
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
template <int K, int NQ, bool INR, int W>
inline cudaError_t staged_set_attr(int smem_optin) {
    return cudaFuncSetAttribute(bf_staged_kernel<K, NQ, INR, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
}
template <int NQ, bool INR, int W>
inline cudaError_t staged_set_attr_orders(int smem_optin) {
    cudaError_t e;
    if ((e = staged_set_attr<1, NQ, INR, W>(smem_optin)) != cudaSuccess) return e;
    if ((e = staged_set_attr<2, NQ, INR, W>(smem_optin)) != cudaSuccess) return e;
    if ((e = staged_set_attr<3, NQ, INR, W>(smem_optin)) != cudaSuccess) return e;
    if ((e = staged_set_attr<4, NQ, INR, W>(smem_optin)) != cudaSuccess) return e;
    if constexpr (NQ <= 1 && W == 0) {
        if ((e = staged_set_attr<6, NQ, INR, W>(smem_optin)) != cudaSuccess) return e;
        if ((e = staged_set_attr<7, NQ, INR, W>(smem_optin)) != cudaSuccess) return e;
        if ((e = staged_set_attr<8, NQ, INR, W>(smem_optin)) != cudaSuccess) return e;
    }
    return staged_set_attr<5, NQ, INR, W>(smem_optin);
}
template <bool INR>
inline bool staged_configure_inr(int smem_optin) {
    // W = 1 (coherence factor) is instantiated for 1, 4 and 8 frames per thread only (run_batch caps the group)
    return staged_set_attr_orders<0, INR, 0>(smem_optin) == cudaSuccess && staged_set_attr_orders<1, INR, 0>(smem_optin) == cudaSuccess &&
           staged_set_attr_orders<2, INR, 0>(smem_optin) == cudaSuccess && staged_set_attr_orders<4, INR, 0>(smem_optin) == cudaSuccess &&
           staged_set_attr_orders<0, INR, 1>(smem_optin) == cudaSuccess && staged_set_attr_orders<1, INR, 1>(smem_optin) == cudaSuccess &&
           staged_set_attr_orders<2, INR, 1>(smem_optin) == cudaSuccess;
}

template <int K, int NQ, bool INR, int W>
inline void launch_staged_k(const BfParams& P, const StagedCfg& c, int sm_count, cudaStream_t st) {
    const size_t smem = staged_smem_bytes(c, NQ);
    const int per_sm = resident_per_sm(bf_staged_kernel<K, NQ, INR, W>, kStgThreads, smem);
    const long long tiles = (long long)c.tiles_x * c.tiles_z * c.groups;
    const long long resident = (long long)sm_count * per_sm;
    bf_staged_kernel<K, NQ, INR, W><<<(unsigned)(tiles < resident ? tiles : resident), kStgThreads, smem, st>>>(P, c);
}
template <int NQ, bool INR, int W>
inline void launch_staged_nq(int order, const BfParams& P, const StagedCfg& c, int sm_count, cudaStream_t st) {
    switch (order) {
    case 1: launch_staged_k<1, NQ, INR, W>(P, c, sm_count, st); break;
    case 2: launch_staged_k<2, NQ, INR, W>(P, c, sm_count, st); break;
    case 3: launch_staged_k<3, NQ, INR, W>(P, c, sm_count, st); break;
    case 4: launch_staged_k<4, NQ, INR, W>(P, c, sm_count, st); break;
    case 5: launch_staged_k<5, NQ, INR, W>(P, c, sm_count, st); break;
    default:
        if constexpr (NQ <= 1 && W == 0) {          // orders 6..8: at most 4 frames per thread, no weighting
            if (order == 6) launch_staged_k<6, NQ, INR, W>(P, c, sm_count, st);
            else if (order == 7) launch_staged_k<7, NQ, INR, W>(P, c, sm_count, st);
            else launch_staged_k<8, NQ, INR, W>(P, c, sm_count, st);
        }
        break;
    }
}
template <bool INR>
inline void launch_staged_inr(int order, int nq, int weight, const BfParams& P, const StagedCfg& c, int sm_count,
                              cudaStream_t st) {
    if (weight == 0) {
        if (nq == 0) launch_staged_nq<0, INR, 0>(order, P, c, sm_count, st);
        else if (nq == 1) launch_staged_nq<1, INR, 0>(order, P, c, sm_count, st);
        else if (nq == 2) launch_staged_nq<2, INR, 0>(order, P, c, sm_count, st);
        else launch_staged_nq<4, INR, 0>(order, P, c, sm_count, st);
    } else {
        if (nq == 0) launch_staged_nq<0, INR, 1>(order, P, c, sm_count, st);
        else if (nq == 1) launch_staged_nq<1, INR, 1>(order, P, c, sm_count, st);
        else launch_staged_nq<2, INR, 1>(order, P, c, sm_count, st);
    }
}
template <bool INR>
inline void launch_staged_t(int order, int nq, int weight, const BfParams& P, int groups, const pab_plan_info& plan,
                            int chunk_cap, int smem_limit, int sm_count, cudaStream_t st) {
    // the plan's chunk is sized for frames_per_thread / 4 quads per channel; fewer quads -> more channels per stage
    const long long slot = (long long)plan.window_samples * (nq == 0 ? 4 : 16 * nq) + (long long)sizeof(ChanEntry);
    // order 1 in groups of 8 / 16 frames is bound by the shared-memory data pipe: 56-row tiles where the row pitch makes
    // 64-row tiles conflict (tile_row, pab_pipe.cuh).  Order 2 (one MUFU per item) loses more to the idle lanes than it
    // gains (measured 0.831 -> 0.859 ms at C2b), so it keeps 64 rows.
    const bool r7 = order == 1 && weight == 0 && nq >= 2 && plan.zs_per_row > 1.0 && plan.zs_per_row <= 8.0 / 7.0 + 1e-9;
    const StagedCfg c = make_cfg(slot, plan.stages, plan.window_samples, nq, chunk_cap, smem_limit, P, groups, r7 ? 56 : kStgRows);
    launch_staged_inr<INR>(order, nq, weight, P, c, sm_count, st);
}

}  // namespace pab
