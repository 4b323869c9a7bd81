// pab_pipe.cuh -- shared-memory pipeline primitives of the staged kernels: mbarrier full/empty ring, 1-D bulk
// async copies (TMA engine: cp.async.bulk, SASS UBLKCP) and explicit shared-space loads.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "pab_types.h"

namespace pab {

// per staged channel: what a consumer needs besides the samples (80 bytes; every read is a warp broadcast)
struct __align__(16) ChanEntry {
    float2 xs[8];           // per pixel column c of the tile: (xs2, c0) of delay_tap, xs = column - element in samples;
                            // in-range launches: xs^2 as a double in the same 8 bytes (delay_tap_f64)
    int base;               // shared-space address such that sample i of the first quad lives at base + i * BPS
    int w0;                 // first staged sample
    int w1m2;               // last valid i0 (staged end - 2)
    int pad;
};
static_assert(sizeof(ChanEntry) == kChanEntryBytes, "ChanEntry size is part of the shared-memory plan");
constexpr int kCE = (int)sizeof(ChanEntry);

__device__ __forceinline__ float2 lds64(uint32_t addr) {
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// The producer's wait on an empty slot: it runs stages ahead of the consumers, so it can afford to sleep between
// polls instead of spinning on try_wait (a spinning producer warp takes issue and MIO slots from the four consumer
// warps of its scheduler, and every consumer warp of the CTA is coupled to the slowest one through the ring).
__device__ __forceinline__ void mbar_wait_relaxed(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "WAIT_%=:\n"
        "nanosleep.u32 256;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@!p bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ float lds32(uint32_t addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}

// ------------------------------------------------------------------------------------------------------
// Tile epilogue of the frame-group kernels.  A consumer warp holds one column and 32 rows of the tile (lanes along
// depth), so a direct store puts every lane in a different 32-byte sector of the image: 32 sectors per warp store,
// 8192 partial-sector writes per tile and frame group of 16, which the SM's store path takes one per clock (5 % of
// the kernel at C2b, all of it with the XU pipe idle because every warp of the CTA is there together).  Instead the
// 4 frames of a quad go through a 64 x 8 x 4 transpose buffer in shared memory and leave as whole 32-byte row
// segments: 4 sectors per warp store.
// ------------------------------------------------------------------------------------------------------
// Row of the tile a consumer thread owns.  64-row tiles: warp half h = warp >> 3 holds rows 32 h + lane.  56-row tiles
// (orders 1, 2 at row pitches in (1, 8/7] samples): a 128-bit shared load is served a quarter-warp at a time, 8 lanes
// on 8 bank groups of 16 bytes; 8 consecutive rows at such a pitch span 9 samples, so the first and the last lane of a
// quarter meet in one bank group and every quarter costs a second wavefront (measured: 28.6 % of the wavefronts of an
// order-1 launch at C2b, whose kernel runs at 94 % of the shared-memory data pipe).  Seven rows never do (span < 8): the
// eighth lane of every quarter repeats its neighbour's row (same address: a broadcast, no wavefront) and stores nothing.
__device__ __forceinline__ int tile_row(int tile_rows, int warp, int lane, bool* live) {
    if (tile_rows == kStgRows) { *live = true; return (warp >> 3) * 32 + lane; }
    *live = (lane & 7) != 7;
    return (warp >> 3) * 28 + (lane >> 3) * 7 + min(lane & 7, 6);
}

__device__ __forceinline__ void consumer_barrier() {
    asm volatile("bar.sync 1, %0;" ::"n"(kStgConsumerWarps * 32) : "memory");
}
// v[f]: this thread's pixel (tile row `row`, tile column `col`) of the quad's 4 frames.  out0 = image of the quad's
// first frame; n_valid = how many of the 4 frames exist.  Every consumer thread of the CTA must call it.
__device__ __forceinline__ void store_quad_transposed(uint32_t ebuf, const float (&v)[4], int warp, int lane, int row, int col,
                                                      float* out0, size_t img, int n_valid, int m0, int j0, int nz, int nx,
                                                      int tile_rows = kStgRows) {
#pragma unroll
    for (int f = 0; f < 4; ++f)
        asm volatile("st.shared.f32 [%0], %1;" ::"r"(ebuf + (uint32_t)(((f * kStgRows + row) * kEpiRowFloats + col) * 4)), "f"(v[f]) : "memory");
    consumer_barrier();
    const int f = warp >> 2, c = lane & 7;
    if (f < n_valid && j0 + c < nx) {
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int r = (warp & 3) * 16 + i * 4 + (lane >> 3);
            float x;
            asm volatile("ld.shared.f32 %0, [%1];" : "=f"(x) : "r"(ebuf + (uint32_t)(((f * kStgRows + r) * kEpiRowFloats + c) * 4)));
            if (r < tile_rows && m0 + r < nz) out0[(size_t)f * img + (size_t)(m0 + r) * nx + (j0 + c)] = x;
        }
    }
    consumer_barrier();                 // the buffer is free for the next quad
}

// Shared-memory bytes of one launch: the plan's chunk is sized for `frames_per_thread / 4` quads per channel;
// with fewer bytes per sample the same chunk fits with room to spare.
inline size_t staged_smem_bytes(const StagedCfg& c, int nq) {
    const int bps = nq == 0 ? 4 : 16, ncopy = nq == 0 ? 1 : nq;
    const size_t tab = ((size_t)c.stages * c.chunk * sizeof(ChanEntry) + 127) & ~(size_t)127;
    return 64 + tab + (size_t)c.stages * c.chunk * c.window * bps * ncopy + (c.epi ? kEpiBytes : 0);
}

// Resident CTAs per SM of a kernel instantiation at a given dynamic shared-memory size, asked of the runtime once per
// (instantiation, device, size) and remembered: the query costs microseconds, which is the whole budget of a
// launch-bound call (config C1).
template <typename Kernel>
inline int resident_per_sm(Kernel kernel, int threads, size_t smem) {
    struct Memo { const void* fn = nullptr; int dev = -1; size_t smem = 0; int per_sm = 1; };
    static thread_local Memo memos[64];          // kernels of one signature share this function: keyed by address
    const void* fn = reinterpret_cast<const void*>(kernel);
    Memo& memo = memos[(reinterpret_cast<uintptr_t>(fn) >> 4) % 64];
    int dev = 0;
    cudaGetDevice(&dev);
    if (memo.fn == fn && memo.dev == dev && memo.smem == smem) return memo.per_sm;
    int per_sm = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        per_sm = 1;
    }
    memo.fn = fn; memo.dev = dev; memo.smem = smem; memo.per_sm = per_sm;
    return per_sm;
}

// Channels per stage for a launch whose channel slot is `slot` bytes, and whether the epilogue buffer fits beside the
// ring: the buffer is taken when at least two channels per stage still fit with it (groups of 8 and 16 frames only).
inline StagedCfg make_cfg(long long slot, int stages, int window, int nq, int chunk_cap, int smem_limit, const BfParams& P, int groups,
                          int tile_rows = kStgRows) {
    auto fit = [&](long long avail) {
        long long ch = avail / (stages * slot);
        if (ch > kStagedMaxChunk) ch = kStagedMaxChunk;
        if (chunk_cap > 0 && ch > chunk_cap) ch = chunk_cap;
        if (ch > P.N) ch = P.N;
        return ch;
    };
    const long long avail = smem_limit - 64 - 128;
    long long chunk = fit(avail);
    int epi = 0;
    if (nq > 1) {            // 4-frame groups keep the direct stores: two block barriers per quad cost them more
        const long long ce = fit(avail - kEpiBytes);
        if (ce >= 2 || ce == chunk) { chunk = ce; epi = 1; }
    }
    if (chunk > 2 && (chunk & 1) && chunk < P.N) --chunk;      // even: the element loop is unrolled by two
    if (chunk < 1) chunk = 1;
    return StagedCfg{(int)chunk, stages, window, (P.nx + kStgCols - 1) / kStgCols, (P.nz + tile_rows - 1) / tile_rows, groups, epi, tile_rows};
}

}  // namespace pab
