// pab_types.h -- parameter blocks and constants shared by the translation units of libpab.so.  No kernels here:
// every kernel header is included by exactly one .cu file (csrc/pab_tu_*.cu), pab_api.cu sees only this header
// and the launch entry points of pab_launch.h.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "../../include/pab.h"
#include "pab_plan.h"

namespace pab {

// ------------------------------------------------------------------------------------------------------
// Parameters of one beamforming launch.
//
// Staged-RF layouts (written by the ingest kernels, device memory owned by the context):
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

// direct kernels: 8 warps = 8 columns, lanes along 32 rows
constexpr int kDirectCols = 8;
constexpr int kDirectRows = 32;

// staged kernels: tile = 64 rows x 8 columns, 16 consumer warps + 1 producer warp
constexpr int kStgRows = 64, kStgCols = 8, kStgConsumerWarps = 16;
constexpr int kStgThreads = (kStgConsumerWarps + 1) * 32;
constexpr int kStgMaxStages = 4;
// epilogue buffer of the frame-group kernels: one quad of frames of a tile, rows padded to 9 floats (conflict-free)
constexpr int kEpiRowFloats = kStgCols + 1;
constexpr int kEpiBytes = 4 * kStgRows * kEpiRowFloats * 4;

struct StagedCfg {
    int chunk;          // channels per stage (<= 32)
    int stages;         // ring depth
    int window;         // samples per channel slot per quad (multiple of 4)
    int tiles_x, tiles_z, groups;   // tile grid: columns / 8, rows / 64, frame groups; tile t = (t % tiles_x, ...)
    int epi;            // 1: the tile's images leave through the shared-memory transpose buffer (coalesced stores)
    int tile_rows;      // 64, or 56: seven rows per quarter-warp, the eighth lane idle (see tile_row in pab_pipe.cuh)
};

// cached interpolation taps (pab_cache.cuh)
constexpr int kCacheBlockBytes = kStgRows * kStgCols * 4;
constexpr int kCacheFracBits = 20;
constexpr int kCacheMaxWindow = 4000;        // the integer part must fit 12 bits

struct CacheGeom {
    double fs, c, pitch, x0, dx, z0, dz;
    int N, S, nx, nz, tiles_x;
    int tile_rows;             // rows of a tile that are in use: 64, or 56 (the block keeps 64 row slots either way)
};
struct CacheTables {
    const uint32_t* taps;      // tile-major 12+20-bit taps, or nullptr when the compact table is in use
    const int* w0s;            // window start of every (tile, element)
    const uint2* compact;      // (d, row) table of translation-invariant geometries, or nullptr
    int q;                     // pitch / dx
    int tile_rows;             // 64, or 56 for the table set of order 1 (seven rows per quarter-warp)
};

// single-frame diagonal kernel (pab_diag.cuh)
constexpr int kDiagMaxWarps = 16;
constexpr int kDiagMaxParts = 16;

struct DiagCfg {
    int q;                  // pitch / dx
    int rows;               // rows per tile = rows along a warp's lanes: 16 or 32; a warp holds 32 / rows column phases
    int tile_rows;          // rows of a tile in use: rows, or 28 (rows = 32: seven rows per quarter-warp, the eighth lane repeats its
                            // neighbour's row; tile_row in pab_pipe.cuh has the reason)
    int cp;                 // column phases per tile: lcm(q, 32 / rows); phase ph = residue ph % q of column block ph / q
    int wpp;                // warps per diagonal part: cp / (32 / rows)
    int parts;              // EP: diagonal parts; warps per CTA = wpp * parts
    int cols;               // P cp: columns per tile
    int tiles_x, tiles_z;
    int quads;              // staged quads per tile: N / 4 + 2 (one zero quad on either side)
    int nd;                 // columns of the tap table
    int part_lo[kDiagMaxParts + 1];     // diagonal groups [part_lo[p], part_lo[p + 1]) of part p, as eg + P / 4 >= 0
};

struct DiagTables {
    const uint2* taps;      // [nd][nz]: (floor(idx), fraction bits) of d = j - q i + q (N - 1 + P); unused by the table-free variant
    const int* qw0;         // [tiles][quads]     first staged sample of the quad's window
    const int* qoff;        // [tiles][quads + 1] byte offset of the quad's window in the staging area (16-byte units x 16)
    // table-free variant (taps computed in the kernel, delay_tap_f64): lateral offset in samples of table column d is
    // xs_a + d xs_b, depth in samples of row m is zs_a + m zs_b
    double xs_a, xs_b, zs_a, zs_b;
    double xs2_max;         // square of the largest lateral offset (samples) of a real (pixel, element) pair
};

// one set of device tables of the diagonal kernel (P = 16 pixels per thread for orders 1..3, P = 8 for orders 4, 5)
struct DiagSet {
    DiagCfg cfg;
    uint2* taps = nullptr;
    int* qw0 = nullptr;
    int* qoff = nullptr;
    int npg = 0;            // pixel groups of 4 per thread
    int smem_bytes = 0;     // dynamic shared memory per CTA; 0: not built / does not fit
    double xs_a = 0.0, xs_b = 0.0, zs_a = 0.0, zs_b = 0.0, xs2_max = 0.0;       // see DiagTables (set for both variants)
};

// nearest-sample delays (pab_nearest.cuh)
constexpr unsigned short kNearestInvalid = 0xFFFFu;
constexpr int kNearBlockBytes = kStgRows * kStgCols * 2;      // one element's delay-table block for one tile
struct NearestGeom {
    double fs, c, pitch, x0, dx, z0, dz;
    int N, S, nx, nz;
};

// post chain (pab_post.cuh)
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
// Taps as the fast post kernels read them (correlation form): out[m] = sum_j hr[j] in[m + shift - 63 + j], hr[j] = h[63 - j].
struct alignas(16) PostTaps64 {
    float hbr[64];   // band-pass taps, zero-padded to 64, reversed
    float hbs[64];   // the same one place on: hbs[j] = hbr[j - 1] (pairs for odd output rows)
    float hhr[64];   // Hilbert taps g[t'] = g(t' - L), zero-padded to 64, reversed (dense case)
    float hhs[64];   // hhs[j] = hhr[j - 1]
    float hhd[64];   // type-III case: the 32 reversed taps of the non-zero parity, each stored twice
};

// image metrics (pab_metrics.cuh)
struct RoiPair { int t[4]; int b[4]; };      // target, background: rows [r0, r1), columns [c0, c1)
struct MetricAcc {
    double sum_in, sum_out, var_out;
    unsigned int max_bits;          // float bits of the largest amplitude of both regions (amplitudes >= 0)
    unsigned int pad;
};

}  // namespace pab
