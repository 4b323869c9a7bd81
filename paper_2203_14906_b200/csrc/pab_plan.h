// pab_plan.h -- host-only logic: tiling / staging plan, delay tables, FIR tap design.  No CUDA calls.
#pragma once
#include <cmath>
#include <cstdint>
#include <vector>
#include "../../include/pab.h"

namespace pab {

constexpr int kSmemOptin = 232448;      // sm_100 opt-in dynamic shared memory per block
constexpr int kStagedTileZ = 64;        // rows per tile of the staged kernel (2 warps deep)
constexpr int kStagedTileX = 8;         // columns per tile
constexpr int kStagedMaxChunk = 32;
constexpr int kChanEntryBytes = 80;     // per staged channel: 8 x (xs hi, 2 lo) + window base and bounds     // channels per stage <= one producer lane per channel

inline int round_up(int v, int m) { return (v + m - 1) / m * m; }

// Upper bound of the RF window (samples) one channel contributes to a tile_z x tile_x pixel tile:
// idx is 1-Lipschitz in z and in x when both are in sample units, so the window spans at most
// span = (tile_z - 1) zs_per_row + (tile_x - 1) xs_per_col samples.  The producer stages
// [floor(idx_min) - 1 rounded down to 4, floor(idx_max) + 3 rounded up to 4): at most span + 12 samples
// (1 + 3 below, 3 + 3 above, 1 + 1 for the two floors).
inline int window_bound(int tile_z, int tile_x, double zs_per_row, double xs_per_col) {
    double span = (tile_z - 1) * zs_per_row + (tile_x - 1) * xs_per_col;
    return round_up((int)std::ceil(span) + 12, 4);
}

struct PlanTuning {
    int frames_per_thread = 0;   // 4, 8 or 16; 0 = default
    int stages = 0;              // 2..4; 0 = default
    int chunk_channels = 0;      // 1..32; 0 = as many as fit
    int host_batch_frames = 0;   // frames per piece of the host entry point's copy/compute pipeline; 0 = default
};
constexpr int kDefaultFramesPerThread = 16;

inline bool plan_geometry(int n_elem, int n_samp, double fs, double c, double pitch, const pab_grid& g,
                          int smem_limit, pab_plan_info* out, const PlanTuning& tune = PlanTuning()) {
    if (n_elem < 1 || n_samp < 2 || !(fs > 0) || !(c > 0) || !(pitch > 0)) return false;
    if (g.nx < 1 || g.nz < 1 || !(g.dx > 0) || !(g.dz > 0) || !(g.z0 >= 0)) return false;
    if (tune.frames_per_thread != 0 && tune.frames_per_thread != 4 && tune.frames_per_thread != 8 &&
        tune.frames_per_thread != 16) return false;
    if (tune.stages != 0 && (tune.stages < 2 || tune.stages > 4)) return false;
    if (tune.chunk_channels < 0 || tune.chunk_channels > kStagedMaxChunk) return false;
    if (smem_limit <= 0) smem_limit = kSmemOptin;
    pab_plan_info p{};
    p.tile_z = kStagedTileZ;
    p.tile_x = kStagedTileX;
    p.zs_per_row = (double)g.dz * fs / c;
    p.xs_per_col = (double)g.dx * fs / c;
    p.frames_per_thread = tune.frames_per_thread ? tune.frames_per_thread : kDefaultFramesPerThread;
    double w = (p.tile_z - 1) * p.zs_per_row + (p.tile_x - 1) * p.xs_per_col;
    p.window_samples = w < 1e6 ? window_bound(p.tile_z, p.tile_x, p.zs_per_row, p.xs_per_col) : 1 << 20;
    if (p.window_samples > round_up(n_samp, 4)) p.window_samples = round_up(n_samp, 4);
    // bytes of one channel slot: window x (frames_per_thread / 4) quads x 16 B, + its 80-byte table entry;
    // 64 bytes of barriers and up to 128 bytes of table padding on top
    const int nq = p.frames_per_thread / 4;
    const long long slot = (long long)p.window_samples * 16 * nq + kChanEntryBytes;
    const int overhead = 64 + 128;
    p.stages = tune.stages ? tune.stages : 3;
    auto fit = [&](int stages) {
        long long ch = (smem_limit - overhead) / (stages * slot);
        if (ch > kStagedMaxChunk) ch = kStagedMaxChunk;
        if (ch > n_elem) ch = n_elem;
        if (tune.chunk_channels && ch > tune.chunk_channels) ch = tune.chunk_channels;
        return (int)ch;
    };
    int chunk = fit(p.stages);
    if (chunk < 4 && !tune.stages) { p.stages = 2; chunk = fit(p.stages); }
    if (chunk >= 1) {
        p.chunk_channels = chunk;
        p.smem_bytes = 64 + round_up(p.stages * chunk * kChanEntryBytes, 128) + p.stages * chunk * p.window_samples * 16 * nq;
    } else {
        p.chunk_channels = 0; p.stages = 0; p.smem_bytes = 0;   // staged kernel does not fit: direct only
    }
    // every delay index of the geometry inside the record, and z > 0 (so the rsqrt argument is never 0)?
    {
        const double k = fs / c;
        const double xe_max = ((double)n_elem - 1.0) / 2.0 * pitch;
        const double xa = std::fabs((double)g.x0), xb = std::fabs((double)g.x0 + (g.nx - 1) * (double)g.dx);
        const double ax = ((xa > xb ? xa : xb) + xe_max) * k;
        const double zl = ((double)g.z0 + (g.nz - 1) * (double)g.dz) * k;
        const double idx_max = std::sqrt(ax * ax + zl * zl);
        p.in_range = (idx_max + 1.0 < (double)n_samp - 1.0) && ((double)g.z0 * k >= 1.0) ? 1 : 0;
    }
    // internal frame batch of the device path: as many frames per launch as 512 MiB of staged RF allow (<= 256), so
    // that small pixel grids still give the persistent kernel many tiles per SM (tail balance); the staged copy is
    // an intermediate that costs 2 x 4 bytes of HBM traffic per sample, far from binding (DESIGN.md Roofline).
    const double frame_bytes = (double)n_elem * n_samp * 4.0;
    int b = (int)(512.0 * 1048576.0 / frame_bytes);
    b = b / 16 * 16;
    if (b < 16) b = 16;
    if (b > 256) b = 256;
    p.batch_frames = b;
    *out = p;
    return true;
}

// Delay tables in sample units, computed in fp64 from the float parameters promoted unchanged
// (the oracle does the same promotion): hi + lo fp32 pairs.
struct DelayTables {
    std::vector<float> xj;     // [nx][2]
    std::vector<float> xe;     // [N][2]
    std::vector<float> zrow;   // [nz][4]: zs_hi, 2 zs_lo, zf - 1/2, zi - 2 * 0x4B400000 (int bits)
};

inline void split_hi_lo(double v, float* hi, float* lo) { *hi = (float)v; *lo = (float)(v - (double)*hi); }

inline DelayTables make_tables(int n_elem, double fs, double c, double pitch, const pab_grid& g) {
    DelayTables t;
    const double k = fs / c;
    t.xj.resize((size_t)g.nx * 2);
    for (int j = 0; j < g.nx; ++j) split_hi_lo(((double)g.x0 + j * (double)g.dx) * k, &t.xj[2 * j], &t.xj[2 * j + 1]);
    t.xe.resize((size_t)n_elem * 2);
    for (int i = 0; i < n_elem; ++i)
        split_hi_lo((((double)i - ((double)n_elem - 1.0) / 2.0) * pitch) * k, &t.xe[2 * i], &t.xe[2 * i + 1]);
    t.zrow.resize((size_t)g.nz * 4);
    for (int m = 0; m < g.nz; ++m) {
        const double zs = ((double)g.z0 + m * (double)g.dz) * k;
        double zi = std::floor(zs);
        if (zi > 1.0e9) zi = 1.0e9;
        // pre-biased for two magic-number roundings; the sum zii + bits(t0) + bits(t1) is taken modulo 2^32
        const uint32_t zii = (uint32_t)(int64_t)zi - 2u * 0x4B400000u;
        float zib;
        static_assert(sizeof(float) == sizeof(int32_t), "");
        __builtin_memcpy(&zib, &zii, 4);
        t.zrow[4 * m + 0] = (float)zs;
        t.zrow[4 * m + 1] = (float)(2.0 * (zs - (double)(float)zs));
        t.zrow[4 * m + 2] = (float)((zs - zi) - 0.5);
        t.zrow[4 * m + 3] = zib;
    }
    return t;
}

// Hamming-windowed ideal band-pass (A8): h[t] = w[t] (2 f_hi sinc(2 f_hi m) - 2 f_lo sinc(2 f_lo m)),
// m = t - (T-1)/2, w[t] = 0.54 - 0.46 cos(2 pi t / (T-1)); frequencies in cycles per row.
inline void design_bandpass(int T, double f_lo, double f_hi, float* h) {
    const double pi = 3.14159265358979323846;
    for (int t = 0; t < T; ++t) {
        const double m = t - 0.5 * (T - 1);
        const double w = 0.54 - 0.46 * std::cos(2.0 * pi * t / (T - 1));
        auto lp = [&](double f) { return m == 0.0 ? 2.0 * f : std::sin(2.0 * pi * f * m) / (pi * m); };
        h[t] = (float)(w * (lp(f_hi) - lp(f_lo)));
    }
}

// Type-III Hilbert FIR (A9): g[t] = 2 / (pi t) for odd t, 0 for even t, |t| <= L, Hamming window
// 0.54 + 0.46 cos(pi t / L); stored at g[t + L].
inline void design_hilbert(int L, float* g) {
    const double pi = 3.14159265358979323846;
    for (int t = -L; t <= L; ++t) {
        const double w = 0.54 + 0.46 * std::cos(pi * t / L);
        g[t + L] = (t & 1) ? (float)(w * 2.0 / (pi * t)) : 0.0f;
    }
}

}  // namespace pab
