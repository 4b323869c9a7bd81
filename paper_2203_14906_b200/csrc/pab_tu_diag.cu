// pab_tu_diag.cu -- translation unit: the single-frame "diagonal" beamforming kernel (pab_diag.cuh) and its tables.
#include <algorithm>
#include <cmath>
#include <vector>
#include "pab_diag.cuh"
#include "pab_launch.h"

namespace pab {

namespace {

// Split the G diagonal groups into `parts` consecutive ranges of nearly equal work.  The work of group g (eg = g - NPG)
// is its number of live pixel groups (blocks with at least one pair on the array).  Returns the largest part's work.
int split_parts(int G, int npg, int nq_real, int parts, int* lo) {
    std::vector<int> w(G);
    int total = 0;
    for (int g = 0; g < G; ++g) {
        const int eg = g - npg;
        int n = 0;
        for (int cg = 0; cg < npg; ++cg) n += (eg + cg + 1 >= 0 && eg + cg < nq_real) ? 1 : 0;
        w[g] = n; total += n;
    }
    int best_cap = total;              // smallest cap such that a greedy left-to-right packing needs <= parts ranges
    for (int cap = (total + parts - 1) / parts; cap <= total; ++cap) {
        int used = 1, acc = 0;
        bool ok = true;
        for (int g = 0; g < G; ++g) {
            if (w[g] > cap) { ok = false; break; }
            if (acc + w[g] > cap) { ++used; acc = 0; }
            acc += w[g];
        }
        if (ok && used <= parts) { best_cap = cap; break; }
    }
    int p = 0, acc = 0;
    lo[0] = 0;
    for (int g = 0; g < G; ++g) {
        if (acc + w[g] > best_cap) { lo[++p] = g; acc = 0; }
        acc += w[g];
    }
    while (p < parts) lo[++p] = G;
    return best_cap;
}

template <int K, int NPG, typename T, int W>
void launch_diag_t(const DiagSet& D, const void* rf, float* out, int F, int N, int S, int nx, int nz, float scale, cudaStream_t st) {
    dim3 grid(D.cfg.tiles_x * D.cfg.tiles_z, F);
    const DiagTables tabs{D.taps, D.qw0, D.qoff, D.xs_a, D.xs_b, D.zs_a, D.zs_b, D.xs2_max};
    if (D.taps)
        bf_diag_kernel<K, NPG, T, false, true, W><<<grid, D.cfg.wpp * D.cfg.parts * 32, D.smem_bytes, st>>>((const T*)rf, out, D.cfg, tabs, N, S, nx, nz, scale);
    else
        bf_diag_kernel<K, NPG, T, false, false, W><<<grid, D.cfg.wpp * D.cfg.parts * 32, D.smem_bytes, st>>>((const T*)rf, out, D.cfg, tabs, N, S, nx, nz, scale);
}
template <int K, int NPG, int W = 0>
void launch_diag_k(int dtype, const DiagSet& D, const void* rf, float* out, int F, int N, int S, int nx, int nz, float scale,
                   cudaStream_t st) {
    if (dtype == PAB_I16) launch_diag_t<K, NPG, int16_t, W>(D, rf, out, F, N, S, nx, nz, scale, st);
    else launch_diag_t<K, NPG, float, W>(D, rf, out, F, N, S, nx, nz, scale, st);
}
template <int K, int NPG, int W = 0>
cudaError_t diag_attr(int smem_optin) {
    cudaError_t e = cudaFuncSetAttribute(bf_diag_kernel<K, NPG, float, false, true, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
    if (e != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(bf_diag_kernel<K, NPG, int16_t, false, true, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(bf_diag_kernel<K, NPG, float, false, false, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(bf_diag_kernel<K, NPG, int16_t, false, false, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin);
}

}  // namespace

// pab_self_check: one frame through the checking instantiation (orders <= 3: K = 3; orders 4, 5: K = 5), float input
cudaError_t xl_diag_check(int order, const DiagSet& D, const float* rf, float* out, int N, int S, int nx, int nz, int* d_viol,
                          cudaStream_t st) {
    dim3 grid(D.cfg.tiles_x * D.cfg.tiles_z, 1);
    const DiagTables tabs{D.taps, D.qw0, D.qoff, D.xs_a, D.xs_b, D.zs_a, D.zs_b, D.xs2_max};
    const size_t smem = (size_t)D.smem_bytes + 2 * D.cfg.quads * 4 + 128;
    cudaError_t e;
    const unsigned threads = D.cfg.wpp * D.cfg.parts * 32;
    auto run = [&](auto kernel) -> cudaError_t {
        cudaError_t err = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (err != cudaSuccess) return err;
        kernel<<<grid, threads, smem, st>>>(rf, out, D.cfg, tabs, N, S, nx, nz, 1.0f, d_viol);
        return cudaSuccess;
    };
    // the set's own form: with its tap table, or table-free (taps computed in the kernel)
    if (order <= 3) e = D.taps ? run(bf_diag_kernel<3, 4, float, true, true>) : run(bf_diag_kernel<3, 4, float, true, false>);
    else e = D.taps ? run(bf_diag_kernel<5, 2, float, true, true>) : run(bf_diag_kernel<5, 2, float, true, false>);
    if (e != cudaSuccess) return e;
    return cudaGetLastError();
}

cudaError_t xl_diag_configure(int smem_optin) {
    cudaError_t e;
    if ((e = diag_attr<1, 4>(smem_optin)) != cudaSuccess) return e;
    if ((e = diag_attr<2, 4>(smem_optin)) != cudaSuccess) return e;
    if ((e = diag_attr<3, 4>(smem_optin)) != cudaSuccess) return e;
    if ((e = diag_attr<4, 2>(smem_optin)) != cudaSuccess) return e;
    if ((e = diag_attr<5, 2>(smem_optin)) != cudaSuccess) return e;
    // coherence-factor weighting: 8 pixels per thread at every order
    if ((e = diag_attr<1, 2, 1>(smem_optin)) != cudaSuccess) return e;
    if ((e = diag_attr<2, 2, 1>(smem_optin)) != cudaSuccess) return e;
    if ((e = diag_attr<3, 2, 1>(smem_optin)) != cudaSuccess) return e;
    if ((e = diag_attr<4, 2, 1>(smem_optin)) != cudaSuccess) return e;
    return diag_attr<5, 2, 1>(smem_optin);
}

void xl_diag_free(DiagSet* D) {
    cudaFree(D->taps); cudaFree(D->qw0); cudaFree(D->qoff);
    *D = DiagSet();
}

// Build the tables of one set (npg = 4: orders 1..3, npg = 2: orders 4, 5).  Leaves D->smem_bytes = 0 when the geometry
// does not qualify (N not a multiple of 4, too many warps, a tile that does not fit in shared memory); returns a CUDA
// error only for failed calls.  Synchronises the device.
// mode 0: tap table + windows; 1: the set of the table-free variant: windows only, one sample of margin on either side;
// 2: the table of the nearest-sample path (row f4): floor(idx + 1/2) with fraction 0, so that the same kernel reads
// s = rf[n] exactly.
cudaError_t xl_diag_build(int N, int S, double fs, double c, const pab_grid& g, int q, int npg, int max_order, int smem_limit,
                          int mode, DiagSet* D) {
    const bool with_taps = mode != 1;
    *D = DiagSet();
    const int P = 4 * npg;
    if (N % 4 != 0 || N < 4 || q < 1 || q > 16) return cudaSuccess;
    // Blocking, measured at C2 and C4: 32-row tiles of one column block, 8 warps per CTA (two CTAs
    // per SM at 128 registers); 16-row tiles, 2..16 warps and 2..4 column blocks per tile were all slower.
    constexpr int kRows = 32, kBlocks = 1, kWarps = 8;
    DiagCfg cfg{};
    cfg.q = q;
    cfg.rows = kRows;
    const int lj = 32 / cfg.rows;
    cfg.cp = (q % lj == 0 ? q : q * lj) * kBlocks;      // lcm(q, lj) x column blocks per tile
    cfg.wpp = cfg.cp / lj;
    cfg.cols = P * cfg.cp;
    cfg.tiles_x = (g.nx + cfg.cols - 1) / cfg.cols;
    // seven rows per quarter-warp where eight would span nine samples (pab_pipe.cuh, tile_row): conflict-free gathers
    const double zs_per_row = (double)g.dz * fs / c;
    cfg.tile_rows = (cfg.rows == 32 && zs_per_row > 1.0 && zs_per_row <= 8.0 / 7.0 + 1e-9) ? 28 : cfg.rows;
    cfg.tiles_z = (g.nz + cfg.tile_rows - 1) / cfg.tile_rows;
    cfg.quads = N / 4 + 2;
    cfg.nd = cfg.tiles_x * cfg.cols + q * (N + P + 4);
    if ((long long)cfg.nd * g.nz >= (1LL << 27) || cfg.wpp > kDiagMaxWarps) return cudaSuccess;
    // warps per CTA = wpp * parts: near the target, the split of the diagonal groups with the least idle warp time
    const int G = N / 4 + npg;
    int best_parts = 0;
    double best_cost = 1e30;
    const int target = kWarps;
    const int max_warps = kDiagMaxWarps;
    const int max_parts = std::max(1, std::min(std::min(kDiagMaxParts, max_warps / cfg.wpp), target / cfg.wpp));
    for (int parts = std::max(1, max_parts - 1); parts <= max_parts; ++parts) {
        int lo[kDiagMaxParts + 1];
        const double cost = (double)split_parts(G, npg, N / 4, parts, lo) * parts;        // warp slots of the CTA, idle ones included
        if (cost <= best_cost) { best_cost = cost; best_parts = parts; }
    }
    if (best_parts == 0) return cudaSuccess;
    cfg.parts = best_parts;
    split_parts(G, npg, N / 4, cfg.parts, cfg.part_lo);

    // lateral offsets (metres) of the first and last table column a real pair uses: d = q P (pixel 0, element N - 1) and
    // d = nx - 1 + q (N - 1 + P) (pixel nx - 1, element 0)
    const double half = (N - 1) / 2.0 * q;
    const double ddx_lo = (double)g.x0 - half * (double)g.dx, ddx_hi = (double)g.x0 + ((double)(g.nx - 1) + half) * (double)g.dx;
    const double ddx_max = std::max(std::fabs(ddx_lo), std::fabs(ddx_hi));
    const DiagGeom geo{fs, c, (double)g.x0, (double)g.dx, (double)g.z0, (double)g.dz, N, S, g.nx, g.nz, q, P, ddx_max, mode == 2 ? 1 : 0};
    const size_t tiles = (size_t)cfg.tiles_x * cfg.tiles_z, nq = tiles * cfg.quads;
    int* d_len = nullptr;
    cudaError_t e;
    if (with_taps && (e = cudaMalloc(&D->taps, (size_t)cfg.nd * g.nz * sizeof(uint2))) != cudaSuccess) return e;
    if ((e = cudaMalloc(&D->qw0, nq * sizeof(int))) != cudaSuccess) { xl_diag_free(D); return e; }
    if ((e = cudaMalloc(&D->qoff, (nq + tiles) * sizeof(int))) != cudaSuccess) { xl_diag_free(D); return e; }
    if ((e = cudaMalloc(&d_len, nq * sizeof(int))) != cudaSuccess) { xl_diag_free(D); return e; }
    if (with_taps) diag_taps_kernel<<<dim3((g.nz + 255) / 256, cfg.nd), 256>>>(geo, D->taps);
    diag_window_kernel<<<dim3((unsigned)tiles, cfg.quads), 256>>>(geo, cfg.tile_rows, cfg.cols, cfg.tiles_x, cfg.quads, with_taps ? 0 : 1, D->qw0, d_len);
    std::vector<int> len(nq), off(nq + tiles);
    e = cudaMemcpy(len.data(), d_len, nq * sizeof(int), cudaMemcpyDeviceToHost);
    cudaFree(d_len);
    if (e != cudaSuccess) { xl_diag_free(D); return e; }
    long long worst = 0;
    for (size_t t = 0; t < tiles; ++t) {
        long long o = 0;
        for (int sq = 0; sq < cfg.quads; ++sq) { off[t * (cfg.quads + 1) + sq] = (int)o; o += (long long)len[t * cfg.quads + sq] * 16; }
        off[t * (cfg.quads + 1) + cfg.quads] = (int)o;
        worst = std::max(worst, o);
    }
    if ((e = cudaMemcpy(D->qoff, off.data(), off.size() * sizeof(int), cudaMemcpyHostToDevice)) != cudaSuccess) { xl_diag_free(D); return e; }
    const long long head = ((cfg.quads + 2 * (npg + 1)) * 4 + 127) & ~127;
    const long long red = (long long)cfg.parts * cfg.wpp * P * max_order * 32 * 4;
    const long long smem = head + std::max(worst, red);
    if (smem > smem_limit) { xl_diag_free(D); return cudaSuccess; }          // a tile does not fit: the caller keeps its other kernels
    D->cfg = cfg;
    D->npg = npg;
    D->smem_bytes = (int)smem;
    // diag_ddx / diag_idx in samples: xs(d) = (x0 + (d - q ((N - 1) / 2 + P)) dx) fs / c, zs(m) = (z0 + m dz) fs / c
    D->xs_b = (double)g.dx * fs / c;
    D->xs_a = ((double)g.x0 - (double)q * ((N - 1) / 2.0 + P) * (double)g.dx) * fs / c;
    D->zs_b = (double)g.dz * fs / c;
    D->zs_a = (double)g.z0 * fs / c;
    D->xs2_max = (ddx_max * fs / c) * (ddx_max * fs / c);
    return cudaDeviceSynchronize();
}

// weight = 1 (coherence factor): D must be the 8-pixel set (npg = 2), whatever the order
void xl_diag(int order, int dtype, int weight, const DiagSet& D, const void* rf, float* out, int F, int N, int S, int nx, int nz,
             float scale, cudaStream_t st) {
    if (weight != 0) {
        switch (order) {
        case 1: launch_diag_k<1, 2, 1>(dtype, D, rf, out, F, N, S, nx, nz, scale, st); break;
        case 2: launch_diag_k<2, 2, 1>(dtype, D, rf, out, F, N, S, nx, nz, scale, st); break;
        case 3: launch_diag_k<3, 2, 1>(dtype, D, rf, out, F, N, S, nx, nz, scale, st); break;
        case 4: launch_diag_k<4, 2, 1>(dtype, D, rf, out, F, N, S, nx, nz, scale, st); break;
        default: launch_diag_k<5, 2, 1>(dtype, D, rf, out, F, N, S, nx, nz, scale, st); break;
        }
        return;
    }
    switch (order) {
    case 1: launch_diag_k<1, 4>(dtype, D, rf, out, F, N, S, nx, nz, scale, st); break;
    case 2: launch_diag_k<2, 4>(dtype, D, rf, out, F, N, S, nx, nz, scale, st); break;
    case 3: launch_diag_k<3, 4>(dtype, D, rf, out, F, N, S, nx, nz, scale, st); break;
    case 4: launch_diag_k<4, 2>(dtype, D, rf, out, F, N, S, nx, nz, scale, st); break;
    default: launch_diag_k<5, 2>(dtype, D, rf, out, F, N, S, nx, nz, scale, st); break;
    }
}

}  // namespace pab
