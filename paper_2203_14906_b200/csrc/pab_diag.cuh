// pab_diag.cuh -- the single-frame beamforming kernel for translation-invariant geometries (calls of 1..3 frames, and the
// 1..3 frames a longer call leaves over after its whole quads).
//
// With one frame per thread nothing amortises the tap fetch, the address and the loop of a (pixel, element) pair: the
// frame-group kernels share them over 16 frames.  When the pitch is an exact integer multiple q of the column spacing
// (pab_cache.cuh: "compact table"), the delay of (column j, element i) depends on j - q i only, so the pairs on a
// DIAGONAL share their tap the way frames do: a thread owns the P pixels of row m at columns j0 + q c, c = 0..P-1, and
// for diagonal e the P pairs (c, element e + c) all have the tap of d = j0 - q e.  One tap fetch and one set of
// addresses then serve P items, and the inner loop is the frame-group kernels' (packed f32x2 interpolation and power
// sums, steps a3..a5), with the P pixels in the place of the 16 frames.
//
// The samples of those P pairs belong to P consecutive channels.  The RF tile is therefore staged CHANNEL-QUAD
// interleaved, [quad g][sample][4 channels 4g..4g+3], so that one 128-bit shared load brings a sample of 4 neighbouring
// channels: diagonal e = 4 eg + r pairs pixel c with component (r + c) % 4 of quad eg + (r + c) / 4, a compile-time
// selection under a 4-way unroll over r.  The staging does the transposition (coalesced global reads along the sample
// axis of the caller's [N][S] frame, 128-bit shared stores), converting int16 on the way, so the frame is read from HBM
// once, in place, without an ingest pass.  Channels before the first and after the last element are a zero quad each,
// so pairs that fall off the array contribute u = 0 to every power sum; whole blocks of 4 x 4 such pairs are skipped.
//
// A CTA owns a tile of 32 rows x (P q) columns and every diagonal; its warps split the columns' q residues and the
// diagonals (EP parts, balanced on the host), and the partial power sums meet in shared memory before the Newton
// combination (step a6).  Per (tile, staged quad) the window start and its place in shared memory come from tables
// built once per geometry in fp64 with the same expression as the taps, so table and window agree exactly.
//
// Two forms.  TAB = true (delay cache on): the tap of every (table column d, row) comes from a table built with that
// expression.  TAB = false (delay cache off: the default): no tap table; the kernel computes the tap of a diagonal itself
// on the FP64 pipe (delay_tap_f64, one per (thread, diagonal), one diagonal ahead of its use), and the windows carry one
// sample of margin because that evaluation agrees with the table expression to ~1e-9 samples, not to the bit.
#pragma once
#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>
#include "pab_math.cuh"
#include "pab_pipe.cuh"

namespace pab {

// idx of (tap-table column d, row m): the lateral offset is x0 + (d - q (N - 1 + P) - ... ) dx; see diag_ddx
struct DiagGeom {
    double fs, c, x0, dx, z0, dz;
    int N, S, nx, nz, q, P;
    double ddx_max;         // largest |pixel column - element| (metres) of a real pair: max over table columns q P and nx - 1 + q (N - 1 + P)
    int nearest;            // 1: the table holds floor(idx + 1/2) with fraction 0 (row f4: integer delays, reading A21)
};
// lateral offset (pixel column - element) of table column d: d = j - q i + q (N - 1 + P), x_j - x_i = x0 + j dx - (i - (N-1)/2) q dx
// Table columns beyond those of the real pairs belong only to pairs that do not exist (pixel columns past nx in a ragged last
// tile, the zero quads beside the array).  Their lateral offset is capped at the largest one a real pair has, so that every
// tap lies inside the record like the real ones (the geometry is in range) and inside the windows, which are built from
// this same expression; what such pairs read is never stored (columns past nx) or is zero (zero quads).
__device__ __forceinline__ double diag_ddx(const DiagGeom& G, int d) {
    const double k = __dsub_rn((double)d, __dmul_rn((double)G.q, __dadd_rn(__ddiv_rn(__dsub_rn((double)G.N, 1.0), 2.0), (double)G.P)));
    return fmin(fabs(__dadd_rn(G.x0, __dmul_rn(k, G.dx))), G.ddx_max);
}
__device__ __forceinline__ double diag_idx(const DiagGeom& G, int d, int m) {
    const double z = __dadd_rn(G.z0, __dmul_rn((double)m, G.dz));
    const double ddx = diag_ddx(G, d);
    return __ddiv_rn(__dmul_rn(G.fs, __dsqrt_rn(__dadd_rn(__dmul_rn(ddx, ddx), __dmul_rn(z, z)))), G.c);
}

// taps[d * nz + m].  grid: (ceil(nz / 256), nd)
__global__ void __launch_bounds__(256) diag_taps_kernel(const DiagGeom G, uint2* __restrict__ taps) {
    const int m = blockIdx.x * blockDim.x + threadIdx.x, d = blockIdx.y;
    if (m >= G.nz) return;
    const double idx = diag_idx(G, d, m);
    if (G.nearest) {            // the integer decision of the nearest-sample path, taken here in fp64 like its uint16 table's
        taps[(size_t)d * G.nz + m] = make_uint2((unsigned)(int)floor(__dadd_rn(idx, 0.5)), 0u);
        return;
    }
    const double fl = floor(idx);
    taps[(size_t)d * G.nz + m] = make_uint2((unsigned)(int)fl, __float_as_uint((float)(idx - fl)));
}

// Window of every (tile, staged quad): first sample and length.  The extremes of idx over the tile lie on its first and
// last row (idx grows with depth), at some column: all columns of both rows are evaluated for the quad's 4 channels.
// grid: (tiles_x * tiles_z, quads); block: 256 threads >= cols * 2 ... (loops).  sq = 0 is the zero quad before the
// array (channels -4..-1), sq = quads - 1 the one after it.
// margin: extra samples on either side (the table-free variant computes its taps in the kernel, to ~1e-9 samples of this
// expression: a floor that falls the other way at a window's edge must still land inside it).
__global__ void __launch_bounds__(256) diag_window_kernel(const DiagGeom G, int rows, int cols, int tiles_x, int quads, int margin,
                                                           int* __restrict__ qw0, int* __restrict__ qlen) {
    __shared__ int s_min, s_max;
    const int tile = blockIdx.x, sq = blockIdx.y;
    const int bx = tile % tiles_x, by = tile / tiles_x;
    if (threadIdx.x == 0) { s_min = 0x7fffffff; s_max = -0x7fffffff; }
    __syncthreads();
    const int r_lo = by * rows, r_hi = min(r_lo + rows, G.nz) - 1;
    int lo = 0x7fffffff, hi = -0x7fffffff;
    for (int t = threadIdx.x; t < cols * 8; t += blockDim.x) {
        const int col = t % cols, ch = (t / cols) % 4, top = t / (cols * 4);
        const int j = bx * cols + col, i = (sq - 1) * 4 + ch;
        const int d = j - G.q * i + G.q * (G.N - 1 + G.P);
        const double ix = diag_idx(G, d, top ? r_hi : r_lo);
        const int fl = (int)floor(G.nearest ? __dadd_rn(ix, 0.5) : ix);
        lo = min(lo, fl); hi = max(hi, fl);
    }
    atomicMin(&s_min, lo);
    atomicMax(&s_max, hi);
    __syncthreads();
    if (threadIdx.x == 0) {
        const bool real = sq >= 1 && sq <= quads - 2;
        int w0 = s_min - margin, w1 = s_max + 2 + margin;    // samples [w0, w1): i0 and i0 + 1 of every pair
        if (real) { w0 = max(w0, 0); w1 = min(w1, G.S); }
        qw0[(size_t)tile * quads + sq] = w0;
        qlen[(size_t)tile * quads + sq] = max(w1 - w0, 0);
    }
}

template <typename T> __device__ __forceinline__ float diag_ld(const T* p) { return (float)__ldg(p); }

// K: order 1..5.  NPG: pixel groups of 4 per thread (P = 4 NPG pixels: 4 for orders 1..3, 2 for orders 4, 5).
// T: float or int16_t (the caller's frame, read in place).  CTAs of up to 16 warps at 128 registers (NPG = 4) or up to 8
// warps at 80 registers, three CTAs per SM (NPG = 2).
// CHK (pab_self_check): every shared-memory gather of the element loop is compared with the staged window of its quad and
// out-of-window accesses are counted in *viol (compute-sanitizer is closed on this GPU pool; this kernel's addressing is
// the most intricate of the library).
// TAB = false: no tap table; the tap of a diagonal comes from delay_tap_f64 (FP64 pipe), computed one diagonal ahead the
// way the table variant prefetches it: 13 instructions per (thread, diagonal), shared by the thread's P pairs.
// W = 1: coherence-factor weighting (row f1): the accumulator row of a pixel grows by sum s^2 (and sum s for even K), and
// the epilogue multiplies e_k by (sum s)^2 / (N sum s^2) (combine_w); 8 pixels per thread for every order.
template <int K, int NPG, typename T, bool CHK = false, bool TAB = true, int W = 0>
__global__ void __launch_bounds__(kDiagMaxWarps * 32, 1) bf_diag_kernel(const T* __restrict__ rf, float* __restrict__ out,
                                                                          const DiagCfg C, const DiagTables D, int N, int S,
                                                                          int nx, int nz, float scale, int* __restrict__ viol = nullptr) {
    constexpr int P = 4 * NPG;
    constexpr int A = kAcc<K, W>;                    // accumulators per pixel
    extern __shared__ __align__(128) unsigned char dg_smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n_warps = blockDim.x >> 5;
    const int tile = blockIdx.x, frame = blockIdx.y;
    const int bx = tile % C.tiles_x, by = tile / C.tiles_x;
    // [NPG + 1 spare][quads][NPG + 1 spare] shared address of sample 0 of each staged quad (the spares are never used
    // for loads: the blocks that would are skipped; they keep the index arithmetic free of clamps)
    int* s_base = reinterpret_cast<int*>(dg_smem) + (NPG + 1);
    const int head_bytes = ((C.quads + 2 * (NPG + 1) + (CHK ? 2 * C.quads : 0)) * 4 + 127) & ~127;
    int* s_lim = s_base + C.quads + (NPG + 1);                               // CHK: [quads][2] window limits
    const uint32_t stage0 = smem_u32(dg_smem) + head_bytes;
    const int* qw0 = D.qw0 + (size_t)tile * C.quads;
    const int* qoff = D.qoff + (size_t)tile * (C.quads + 1);

    // ---- staging: transpose the tile's windows into the channel-quad layout (a1) ----
    const T* fr = rf + (size_t)frame * N * (size_t)S;
    for (int sq = warp; sq < C.quads; sq += n_warps) {
        const int w0 = __ldg(qw0 + sq), o0 = __ldg(qoff + sq), len = (__ldg(qoff + sq + 1) - o0) >> 4;
        if (lane == 0) s_base[sq] = (int)(stage0 + o0) - w0 * 16;
        if (CHK && lane == 0) { s_lim[2 * sq] = (int)(stage0 + o0); s_lim[2 * sq + 1] = (int)(stage0 + o0) + len * 16 - 32; }
        const bool real = sq >= 1 && sq <= C.quads - 2;
        const T* ch0 = fr + (size_t)((sq - 1) * 4) * S + w0;
        for (int s0 = 0; s0 < len; s0 += 64) {                               // two samples per lane in flight
            float4 v[2];
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int s = s0 + u * 32 + lane;
                v[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (real && s < len)
                    v[u] = make_float4(scale * diag_ld(ch0 + s), scale * diag_ld(ch0 + S + s), scale * diag_ld(ch0 + 2 * (size_t)S + s),
                                       scale * diag_ld(ch0 + 3 * (size_t)S + s));
            }
#pragma unroll
            for (int u = 0; u < 2; ++u) {
                const int s = s0 + u * 32 + lane;
                if (s < len)
                    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(stage0 + o0 + s * 16), "f"(v[u].x), "f"(v[u].y),
                                 "f"(v[u].z), "f"(v[u].w) : "memory");
            }
        }
    }
    __syncthreads();

    // ---- a2..a5 over this warp's diagonals ----
    // lane = (row of the tile, column phase inside the warp); phase ph = residue ph % q of column block ph / q
    const int part = warp / C.wpp, wph = warp % C.wpp;
    const int ph = wph * (32 / C.rows) + lane / C.rows;
    // 28-row tiles (row pitches in (1, 8/7] samples): seven rows per quarter-warp keep the 128-bit gathers of a quarter on
    // 8 distinct bank groups; the eighth lane repeats its neighbour's row (same addresses: a broadcast) and stores nothing
    const bool r7 = C.tile_rows != C.rows;
    const int trow = r7 ? (lane >> 3) * 7 + min(lane & 7, 6) : lane % C.rows;
    const bool live = !r7 || (lane & 7) != 7;
    const int m = by * C.tile_rows + trow;
    const int j0 = bx * C.cols + (ph % C.q) + (ph / C.q) * (P * C.q);
    const int mc = min(m, nz - 1);
    float2 pp[P / 2][A];
#pragma unroll
    for (int f = 0; f < P / 2; ++f)
#pragma unroll
        for (int k = 0; k < A; ++k) pp[f][k] = make_float2(0.0f, 0.0f);
    const int n_quads_real = C.quads - 2;
    // Tap of diagonal e = 4 eg + r: table column d = j0 - q e + q (N - 1 + P), i.e. entry t0 - f * tstep for the flat
    // diagonal index f = 4 egp + r (egp = eg + NPG >= 0).  The table is wide enough for every f a part can touch, one
    // past its end included (the prefetch), so there are no clamps.  The tap of diagonal f + 1 is fetched while f computes.
    const uint32_t tstep = (uint32_t)C.q * (uint32_t)nz;
    const uint32_t t0 = (uint32_t)(j0 + C.q * (N - 1 + P + 4 * NPG)) * (uint32_t)nz + (uint32_t)mc;
    const int f_lo = 4 * C.part_lo[part];
    // table-free: lateral offset (samples) of the next diagonal, stepped by -q xs_b per diagonal; depth of this lane's row
    double xs_next = 0.0, xs_step = 0.0, zs = 0.0;
    int i0_cap = 0x7fffffff;
    uint2 tap_next;
    if constexpr (TAB) {
        tap_next = __ldg(D.taps + (t0 - (uint32_t)f_lo * tstep));
    } else {
        xs_step = -(double)C.q * D.xs_b;
        xs_next = fma((double)(j0 + C.q * (N - 1 + P + 4 * NPG) - C.q * f_lo), D.xs_b, D.xs_a);
        zs = fma((double)mc, D.zs_b, D.zs_a);
        // diag_ddx's cap on the lateral offset, as one integer minimum per tap: no real pair of this row has a delay beyond
        // that of the largest real offset (+1: the two evaluations may floor a borderline value differently; the windows
        // of this form carry that sample of margin)
        i0_cap = delay_tap_f64(D.xs2_max, zs).i0 + 1;
        const Tap t = delay_tap_f64(xs_next * xs_next, zs);
        tap_next = make_uint2((unsigned)min(t.i0, i0_cap), __float_as_uint(t.wa));
        xs_next += xs_step;
    }
    for (int egp = C.part_lo[part]; egp < C.part_lo[part + 1]; ++egp) {
        const int eg = egp - NPG;                                      // first quad (unpadded index) of the group
        const uint32_t tg = t0 - (uint32_t)(4 * egp + 1) * tstep;      // entry of the group's second diagonal
        int qb[NPG + 1];
#pragma unroll
        for (int k = 0; k <= NPG; ++k) qb[k] = s_base[eg + k + 1];
        // GUARD: pixel groups whose 4 x 4 block of pairs lies off the array are skipped (the ends of the diagonal range);
        // the test is uniform over the warp
        auto diagonal = [&](auto rc, auto gc) {
            constexpr int r = decltype(rc)::value;
            constexpr bool GUARD = decltype(gc)::value;
            const float a = __uint_as_float(tap_next.y);
            const uint32_t off = tap_next.x * 16u;
            if constexpr (TAB) {
                tap_next = __ldg(D.taps + (tg - (uint32_t)r * tstep));       // diagonal f + 1
            } else {
                const Tap t = delay_tap_f64(xs_next * xs_next, zs);
                tap_next = make_uint2((unsigned)min(t.i0, i0_cap), __float_as_uint(t.wa));
                xs_next += xs_step;
            }
            float4 lo0, lo1;                                                   // samples i0, i0 + 1 of quad eg + cg
            bool have = false;
#pragma unroll
            for (int cg = 0; cg < NPG; ++cg) {
                if constexpr (GUARD) {
                    if (!(eg + cg + 1 >= 0 && eg + cg < n_quads_real)) { have = false; continue; }      // no channel of the block is real
                }
                if constexpr (CHK) {          // both quads of the block: [first byte, last 32-byte pair] of their staged windows
#pragma unroll
                    for (int k = 0; k < (r != 0 ? 2 : 1); ++k) {
                        const int sq = eg + cg + k + 1, a = qb[cg + k] + (int)off;
                        const int* lim = s_lim + 2 * sq;
                        if (a < lim[0] || a > lim[1]) atomicAdd(viol, 1);
                    }
                }
                if (GUARD ? !have : (cg == 0 || r == 0)) { lo0 = lds128((uint32_t)qb[cg] + off); lo1 = lds128((uint32_t)qb[cg] + off + 16); }
                float4 hi0 = lo0, hi1 = lo1;
                if constexpr (r != 0) { hi0 = lds128((uint32_t)qb[cg + 1] + off); hi1 = lds128((uint32_t)qb[cg + 1] + off + 16); }
                // pixel c = 4 cg + t pairs with component r + t: of lo for r + t < 4, of hi otherwise
                const float s0v[8] = {lo0.x, lo0.y, lo0.z, lo0.w, hi0.x, hi0.y, hi0.z, hi0.w};
                const float s1v[8] = {lo1.x, lo1.y, lo1.z, lo1.w, hi1.x, hi1.y, hi1.z, hi1.w};
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const float2 x0 = make_float2(s0v[r + 2 * h], s0v[r + 2 * h + 1]);
                    const float2 x1 = make_float2(s1v[r + 2 * h], s1v[r + 2 * h + 1]);
                    float2 v;
                    if constexpr ((r & 1) == 0) v = interp2(a, x0, x1);            // an aligned register pair: packed
                    else v = make_float2(fmaf(a, x1.x - x0.x, x0.x), fmaf(a, x1.y - x0.y, x0.y));
                    accumulate2_w<K, W>(v, pp[2 * cg + h]);
                }
                if constexpr (r != 0) { lo0 = hi0; lo1 = hi1; have = true; }
            }
        };
        if (eg >= -1 && eg + NPG - 1 < n_quads_real) {
            diagonal(std::integral_constant<int, 0>{}, std::false_type{});
            diagonal(std::integral_constant<int, 1>{}, std::false_type{});
            diagonal(std::integral_constant<int, 2>{}, std::false_type{});
            diagonal(std::integral_constant<int, 3>{}, std::false_type{});
        } else {
            diagonal(std::integral_constant<int, 0>{}, std::true_type{});
            diagonal(std::integral_constant<int, 1>{}, std::true_type{});
            diagonal(std::integral_constant<int, 2>{}, std::true_type{});
            diagonal(std::integral_constant<int, 3>{}, std::true_type{});
        }
    }

    // ---- partial power sums of the parts meet in shared memory (the staging area is dead now) ----
    __syncthreads();
    float* red = reinterpret_cast<float*>(dg_smem + head_bytes);       // [part][warp of the part][P][A][32]
    {
        float* mine = red + (size_t)((part * C.wpp + wph) * P * A) * 32 + lane;
#pragma unroll
        for (int f = 0; f < P / 2; ++f)
#pragma unroll
            for (int k = 0; k < A; ++k) {
                mine[((2 * f) * A + k) * 32] = pp[f][k].x;
                mine[((2 * f + 1) * A + k) * 32] = pp[f][k].y;
            }
    }
    __syncthreads();
    // ---- a6: pixel c of this lane's column phase is finished by part c % parts ----
    const size_t img = (size_t)nz * nx;
    const float inv_n = 1.0f / (float)N;
    for (int c = part; c < P; c += C.parts) {
        float p[A];
#pragma unroll
        for (int k = 0; k < A; ++k) p[k] = 0.0f;
        for (int pt = 0; pt < C.parts; ++pt) {
            const float* src = red + (size_t)(((pt * C.wpp + wph) * P + c) * A) * 32 + lane;
#pragma unroll
            for (int k = 0; k < A; ++k) p[k] += src[k * 32];
        }
        const int j = j0 + C.q * c;
        if (live && j < nx && m < nz) out[(size_t)frame * img + (size_t)m * nx + j] = combine_w<K, W>(p, inv_n);
    }
}

}  // namespace pab
