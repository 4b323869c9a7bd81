// pab_math.cuh -- per-item arithmetic of the DMAS-k hot path (steps a2..a6 of DESIGN.md).
//
// Everything here is fp32 on the plain ALUs: FMA/ALU pipes plus the XU (MUFU) pipe for the roots.
// Explicit approximate PTX intrinsics are used instead of a fast-math flag:
//   lg2.approx.ftz / ex2.approx.ftz for the cube and fifth root, sqrt.approx.ftz for order 2,
//   rsqrt.approx.ftz twice for the fourth root, rcp.approx.ftz + sqrt.approx.ftz for the delay.
// lg2(0) = -inf and ex2(-inf) = +0, rsqrt(0) = +inf and rsqrt(+inf) = +0, so the root of zero is zero
// without a branch; a negative argument never reaches a root (|s| is taken first, the sign copied back:
// PAPER.md:41, :62, reading A3).
#pragma once
#include <cuda_runtime.h>

namespace pab {

__device__ __forceinline__ float lg2_approx(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float sqrt_approx(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rsqrt_approx(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rcp_approx(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// The same MUFU operations as volatile statements: ptxas keeps volatile asm statements in program order, which is how
// accumulate_batch pins its stage structure (otherwise the scheduler pulls every consumer up behind its MUFU).
__device__ __forceinline__ float lg2_pinned(float x) { float y; asm volatile("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float ex2_pinned(float x) { float y; asm volatile("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float sqrt_pinned(float x) { float y; asm volatile("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rsqrt_pinned(float x) { float y; asm volatile("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// copysign(|r|, s) as one LOP3: (r & 0x7fffffff) | (s & 0x80000000)
__device__ __forceinline__ float copy_sign(float r, float s) {
    return __uint_as_float((__float_as_uint(r) & 0x7fffffffu) | (__float_as_uint(s) & 0x80000000u));
}

// Step a4 + a5: signed k-th root u = sgn(s)|s|^(1/k) and the running power sums p_m += u^m, m = 1..k,
// with p_k += s (odd k) or |s| (even k), which needs no root (Table I :86-95).
template <int K>
__device__ __forceinline__ void accumulate(float s, float (&p)[K]) {
    if constexpr (K == 1) {
        p[0] += s;                                            // eq. (1)
    } else if constexpr (K == 2) {
        const float u = copy_sign(sqrt_approx(fabsf(s)), s);  // eq. (3)
        p[0] += u;
        p[1] += fabsf(s);
    } else if constexpr (K == 3) {
        const float r = ex2_approx(lg2_approx(fabsf(s)) * (1.0f / 3.0f));
        const float u = copy_sign(r, s);                      // eq. (7): real cube root (A3)
        p[0] += u;
        p[1] = fmaf(u, u, p[1]);
        p[2] += s;
    } else if constexpr (K == 4) {
        const float r = rsqrt_approx(rsqrt_approx(fabsf(s))); // |s|^(1/4); 0 -> inf -> 0
        const float u = copy_sign(r, s);                      // eq. (8): signed fourth root
        const float u2 = r * r;
        p[0] += u;
        p[1] += u2;
        p[2] = fmaf(u2, u, p[2]);
        p[3] += fabsf(s);
    } else if constexpr (K == 5) {
        const float r = ex2_approx(lg2_approx(fabsf(s)) * 0.2f);
        const float u = copy_sign(r, s);                      // eq. (9): real fifth root (A3)
        const float u2 = r * r;
        p[0] += u;
        p[1] += u2;
        p[2] = fmaf(u2, u, p[2]);
        p[3] = fmaf(u2, u2, p[3]);
        p[4] += s;
    } else {
        // Row f2, orders above 5 ("this can be done for higher orders as well").  The power-sum /
        // Newton form loses accuracy to cancellation as k grows (fp32, absorber-free noise frames: 1e-4 at k = 5,
        // 1e-3 at k = 8), so these orders carry the elementary symmetric sums themselves: E_j += u E_(j-1) for
        // j = K..1 (E_0 = 1), O(N) per pixel like the paper's forms, K FMAs per sample, no cancellation.
        // p[j-1] holds E_j; combine<K> returns p[K-1].
        static_assert(K >= 6 && K <= 8, "orders 1..8");
        const float r = ex2_approx(lg2_approx(fabsf(s)) * (1.0f / (float)K));
        const float u = copy_sign(r, s);
#pragma unroll
        for (int j = K - 1; j >= 1; --j) p[j] = fmaf(u, p[j - 1], p[j]);
        p[0] += u;
    }
}

// Step a6: e_k from p_1..p_k by Newton's identities, m e_m = sum_{i=1..m} (-1)^(i-1) e_{m-i} p_i.
// Expanded, these are the paper's eqs. (3), (7), (8), (9) (eq. 9 with the lost square restored, reading A1).
template <int K>
__device__ __forceinline__ float combine(const float (&p)[K]) {
    const float e1 = p[0];
    if constexpr (K == 1) return e1;
    else {
        const float e2 = 0.5f * fmaf(e1, p[0], -p[1]);
        if constexpr (K == 2) return e2;
        else {
            const float e3 = (1.0f / 3.0f) * (fmaf(e2, p[0], -e1 * p[1]) + p[2]);
            if constexpr (K == 3) return e3;
            else {
                const float e4 = 0.25f * ((fmaf(e3, p[0], -e2 * p[1]) + e1 * p[2]) - p[3]);
                if constexpr (K == 4) return e4;
                else if constexpr (K == 5) return 0.2f * (((fmaf(e4, p[0], -e3 * p[1]) + e2 * p[2]) - e1 * p[3]) + p[4]);
                else return p[K - 1];       // orders 6..8 carry E_1..E_K directly (accumulate<K>)
            }
        }
    }
}

// Row f1 (reading A20): coherence-factor weighting, out = CF e_k with CF = (sum s)^2 / (N sum s^2).
// W = 0: none; W = 1: CF.  The accumulator row of one frame is p[0..K-1] (the power sums) followed, for W = 1,
// by sum s^2 and, for even K only (where p_K = sum |s|), by sum s: kAcc<K, W> floats.
template <int K, int W> constexpr int kAcc = K + (W == 0 ? 0 : ((K & 1) ? 1 : 2));

template <int K, int W>
__device__ __forceinline__ void accumulate_w(float s, float (&p)[kAcc<K, W>]) {
    accumulate<K>(s, reinterpret_cast<float (&)[K]>(p));
    if constexpr (W == 1) {
        p[K] = fmaf(s, s, p[K]);
        if constexpr ((K & 1) == 0) p[K + 1] += s;
    }
}

// inv_n = 1 / N.  sum s^2 = 0 (every sample zero or outside the record) gives CF = 0.
template <int K, int W>
__device__ __forceinline__ float combine_w(const float (&p)[kAcc<K, W>], float inv_n) {
    const float e = combine<K>(reinterpret_cast<const float (&)[K]>(p));
    if constexpr (W == 0) return e;
    else {
        const float sum = (K & 1) ? p[K - 1] : p[K + 1];
        const float sq = p[K];
        return sq > 0.0f ? e * (sum * sum * inv_n) * rcp_approx(sq) : 0.0f;
    }
}

// ------------------------------------------------------------------------------------------------------
// Packed forms of a3..a5 for the frame-group kernels: Blackwell issues two independent fp32 operations, each rounded
// as its scalar counterpart, in one slot (PTX add/sub/mul/fma .f32x2, SASS FADD2 / FMUL2 / FFMA2).  The frames a thread
// carries are natural pairs (the x,y and z,w halves of a 128-bit staged sample), so the interpolation, the scaling of
// the logarithm and the power-sum updates take one slot per two frames; the MUFU roots and the LOP3 sign copy stay
// scalar.  Order 3: 6.5 instead of 9 issue slots per item beside the shared loads.
// ------------------------------------------------------------------------------------------------------
#define PAB_U64(v) (reinterpret_cast<unsigned long long&>(v))
__device__ __forceinline__ float2 add2(float2 a, float2 b) {
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(PAB_U64(a)), "l"(PAB_U64(b)));
    return reinterpret_cast<float2&>(r);
}
__device__ __forceinline__ float2 sub2(float2 a, float2 b) {
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(PAB_U64(a)), "l"(PAB_U64(b)));
    return reinterpret_cast<float2&>(r);
}
__device__ __forceinline__ float2 mul2(float2 a, float2 b) {
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(PAB_U64(a)), "l"(PAB_U64(b)));
    return reinterpret_cast<float2&>(r);
}
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) {
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(PAB_U64(a)), "l"(PAB_U64(b)), "l"(PAB_U64(c)));
    return reinterpret_cast<float2&>(r);
}
#undef PAB_U64
__device__ __forceinline__ float2 bcast2(float a) { return make_float2(a, a); }

// a3 for an in-range tap: s = s0 + a (s1 - s0) on two frames
__device__ __forceinline__ float2 interp2(float a, float2 s0, float2 s1) { return fma2(bcast2(a), sub2(s1, s0), s0); }

// Signed cube root of two samples on the FMA and ALU pipes only (no MUFU), so that a fraction of a thread's frames can
// take their root beside the XU pipe instead of queueing for it ("move a fraction of cube roots to a
// division-free Newton iteration for x^(-1/k) on the FMA pipe to balance the two pipes").  y ~ |s|^(-1/3): integer seed
// (magic - bits / 3, residual 1 - |s| y^3 within 0.103), one third-order step y (1 + e/3 + 2 e^2/9), one Newton step
// y (1 + e/3); u = (s y) y carries the sign of s.  Relative error <= 3.8e-7 over 1e-30 .. 1e30 (the lg2/ex2 pair:
// 5e-7 .. 2.7e-6); s = 0 gives 0 (y stays finite).
__device__ __forceinline__ float2 cbrt_fma2(float2 s) {
    const float2 x = make_float2(fabsf(s.x), fabsf(s.y));
    float2 y = make_float2(__uint_as_float(0x54a20000u - __umulhi(__float_as_uint(x.x), 0x55555556u)),
                           __uint_as_float(0x54a20000u - __umulhi(__float_as_uint(x.y), 0x55555556u)));
    float2 e = fma2(mul2(x, y), mul2(y, y), bcast2(-1.0f));                  // -(residual) = |s| y^3 - 1
    y = mul2(y, fma2(fma2(e, bcast2(2.0f / 9.0f), bcast2(-1.0f / 3.0f)), e, bcast2(1.0f)));
    e = fma2(mul2(x, y), mul2(y, y), bcast2(-1.0f));
    y = fma2(mul2(y, e), bcast2(-1.0f / 3.0f), y);
    return mul2(mul2(s, y), y);
}

// a4 + a5 on two frames: p[m] holds the pair's p_(m+1).  The even powers need no sign, so they are formed from the
// unsigned root r; p_K = sum s (odd K) is accumulated from s itself; for even K, |s| = r^K to 2^-22 relative.
// FMA_ROOT (order 3 only): the root of this pair is taken on the FMA pipe (cbrt_fma2) instead of MUFU lg2 + ex2.
template <int K, bool FMA_ROOT = false>
__device__ __forceinline__ void accumulate2(float2 s, float2 (&p)[K]) {
    if constexpr (K == 3 && FMA_ROOT) {
        const float2 u = cbrt_fma2(s);
        p[0] = add2(p[0], u);
        p[1] = fma2(u, u, p[1]);
        p[2] = add2(p[2], s);
    } else if constexpr (K == 1) {
        p[0] = add2(p[0], s);
    } else if constexpr (K == 2) {
        const float2 r = make_float2(sqrt_approx(fabsf(s.x)), sqrt_approx(fabsf(s.y)));
        p[0] = add2(p[0], make_float2(copy_sign(r.x, s.x), copy_sign(r.y, s.y)));
        p[1] = fma2(r, r, p[1]);
    } else if constexpr (K == 3) {
        const float2 t = mul2(make_float2(lg2_approx(fabsf(s.x)), lg2_approx(fabsf(s.y))), bcast2(1.0f / 3.0f));
        const float2 r = make_float2(ex2_approx(t.x), ex2_approx(t.y));
        p[0] = add2(p[0], make_float2(copy_sign(r.x, s.x), copy_sign(r.y, s.y)));
        p[1] = fma2(r, r, p[1]);
        p[2] = add2(p[2], s);
    } else if constexpr (K == 4) {
        const float2 r = make_float2(rsqrt_approx(rsqrt_approx(fabsf(s.x))), rsqrt_approx(rsqrt_approx(fabsf(s.y))));
        const float2 u = make_float2(copy_sign(r.x, s.x), copy_sign(r.y, s.y));
        const float2 u2 = mul2(r, r);
        p[0] = add2(p[0], u);
        p[1] = add2(p[1], u2);
        p[2] = fma2(u2, u, p[2]);
        p[3] = fma2(u2, u2, p[3]);
    } else if constexpr (K == 5) {
        const float2 t = mul2(make_float2(lg2_approx(fabsf(s.x)), lg2_approx(fabsf(s.y))), bcast2(0.2f));
        const float2 r = make_float2(ex2_approx(t.x), ex2_approx(t.y));
        const float2 u = make_float2(copy_sign(r.x, s.x), copy_sign(r.y, s.y));
        const float2 u2 = mul2(r, r);
        p[0] = add2(p[0], u);
        p[1] = add2(p[1], u2);
        p[2] = fma2(u2, u, p[2]);
        p[3] = fma2(u2, u2, p[3]);
        p[4] = add2(p[4], s);
    } else {
        static_assert(K >= 6 && K <= 8, "orders 1..8");          // row f2: E_j += u E_(j-1), j = K..1
        const float2 t = mul2(make_float2(lg2_approx(fabsf(s.x)), lg2_approx(fabsf(s.y))), bcast2(1.0f / (float)K));
        const float2 r = make_float2(ex2_approx(t.x), ex2_approx(t.y));
        const float2 u = make_float2(copy_sign(r.x, s.x), copy_sign(r.y, s.y));
#pragma unroll
        for (int j = K - 1; j >= 1; --j) p[j] = fma2(u, p[j - 1], p[j]);
        p[0] = add2(p[0], u);
    }
}

template <int K, int W, bool FMA_ROOT = false>
__device__ __forceinline__ void accumulate2_w(float2 s, float2 (&p)[kAcc<K, W>]) {
    accumulate2<K, FMA_ROOT>(s, reinterpret_cast<float2 (&)[K]>(p));
    if constexpr (W == 1) {
        p[K] = fma2(s, s, p[K]);
        if constexpr ((K & 1) == 0) p[K + 1] = add2(p[K + 1], s);
    }
}

// a4 + a5 for the NP frame pairs a thread carries, stage by stage over all pairs: every first-stage MUFU of the tap,
// then the scalings, then every second-stage MUFU, then the sign copies and the power-sum updates.  A warp issues in
// order and stalls at the first instruction whose operand is not back yet; the XU pipe serves a warp's MUFU in 8 clocks
// and is shared by the scheduler's warps, so a result returns tens to hundreds of clocks after issue.  Pair by pair
// (accumulate2) the consumer sits a few instructions behind its MUFU and every warp keeps draining the XU queue and
// waiting for it; stage by stage the consumer of MUFU j sits NP - 1 MUFU pairs behind it and the queue stays fed.
// FM: bit j set = pair j takes its root on the FMA pipe (order 3 only, cbrt_fma2).
template <int K, int W, int NP, unsigned FM = 0u>
__device__ __forceinline__ void accumulate_batch(const float2 (&s)[NP], float2 (&p)[NP][kAcc<K, W>]) {
    if constexpr (K == 1) {
#pragma unroll
        for (int j = 0; j < NP; ++j) accumulate2_w<K, W>(s[j], p[j]);
    } else {
        float2 r[NP];
        constexpr bool kLog = K == 3 || K >= 5;             // lg2 -> x 1/K -> ex2; else sqrt (K = 2) or rsqrt twice (K = 4)
#pragma unroll
        for (int j = 0; j < NP; ++j) {
            if ((FM >> j) & 1u) continue;
            if constexpr (kLog) r[j] = make_float2(lg2_pinned(fabsf(s[j].x)), lg2_pinned(fabsf(s[j].y)));
            else if constexpr (K == 2) r[j] = make_float2(sqrt_pinned(fabsf(s[j].x)), sqrt_pinned(fabsf(s[j].y)));
            else r[j] = make_float2(rsqrt_pinned(fabsf(s[j].x)), rsqrt_pinned(fabsf(s[j].y)));
        }
        if constexpr (kLog) {
#pragma unroll
            for (int j = 0; j < NP; ++j)
                if (!((FM >> j) & 1u)) r[j] = mul2(r[j], bcast2(1.0f / (float)K));
        }
        if constexpr (K != 2) {
#pragma unroll
            for (int j = 0; j < NP; ++j) {
                if ((FM >> j) & 1u) continue;
                if constexpr (kLog) r[j] = make_float2(ex2_pinned(r[j].x), ex2_pinned(r[j].y));
                else r[j] = make_float2(rsqrt_pinned(r[j].x), rsqrt_pinned(r[j].y));
            }
        }
#pragma unroll
        for (int j = 0; j < NP; ++j) {
            float2 u;
            if ((FM >> j) & 1u) { u = cbrt_fma2(s[j]); r[j] = u; }           // r only enters through r^2 below
            else u = make_float2(copy_sign(r[j].x, s[j].x), copy_sign(r[j].y, s[j].y));
            float2 (&q)[kAcc<K, W>] = p[j];
            if constexpr (K == 2) {
                q[0] = add2(q[0], u);
                q[1] = fma2(r[j], r[j], q[1]);
            } else if constexpr (K == 3) {
                q[0] = add2(q[0], u);
                q[1] = fma2(r[j], r[j], q[1]);
                q[2] = add2(q[2], s[j]);
            } else if constexpr (K == 4 || K == 5) {
                const float2 u2 = mul2(r[j], r[j]);
                q[0] = add2(q[0], u);
                q[1] = add2(q[1], u2);
                q[2] = fma2(u2, u, q[2]);
                q[3] = fma2(u2, u2, q[3]);
                if constexpr (K == 5) q[4] = add2(q[4], s[j]);
            } else {
#pragma unroll
                for (int m = K - 1; m >= 1; --m) q[m] = fma2(u, q[m - 1], q[m]);
                q[0] = add2(q[0], u);
            }
            if constexpr (W == 1) {
                q[K] = fma2(s[j], s[j], q[K]);
                if constexpr ((K & 1) == 0) q[K + 1] = add2(q[K + 1], s[j]);
            }
        }
    }
}

// the pair's accumulator rows unpacked: half h (0 / 1) of p[0..kAcc) as the scalar row combine_w expects
template <int K, int W>
__device__ __forceinline__ float combine2_w(const float2 (&p)[kAcc<K, W>], int h, float inv_n) {
    float q[kAcc<K, W>];
#pragma unroll
    for (int k = 0; k < kAcc<K, W>; ++k) q[k] = h == 0 ? p[k].x : p[k].y;
    return combine_w<K, W>(q, inv_n);
}

// Step a2 + the index half of a3, once per (pixel, element), shared by every frame a thread carries.
//   xs2, c0      the lateral offset xs = pixel - element (samples) enters only through its square, passed as
//                xs2 = fl(xs_hi^2) and c0 = xs2 - xs^2 (the rounding error of the square plus the low part of xs),
//                both uniform over a warp and computed once per (tile, element) by the producer
//   row  (zs_hi, 2 zs_lo, zf - 1/2, zi - 2 * 0x4B400000 as int bits): zs = z fs / c = zs_hi + zs_lo = zi + zf,
//        zi = floor(zs), all from an fp64 host computation
//   idx = fs sqrt(dx^2 + z^2) / c = zs + delta, where delta >= 0 solves
//         delta (delta + 2 zs) = xs^2.
// The signed k-th root is not Lipschitz at 0, so an index error e costs ~e^(5/6) in the image: the index is
// therefore carried to ~1e-6 samples, not to an fp32 ulp of the 11-12 bit index (DESIGN.md "Delay index
// precision").  One MUFU (rsqrt) gives d0 ~ sqrt(xs^2 + zs^2); delta0 = d0 - zs; one Newton step on
// f(delta) = delta (delta + 2 zs) - xs^2 (f' ~ 2 d0, step -f r / 2) with f evaluated in compensated arithmetic:
// exact xs^2 = xs2 + xs2_lo (FMA), exact delta0 + 2 zs = t_hi + t_lo (branch-free TwoSum), and the first-order terms of
// the low parts of xs and zs.  The correction is NOT folded back into delta0: delta0 is split exactly into an
// integer n0 and a fraction, and the fractions (of zs, of delta0, the correction) are summed at full relative
// precision; floor(zs) and n0 only ever meet as integers.
// INR = true: the host has checked that every (pixel, element) index of the geometry lies inside the record
// and z > 0, so no validity mask is produced and s = s0 + wa (s1 - s0).  INR = false: i0 is clamped into
// [0, S-2] and wa, wb are both 0 when the delayed sample falls outside the record (reading A6).
struct Tap { int i0; float wa, wb; };

template <bool INR>
__device__ __forceinline__ Tap delay_tap(float xs2, float c0, const float4 row, int S) {
    const float kMagic = 12582912.0f;                           // 1.5 * 2^23: adding it rounds to an integer
    float q = fmaf(row.x, row.x, xs2);
    if constexpr (!INR) q = fmaxf(q, 1e-30f);
    const float r = rsqrt_approx(q);
    const float d0 = q * r;
    float delta0 = d0 - row.x;
    if constexpr (!INR) delta0 = fminf(fmaxf(delta0, 0.0f), 2097152.0f);
    const float z2 = row.x + row.x;
    const float t_hi = z2 + delta0;                             // delta0 + 2 zs_hi = t_hi + t_lo exactly: TwoSum, valid
    const float bb = t_hi - z2;                                 // for either order of magnitudes (delta0 > 2 zs for
    const float t_lo = (z2 - (t_hi - bb)) + (delta0 - bb);      // shallow rows seen by far elements)
    float g = fmaf(delta0, t_lo, c0);                           // low-order part of f: delta0 t_lo - (xs^2 - xs2)
    g = fmaf(delta0, row.y, g);                                 //                      + delta0 * 2 zs_lo
    const float f = fmaf(delta0, t_hi, -xs2) + g;
    const float t0 = delta0 + kMagic;
    const float n0 = t0 - kMagic;                               // nearest integer to delta0 (exact)
    // Newton step -f r / 2, kept apart from delta0: idx - zi - n0 - 1/2 = frac parts + step, |w| <= ~1
    const float w = fmaf(f * r, -0.5f, row.z + (delta0 - n0));
    const float t1 = w + kMagic;
    const float fl = t1 - kMagic;
    const int i0 = __float_as_int(row.w) + __float_as_int(t0) + __float_as_int(t1);   // zi + n0 + floor part
    const float a = (w - fl) + 0.5f;
    Tap o;
    if constexpr (INR) {
        o.i0 = i0; o.wa = a; o.wb = 0.0f;
    } else {
        const bool ok = (unsigned)i0 <= (unsigned)(S - 2);
        o.i0 = ok ? i0 : 0;
        o.wa = ok ? a : 0.0f;
        o.wb = ok ? 1.0f - a : 0.0f;
    }
    return o;
}

// The same step for in-range geometries on the FP64 pipe (B200: 64 lanes/clk/SM beside the FP32 pipes, otherwise idle in
// this library): idx = sqrt(xs^2 + zs^2) from one MUFU.RSQ64H seed and one Newton step in double (relative error ~1e-12),
// then floor and fraction by two rounding constants, with no conversion instruction (F2I / F2F would queue on the XU pipe
// beside the roots): M = 1.5 * 2^52 has ulp 1, so t = (idx - 1/2) + M holds floor(idx) in its low word (ties fall either
// way); M2 = 1.5 * 2^29 has ulp 2^-23, so u = idx + ((M + M2) - t) = fraction + M2 (the inner difference is exact) holds
// round(fraction * 2^23) = 0 .. 2^23 in its low word, and 0x3f800000 + that is the float 1 + fraction, up to 2.0 when the
// fraction rounds to 1 or a tie went down: weight 1 on the upper sample, the same value.  11 instructions per call, 10 of
// them on the FP64 pipe, against 23 on the FP32 / ALU pipes above.
//   xs2d  the lateral offset squared, in samples^2 (double; warp-uniform, from the producer)
//   zs    z fs / c (double)
// Returns floor(idx) (or floor(idx) - 1 with fraction 1) and the fraction in [0, 1], good to 2^-24 samples.
__device__ __forceinline__ Tap delay_tap_f64(double xs2d, double zs) {
    const double q = fma(zs, zs, xs2d);
    double r;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(q));
    double d = q * r;
    const double e = fma(-d, d, q);
    d = fma(e * r, 0.5, d);                                        // sqrt(q) to ~1e-12 relative
    const double kM = 6755399441055744.0;                          // 1.5 * 2^52
    const double kMM2 = 6755400246362112.0;                        // 1.5 * 2^52 + 1.5 * 2^29, exact
    const double t = (d - 0.5) + kM;
    const double u = d + (kMM2 - t);
    Tap o;
    o.i0 = __double2loint(t);
    o.wa = __int_as_float(0x3f800000 + __double2loint(u)) - 1.0f;
    o.wb = 0.0f;
    return o;
}

// (xs2, c0) of delay_tap from the hi + lo table entries of a pixel column and an element, in fp32 with
// error-free differences (the direct kernel; the staged kernel's producer does this in fp64)
__device__ __forceinline__ float2 lateral_square(float2 xj, float2 xe) {
    const float a = xj.x - xe.x;
    const float bv = a - xj.x;
    const float ea = (xj.x - (a - bv)) - (xe.x + bv);           // a + ea = xj.x - xe.x exactly
    const float l = ea + (xj.y - xe.y);
    const float hi = a + l;
    const float lo = l - (hi - a);
    const float xs2 = hi * hi;
    return make_float2(xs2, -fmaf(hi, lo + lo, fmaf(hi, hi, -xs2)));
}

// Step a3: the interpolated sample from its two neighbours.
template <bool INR>
__device__ __forceinline__ float interp(const Tap& t, float s0, float s1) {
    if constexpr (INR) return fmaf(t.wa, s1 - s0, s0);
    else return fmaf(t.wa, s1, t.wb * s0);
}
// the same on two frames (packed)
template <bool INR>
__device__ __forceinline__ float2 interp2(const Tap& t, float2 s0, float2 s1) {
    if constexpr (INR) return interp2(t.wa, s0, s1);
    else return fma2(bcast2(t.wa), s1, mul2(bcast2(t.wb), s0));
}

}  // namespace pab
