/*
 * pab_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of what the hot path of arxiv 2203.14906
 * ("Higher-order correlation based real-time beamforming in photoacoustic
 * imaging") computes: delay -> linear interpolation -> order-k DMAS
 * combination -> axial band-pass -> Hilbert-FIR envelope -> log compression.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this file.  It shares no code, header, table
 * or constant with the CUDA library (paper_2203_14906_b200/csrc) and neither
 * includes the other.
 *
 * No blocking, no tables, no fusion: every function is the definition in the
 * cited passage written out as loops.  OpenMP only splits the outermost pixel
 * row loop across host cores (no change in per-pixel arithmetic or order).
 *
 * Citations are PAPER.md:<line> and the reading
 * numbers A1..A19 of DESIGN.md ("Readings of the paper").
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"):
 *   orc_gather            numpy np.interp on numpy-computed delays; linear-ramp closed form (P7)
 *   orc_combine_recur     brute-force k-subset enumeration (orc_combine_brute = eqs. 2,4,5,6 as
 *                         printed), binomial closed form C(N,k)*a (P4), fewer-than-k-nonzero -> 0 (P5),
 *                         python itertools re-enumeration on tiny N
 *   orc_combine_closed    the paper's printed eqs. (3),(7),(8),(9) vs the two above (eq. 9 with
 *                         repair A1; the as-printed form is also kept and shown NOT to be e5)
 *   orc_beamform          order 1 == orc_das bitwise (P1); point absorber peaks at its pixel (P8);
 *                         homogeneity and channel-reversal symmetry (P6)
 *   orc_beamform_ex       interp = 0, weight = 0 == orc_beamform bitwise; nearest: numpy rint gather written
 *                         independently, staircase-RF closed form; CF: hand value 6/7 for (1,2,3), CF = 1 for equal
 *                         samples, 0 for +-a pairs, bounds [0,1], scale invariance, constant-RF closed form C(N,k) a
 *   orc_image_metrics     numpy mean / std / histogram written independently; gCNR = 1 for disjoint and 0 for
 *                         identical regions; SNR, CR of constant regions; FWHM of a sampled Gaussian = 2.3548 sigma
 *   orc_bandpass_taps     scipy.signal.firwin(scale=False) ; symmetry
 *   orc_hilbert_taps      antisymmetry, zero even taps, closed form 2/(pi t) * Hamming
 *   orc_fir_axial         numpy.convolve
 *   orc_envelope          scipy.signal.hilbert (FFT analytic signal) on an in-band tone (P9)
 *   orc_logcompress       closed form on known ratios
 * Nothing in the paper prints a beamformed pixel value, so no pin is a paper-printed number;
 * absolute values are pinned by the closed forms and brute force above.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_F32 0
#define ORC_I16 1

typedef struct {
    int nx, nz;          /* columns (lateral), rows (depth) */
    double x0, dx, z0, dz; /* metres; pixel (m, j) centre = (x0 + j*dx, z0 + m*dz) */
} orc_grid;

static double rf_at(const void* rf, int dtype, double scale, size_t off) {
    if (dtype == ORC_I16) return scale * (double)((const int16_t*)rf)[off]; /* A15: exact int16 -> double */
    return scale * (double)((const float*)rf)[off];
}

/* O1: element i of a linear array centred on x = 0 at z = 0 (reading A5). */
double orc_elem_x(int i, int n_elem, double pitch) { return ((double)i - ((double)n_elem - 1.0) / 2.0) * pitch; }

/* O3: one-way time of flight in samples, record starts at t = 0 (eq. 1's Delta_i; A5). */
double orc_delay_idx(double x, double z, double xe, double fs, double c) {
    double ddx = x - xe;
    return fs * sqrt(ddx * ddx + z * z) / c;
}

/* O4: linear interpolation of one channel at fractional index idx; 0 outside the record
 * (eq. 1 PAPER.md:29 with readings A4, A6). */
static double interp_chan(const void* rf, int dtype, double scale, size_t chan_off, int S, double idx) {
    double fl = floor(idx);
    double a = idx - fl;
    if (!(fl >= 0.0) || !(fl + 1.0 <= (double)(S - 1))) return 0.0;
    size_t i0 = (size_t)fl;
    double s0 = rf_at(rf, dtype, scale, chan_off + i0);
    double s1 = rf_at(rf, dtype, scale, chan_off + i0 + 1);
    return (1.0 - a) * s0 + a * s1;
}

/* delayed samples s_i of every element for one pixel of one frame */
static void pixel_samples(const void* rf, int dtype, double scale, int frame, int N, int S, double fs, double c,
                          double pitch, double x, double z, double* s) {
    for (int i = 0; i < N; ++i) {
        double xe = orc_elem_x(i, N, pitch);
        double idx = orc_delay_idx(x, z, xe, fs, c);
        s[i] = interp_chan(rf, dtype, scale, ((size_t)frame * N + i) * (size_t)S, S, idx);
    }
}

/* all delay indices, idx_out[nz][nx][N]  (test hook for O1-O3) */
void orc_delays(int N, double fs, double c, double pitch, const orc_grid* g, double* idx_out) {
    for (int m = 0; m < g->nz; ++m)
        for (int j = 0; j < g->nx; ++j)
            for (int i = 0; i < N; ++i)
                idx_out[((size_t)m * g->nx + j) * N + i] =
                    orc_delay_idx(g->x0 + j * g->dx, g->z0 + m * g->dz, orc_elem_x(i, N, pitch), fs, c);
}

/* all delayed samples of one frame, s_out[nz][nx][N]  (test hook for O4) */
void orc_gather(const void* rf, int dtype, double scale, int frame, int N, int S, double fs, double c, double pitch,
                const orc_grid* g, double* s_out) {
    for (int m = 0; m < g->nz; ++m)
        for (int j = 0; j < g->nx; ++j)
            pixel_samples(rf, dtype, scale, frame, N, S, fs, c, pitch, g->x0 + j * g->dx, g->z0 + m * g->dz,
                          s_out + ((size_t)m * g->nx + j) * N);
}

/* signed k-th root: sgn(s) |s|^(1/k)  (reading A3: real odd root, never pow(negative)) */
static double sroot(double s, int k) {
    double a = fabs(s), r;
    if (k == 1) return s;
    if (k == 2) r = sqrt(a);
    else if (k == 3) r = cbrt(a);
    else r = pow(a, 1.0 / (double)k);
    return s < 0.0 ? -r : r;
}

/* ---- O5 route A: the definition.  Sum over all k-subsets i1<...<ik of sgn(prod) |prod|^(1/k),
 * the root taken of the PRODUCT of un-rooted samples, exactly as eqs. (1),(2),(4),(5),(6) print it
 * (PAPER.md:29, :39, :54-60). */
static double brute_rec(const double* s, int n, int k, int start, int depth, double prod) {
    if (depth == k) return sroot(prod, k);
    double acc = 0.0;
    for (int i = start; i <= n - (k - depth); ++i) acc += brute_rec(s, n, k, i + 1, depth + 1, prod * s[i]);
    return acc;
}
double orc_combine_brute(const double* s, int n, int k) {
    if (k < 1 || k > n) return 0.0;
    return brute_rec(s, n, k, 0, 0, 1.0);
}

/* ---- O5 route B: e_k(u), u_i = signed k-th root of s_i, by the textbook recurrence for elementary
 * symmetric sums E[j] += u_i E[j-1].  Equals route A because the k-th root of a product is the product
 * of signed k-th roots.  Exact for any N, no cancellation-prone powers. */
double orc_combine_recur(const double* s, int n, int k) {
    double E[16];
    if (k < 1 || k > 15) return NAN;
    for (int j = 0; j <= k; ++j) E[j] = 0.0;
    E[0] = 1.0;
    for (int i = 0; i < n; ++i) {
        double u = sroot(s[i], k);
        for (int j = k; j >= 1; --j) E[j] += u * E[j - 1];
    }
    return E[k];
}

/* ---- O5 route C: the paper's printed closed forms, eqs. (3), (7), (8) and (9).
 * repaired = 1 applies reading A1 to eq. (9): the term at PAPER.md:79 is 15 (sum u^2)^2 (sum u);
 * repaired = 0 evaluates that line as extracted, 15 (sum u^2)(sum u), kept only to document the repair. */
double orc_combine_closed(const double* s, int n, int k, int repaired) {
    double p1 = 0, p2 = 0, p3 = 0, p4 = 0, p5 = 0;
    for (int i = 0; i < n; ++i) {
        double u = sroot(s[i], k);
        p1 += u; p2 += u * u; p3 += u * u * u; p4 += u * u * u * u; p5 += u * u * u * u * u;
    }
    switch (k) {
    case 1: return p1;                                                            /* eq. (1) */
    case 2: {                                                                     /* eq. (3): second sum is sum |s_i| */
        double sabs = 0; for (int i = 0; i < n; ++i) sabs += fabs(s[i]);
        return (p1 * p1 - sabs) / 2.0;
    }
    case 3: {                                                                     /* eq. (7): 2 sum s_i */
        double ss = 0; for (int i = 0; i < n; ++i) ss += s[i];
        return (p1 * p1 * p1 + 2.0 * ss - 3.0 * p1 * p2) / 6.0;
    }
    case 4: {                                                                     /* eq. (8): sum|s|, sum sqrt|s| */
        double sabs = 0, ssq = 0;
        for (int i = 0; i < n; ++i) { sabs += fabs(s[i]); ssq += sqrt(fabs(s[i])); }
        return (p1 * p1 * p1 * p1 - 6.0 * sabs + 3.0 * ssq * ssq - 6.0 * ssq * p1 * p1 + 8.0 * p3 * p1) / 24.0;
    }
    case 5: {                                                                     /* eq. (9) */
        double ss = 0; for (int i = 0; i < n; ++i) ss += s[i];
        double t79 = repaired ? 15.0 * p2 * p2 * p1 : 15.0 * p2 * p1;
        return (p1 * p1 * p1 * p1 * p1 + 24.0 * ss - 30.0 * p1 * p4 + 20.0 * p3 * p1 * p1 - 20.0 * p3 * p2 + t79
                - 10.0 * p2 * p1 * p1 * p1) / 120.0;
    }
    default: return NAN;
    }
}

/* separately written DAS, eq. (1) PAPER.md:29 (pin P1) */
void orc_das(const void* rf, int dtype, double scale, int F, int N, int S, double fs, double c, double pitch,
             const orc_grid* g, double* out) {
    for (int f = 0; f < F; ++f)
        for (int m = 0; m < g->nz; ++m)
            for (int j = 0; j < g->nx; ++j) {
                double x = g->x0 + j * g->dx, z = g->z0 + m * g->dz, acc = 0.0;
                for (int i = 0; i < N; ++i) {
                    double xe = ((double)i - ((double)N - 1.0) / 2.0) * pitch;
                    double d = sqrt((x - xe) * (x - xe) + z * z);
                    double idx = fs * d / c;
                    double fl = floor(idx);
                    double v = 0.0;
                    if (fl >= 0.0 && fl + 1.0 <= (double)(S - 1)) {
                        size_t o = ((size_t)f * N + i) * (size_t)S + (size_t)fl;
                        v = (1.0 - (idx - fl)) * rf_at(rf, dtype, scale, o) + (idx - fl) * rf_at(rf, dtype, scale, o + 1);
                    }
                    acc += v;
                }
                out[((size_t)f * g->nz + m) * g->nx + j] = acc;
            }
}

/* The reference image: O1-O4 then the chosen route (0 = A brute, 1 = B recurrence, 2 = C closed forms).
 * out[F][nz][nx].  nthreads <= 0: all cores OpenMP gives.  Returns the thread count used. */
int orc_beamform(const void* rf, int dtype, double scale, int F, int N, int S, double fs, double c, double pitch,
                 const orc_grid* g, int order, int route, double* out, int nthreads) {
    int used = 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
    else omp_set_num_threads(omp_get_num_procs());
#pragma omp parallel
    {
#pragma omp single
        used = omp_get_num_threads();
    }
#endif
    for (int f = 0; f < F; ++f) {
#pragma omp parallel for schedule(dynamic, 4)
        for (int m = 0; m < g->nz; ++m) {
            double* s = (double*)malloc(sizeof(double) * (size_t)N);
            for (int j = 0; j < g->nx; ++j) {
                pixel_samples(rf, dtype, scale, f, N, S, fs, c, pitch, g->x0 + j * g->dx, g->z0 + m * g->dz, s);
                double v;
                if (route == 0) v = orc_combine_brute(s, N, order);
                else if (route == 2) v = orc_combine_closed(s, N, order, 1);
                else v = orc_combine_recur(s, N, order);
                out[((size_t)f * g->nz + m) * g->nx + j] = v;
            }
            free(s);
        }
    }
    return used;
}

/* same, on a list of sampled pixels only: pix[2*p] = row m, pix[2*p+1] = column j; out[F][n_pix] */
void orc_beamform_pixels(const void* rf, int dtype, double scale, int F, int N, int S, double fs, double c, double pitch,
                         const orc_grid* g, int order, int route, const int* pix, int n_pix, double* out) {
    double* s = (double*)malloc(sizeof(double) * (size_t)N);
    for (int f = 0; f < F; ++f)
        for (int p = 0; p < n_pix; ++p) {
            int m = pix[2 * p], j = pix[2 * p + 1];
            pixel_samples(rf, dtype, scale, f, N, S, fs, c, pitch, g->x0 + j * g->dx, g->z0 + m * g->dz, s);
            double v;
            if (route == 0) v = orc_combine_brute(s, N, order);
            else if (route == 2) v = orc_combine_closed(s, N, order, 1);
            else v = orc_combine_recur(s, N, order);
            out[(size_t)f * n_pix + p] = v;
        }
    free(s);
}

/* ---------------------------------------------------------------------------------------------------------
 * f4 nearest-sample delays (the literal eq. 1) and f1 coherence-factor weighting.
 * ------------------------------------------------------------------------------------------------------- */

/* f4, reading A21: eq. (1) PAPER.md:29 indexes an integer sample, s_i[k + Delta_i].  Nearest-sample gather:
 * n = floor(idx + 1/2); s_i = rf_i[n] when 0 <= n <= S-1, else 0 (A6). */
static double nearest_chan(const void* rf, int dtype, double scale, size_t chan_off, int S, double idx) {
    double n = floor(idx + 0.5);
    if (!(n >= 0.0) || !(n <= (double)(S - 1))) return 0.0;
    return rf_at(rf, dtype, scale, chan_off + (size_t)n);
}

/* f1, reading A20: PAPER.md:207 ("can be combined with coherence based real-time weighting factors") names no
 * formula; the coherence factor of the beamforming literature is taken:
 *   CF = (sum_i s_i)^2 / (N sum_i s_i^2),  0 when every s_i = 0;  N counts every element (A6: N is not reduced).
 * 0 <= CF <= 1 by Cauchy-Schwarz, CF = 1 iff all s_i are equal. */
double orc_coherence_factor(const double* s, int n) {
    double sum = 0.0, sq = 0.0;
    for (int i = 0; i < n; ++i) { sum += s[i]; sq += s[i] * s[i]; }
    if (!(sq > 0.0)) return 0.0;
    return sum * sum / ((double)n * sq);
}

/* Reference image with the options of rows f1 / f4: interp 0 = linear (O4), 1 = nearest (A21);
 * weight 0 = none, 1 = out = CF * e_k (A20).  Same loops as orc_beamform otherwise.  Returns threads used. */
int orc_beamform_ex(const void* rf, int dtype, double scale, int F, int N, int S, double fs, double c, double pitch,
                    const orc_grid* g, int order, int route, int interp, int weight, double* out, int nthreads) {
    int used = 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
    else omp_set_num_threads(omp_get_num_procs());
#pragma omp parallel
    {
#pragma omp single
        used = omp_get_num_threads();
    }
#endif
    for (int f = 0; f < F; ++f) {
#pragma omp parallel for schedule(dynamic, 4)
        for (int m = 0; m < g->nz; ++m) {
            double* s = (double*)malloc(sizeof(double) * (size_t)N);
            for (int j = 0; j < g->nx; ++j) {
                const double x = g->x0 + j * g->dx, z = g->z0 + m * g->dz;
                for (int i = 0; i < N; ++i) {
                    double idx = orc_delay_idx(x, z, orc_elem_x(i, N, pitch), fs, c);
                    size_t off = ((size_t)f * N + i) * (size_t)S;
                    s[i] = interp == 1 ? nearest_chan(rf, dtype, scale, off, S, idx)
                                       : interp_chan(rf, dtype, scale, off, S, idx);
                }
                double v;
                if (route == 0) v = orc_combine_brute(s, N, order);
                else if (route == 2) v = orc_combine_closed(s, N, order, 1);
                else v = orc_combine_recur(s, N, order);
                if (weight == 1) v *= orc_coherence_factor(s, N);
                out[((size_t)f * g->nz + m) * g->nx + j] = v;
            }
            free(s);
        }
    }
    return used;
}

/* nearest-sample index n[nz][nx][N] as the oracle decides it (-1 when outside the record): test hook for A21 */
void orc_nearest_index(int N, int S, double fs, double c, double pitch, const orc_grid* g, int* n_out) {
    for (int m = 0; m < g->nz; ++m)
        for (int j = 0; j < g->nx; ++j)
            for (int i = 0; i < N; ++i) {
                double idx = orc_delay_idx(g->x0 + j * g->dx, g->z0 + m * g->dz, orc_elem_x(i, N, pitch), fs, c);
                double n = floor(idx + 0.5);
                n_out[((size_t)m * g->nx + j) * N + i] = (n >= 0.0 && n <= (double)(S - 1)) ? (int)n : -1;
            }
}

/* ---------------------------------------------------------------------------------------------------------
 * image-quality metrics, eqs. (10)-(12) and FWHM.
 * The image is the float32 array the beamformer delivers (envelope, linear scale); sums are in double.
 * Readings A22: regions are pixel rectangles rows [r0, r1) x columns [c0, c1); sigma_out is the population
 * standard deviation; gCNR's x is the amplitude divided by the largest amplitude of the two regions, binned into
 * n_bins equal bins on [0, 1] (x = 1 in the last bin), the bin index decided in float32 arithmetic (the image's own
 * precision) so that both implementations take the same integer decision; FWHM is measured on one image row inside
 * the target's columns: width between the two half-maximum crossings next to the row's first maximum, crossings
 * placed by linear interpolation, clipped to the region, in metres (pixels times dx).
 * out[0..6] = mu_in, mu_out, sigma_out, SNR dB (eq. 10), CR dB (eq. 11), gCNR (eq. 12), FWHM m.
 * ------------------------------------------------------------------------------------------------------- */
void orc_image_metrics(const float* img, int nz, int nx, const int* tgt, const int* bkg, int n_bins, int fwhm_row,
                       double dx, double* out) {
    (void)nz;
    double s_in = 0.0, s_out = 0.0;
    float vmax = 0.0f;
    long n_in = 0, n_out = 0;
    for (int r = tgt[0]; r < tgt[1]; ++r)
        for (int c = tgt[2]; c < tgt[3]; ++c) { float v = img[(size_t)r * nx + c]; s_in += v; ++n_in; if (v > vmax) vmax = v; }
    for (int r = bkg[0]; r < bkg[1]; ++r)
        for (int c = bkg[2]; c < bkg[3]; ++c) { float v = img[(size_t)r * nx + c]; s_out += v; ++n_out; if (v > vmax) vmax = v; }
    double mu_in = s_in / (double)n_in, mu_out = s_out / (double)n_out, var = 0.0;
    for (int r = bkg[0]; r < bkg[1]; ++r)
        for (int c = bkg[2]; c < bkg[3]; ++c) { double d = (double)img[(size_t)r * nx + c] - mu_out; var += d * d; }
    double sigma = sqrt(var / (double)n_out);
    /* eq. (12): gCNR = 1 - sum_x min(h_i(x), h_o(x)) */
    double* hi = (double*)calloc((size_t)n_bins, sizeof(double));
    double* ho = (double*)calloc((size_t)n_bins, sizeof(double));
    for (int pass = 0; pass < 2; ++pass) {
        const int* R = pass == 0 ? tgt : bkg;
        double* h = pass == 0 ? hi : ho;
        for (int r = R[0]; r < R[1]; ++r)
            for (int c = R[2]; c < R[3]; ++c) {
                float v = img[(size_t)r * nx + c];
                volatile float q = v / vmax;                    /* float32 division, then float32 product */
                volatile float t = q * (float)n_bins;
                int b = vmax > 0.0f ? (int)floorf(t) : 0;
                if (b < 0) b = 0;
                if (b > n_bins - 1) b = n_bins - 1;
                h[b] += 1.0;
            }
    }
    double ovl = 0.0;
    for (int b = 0; b < n_bins; ++b) {
        double a = hi[b] / (double)n_in, o = ho[b] / (double)n_out;
        ovl += a < o ? a : o;
    }
    free(hi); free(ho);
    /* FWHM on row fwhm_row, columns [c0, c1) of the target */
    double fwhm = NAN;
    if (fwhm_row >= 0) {
        const float* p = img + (size_t)fwhm_row * nx;
        int c0 = tgt[2], c1 = tgt[3], pk = c0;
        for (int c = c0; c < c1; ++c) if (p[c] > p[pk]) pk = c;
        double half = 0.5 * (double)p[pk], left = (double)c0, right = (double)(c1 - 1);
        for (int c = pk; c > c0; --c)
            if ((double)p[c - 1] < half) { left = (double)(c - 1) + (half - (double)p[c - 1]) / ((double)p[c] - (double)p[c - 1]); break; }
        for (int c = pk; c < c1 - 1; ++c)
            if ((double)p[c + 1] < half) { right = (double)c + ((double)p[c] - half) / ((double)p[c] - (double)p[c + 1]); break; }
        fwhm = (right - left) * dx;
    }
    out[0] = mu_in; out[1] = mu_out; out[2] = sigma;
    out[3] = 20.0 * log10(mu_in / sigma);        /* eq. (10) */
    out[4] = 20.0 * log10(mu_in / mu_out);       /* eq. (11) */
    out[5] = 1.0 - ovl;                          /* eq. (12) */
    out[6] = fwhm;
}

/* ---------------------------------------------------------------------------------------------------------
 * Post chain ("a bandpass filter was applied at the appropriate frequency range. Envelope
 * detection using Hilbert transformation and log compression were applied"; readings A8-A12).
 * ------------------------------------------------------------------------------------------------------- */
static double sinc_pi(double x) { return x == 0.0 ? 1.0 : sin(M_PI * x) / (M_PI * x); }

/* O6 taps: Hamming-windowed ideal band-pass, T taps, band [f_lo, f_hi] in cycles per row (A8). */
void orc_bandpass_taps(int T, double f_lo, double f_hi, double* h) {
    for (int t = 0; t < T; ++t) {
        double m = (double)t - ((double)T - 1.0) / 2.0;
        double w = 0.54 - 0.46 * cos(2.0 * M_PI * (double)t / ((double)T - 1.0));
        h[t] = w * (2.0 * f_hi * sinc_pi(2.0 * f_hi * m) - 2.0 * f_lo * sinc_pi(2.0 * f_lo * m));
    }
}

/* O7 taps: type-III Hilbert FIR, g[t] = 2/(pi t) for odd t, 0 for even t, t = -L..L, Hamming window (A9).
 * g_out[t + L]. */
void orc_hilbert_taps(int L, double* g_out) {
    for (int t = -L; t <= L; ++t) {
        double w = 0.54 + 0.46 * cos(M_PI * (double)t / (double)L);
        g_out[t + L] = (t % 2 != 0) ? w * 2.0 / (M_PI * (double)t) : 0.0;
    }
}

/* O6: y[m] = sum_{t=0}^{T-1} h[t] x[m + T/2 - t], x = 0 outside [0, nz), per column, per frame (A11, A12). */
void orc_fir_axial(const double* x, int F, int nz, int nx, const double* h, int T, double* y) {
    for (int f = 0; f < F; ++f)
        for (int m = 0; m < nz; ++m)
            for (int j = 0; j < nx; ++j) {
                double acc = 0.0;
                for (int t = 0; t < T; ++t) {
                    int r = m + T / 2 - t;
                    if (r >= 0 && r < nz) acc += h[t] * x[((size_t)f * nz + r) * nx + j];
                }
                y[((size_t)f * nz + m) * nx + j] = acc;
            }
}

/* O7: q[m] = sum_{t=-L}^{L} g[t] y[m - t]; env = sqrt(y^2 + q^2) */
void orc_envelope(const double* y, int F, int nz, int nx, const double* g, int L, double* env) {
    for (int f = 0; f < F; ++f)
        for (int m = 0; m < nz; ++m)
            for (int j = 0; j < nx; ++j) {
                double q = 0.0;
                for (int t = -L; t <= L; ++t) {
                    int r = m - t;
                    if (r >= 0 && r < nz) q += g[t + L] * y[((size_t)f * nz + r) * nx + j];
                }
                double v = y[((size_t)f * nz + m) * nx + j];
                env[((size_t)f * nz + m) * nx + j] = sqrt(v * v + q * q);
            }
}

/* O8: out = max(20 log10(env / M), -DR), M = per-frame max of env; env = 0 or M = 0 gives -DR (A10). */
void orc_logcompress(const double* env, int F, int nz, int nx, double dyn_range_db, double* out) {
    size_t n = (size_t)nz * nx;
    for (int f = 0; f < F; ++f) {
        const double* e = env + (size_t)f * n;
        double M = 0.0;
        for (size_t p = 0; p < n; ++p) if (e[p] > M) M = e[p];
        for (size_t p = 0; p < n; ++p) {
            double v = -dyn_range_db;
            if (M > 0.0 && e[p] > 0.0) {
                v = 20.0 * log10(e[p] / M);
                if (v < -dyn_range_db) v = -dyn_range_db;
            }
            out[(size_t)f * n + p] = v;
        }
    }
}
