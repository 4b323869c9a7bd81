/*
 * pab.h -- C ABI of libpab.so: linear-array photoacoustic image reconstruction by order-k
 * delay-multiply-and-sum (DMAS-k, k = 1..5) beamforming in its O(N)-per-pixel form, for one
 * NVIDIA B200 (sm_100a).  Method: arXiv 2203.14906, "Higher-order correlation based real-time
 * beamforming in photoacoustic imaging".  Citations are PAPER.md:<line> (the paper's text) and
 * DESIGN.md reading numbers A1..A19.
 *
 * What the library computes, per pixel (x_j, z_m) and frame:
 *   delay      idx_i = fs * sqrt((x_j - xe_i)^2 + z_m^2) / c            (eq. 1's Delta_i; A5)
 *   sample     s_i   = (1-a) rf_i[i0] + a rf_i[i0+1], i0 = floor(idx_i), a = idx_i - i0,
 *                      0 when i0 < 0 or i0+1 > n_samp-1                 (eq. 1; A4, A6)
 *   root       u_i   = sgn(s_i) |s_i|^(1/k)                             (A3)
 *   power sums p_m   = sum_i u_i^m, m = 1..k   (p_k = sum s_i or sum |s_i|)
 *   output     e_k(u_1..u_N) from p_1..p_k by Newton's identities       (eqs. 1, 3, 7, 8, 9: PAPER.md:29, :45,
 *                                                                        :66, :69, :71-82 with repair A1)
 *   optional   axial band-pass FIR -> Hilbert-FIR envelope -> log compression   (A8-A12)
 *
 * All pointers named *_dev are CUDA device pointers, *_host are host pointers.  No torch types, no
 * exceptions, no global state.  Every function returns PAB_OK (0) or a negative error code; on an argument
 * error nothing is written and nothing is launched.  There is no CPU fallback: without a usable sm_100
 * device pab_create fails with PAB_ERR_DEVICE.
 */
#ifndef PAB_H_
#define PAB_H_

#ifdef __cplusplus
extern "C" {
#endif

#define PAB_OK            0
#define PAB_ERR_INVALID  (-1)   /* null pointer, non-positive size, order outside 1..8, misaligned pointer        */
#define PAB_MAX_ORDER 8
#define PAB_ERR_DEVICE   (-2)   /* no CUDA device, or the current device is not compute capability 10.x           */
#define PAB_ERR_ALLOC    (-3)   /* device or pinned-host allocation failed                                        */
#define PAB_ERR_CUDA     (-4)   /* a CUDA call or kernel launch failed (see pab_last_cuda_error)                  */
#define PAB_ERR_LIMIT    (-5)   /* a size beyond the fixed maximum of a no-allocation entry point (pab_post_no_alloc) */

/* input sample type (pab_set_input) */
#define PAB_F32 0
#define PAB_I16 1

/* post-processing mode (pab_set_post): what `out` holds */
#define PAB_RAW      0   /* the beamformed image e_k (pre-band-pass); default                                     */
#define PAB_BANDPASS 1   /* after the axial band-pass FIR                                                         */
#define PAB_ENVELOPE 2   /* after band-pass and Hilbert-FIR envelope                                              */
#define PAB_LOG      3   /* after band-pass, envelope and log compression, dB <= 0                                */

/* delay handling (pab_set_interp) */
#define PAB_INTERP_LINEAR  0   /* s_i = linear interpolation at the fractional delay index (A4); default           */
#define PAB_INTERP_NEAREST 1   /* s_i = rf_i[floor(idx_i + 1/2)]: the literal integer-delay eq. (1) (A21)           */

/* cached interpolation taps (pab_set_delay_cache) */
#define PAB_CACHE_OFF    0   /* delays computed in-kernel on every call; default                                   */
#define PAB_CACHE_SINGLE 1   /* calls of 1..3 frames read their taps from the cached table                         */
#define PAB_CACHE_ALL    2   /* ... and so do the frame groups of longer calls                                      */

/* pixel weighting (pab_set_weight) */
#define PAB_WEIGHT_NONE 0   /* out = e_k                                                                          */
#define PAB_WEIGHT_CF   1   /* out = CF e_k, CF = (sum_i s_i)^2 / (N sum_i s_i^2), 0 when every s_i = 0             */

/* beamforming kernel variant (pab_set_variant) */
#define PAB_VARIANT_AUTO   0   /* staged when its shared-memory plan fits, else direct                            */
#define PAB_VARIANT_DIRECT 1   /* per-thread gathers through L1/L2 from the staged RF copy, no shared memory      */
#define PAB_VARIANT_STAGED 2   /* per-tile RF windows bulk-copied (TMA 1-D) into shared memory, mbarrier pipeline */

typedef struct pab_ctx pab_ctx;     /* opaque; created by pab_create, owned by the library, freed by pab_destroy  */

/* Pixel grid (A5).  Pixel (m, j), row m in depth and column j laterally, has its centre at
 * (x, z) = (x0 + j*dx, z0 + m*dz), metres.  The array lies on z = 0, centred on x = 0. */
typedef struct {
    int   nx, nz;            /* columns (lateral), rows (depth); both >= 1                                        */
    float x0, dx, z0, dz;    /* metres; dx > 0, dz > 0, z0 >= 0                                                    */
} pab_grid;

/* The plan the library derives from a geometry (host logic only; see pab_plan). */
typedef struct {
    int   tile_z, tile_x;        /* pixel tile of one thread block of the staged kernel (rows, columns)            */
    int   window_samples;        /* upper bound of the per-channel RF window a tile needs, samples (mult. of 4)    */
    int   chunk_channels;        /* channels staged per pipeline stage                                             */
    int   stages;                /* pipeline depth                                                                 */
    int   smem_bytes;            /* dynamic shared memory per block, bytes; 0 when the staged kernel does not fit  */
    int   frames_per_thread;     /* frames each thread carries in registers when enough frames are given (4, 8, 16)*/
    int   batch_frames;          /* internal frame batch per pass (ingest -> beamform -> post)                     */
    int   in_range;              /* 1 when every (pixel, element) delay index lies inside the record and z0 is at
                                    least one sample deep: the kernels then skip the out-of-record masks (A6)     */
    int   diagonal;              /* single-frame diagonal kernel (translation-invariant geometry: pitch an exact integer
                                    multiple q <= 16 of dx, in range): 1 once pab_set_delay_cache (or pab_set_interp, for the
                                    nearest-sample path) has built its tap tables;
                                    2 once a call of 1..3 frames with the delay cache off has built the windows of its
                                    table-free form (taps computed in the kernel); else 0                             */
    double zs_per_row;           /* dz * fs / c : delay samples per pixel row                                      */
    double xs_per_col;           /* dx * fs / c : delay samples per pixel column at grazing incidence              */
} pab_plan_info;

/*
 * pab_create -- build a context for one array + grid (N-element linear array,
 * pitch, sampling frequency fs, speed of sound c; one-way time of flight, record starts at t = 0: A5).
 *   out       receives the handle (host pointer, written only on success)
 *   n_elem    N >= 1, element i at x = (i - (N-1)/2) * pitch_m, z = 0
 *   n_samp    S >= 2 samples per channel per frame
 *   fs_hz, c_m_s, pitch_m   > 0
 *   grid      host pointer, copied
 * Uploads the per-row / per-column / per-element delay tables (computed in fp64 on the host, stored as
 * fp32 hi+lo pairs in sample units) and allocates scratch.  Uses the CUDA device current at the call.
 * Errors: PAB_ERR_INVALID, PAB_ERR_DEVICE, PAB_ERR_ALLOC, PAB_ERR_CUDA.
 */
int pab_create(pab_ctx** out, int n_elem, int n_samp, float fs_hz, float c_m_s, float pitch_m,
               const pab_grid* grid);

/* pab_set_input -- RF sample type and scale: sample value = scale * stored value (A15).  Default PAB_F32, 1.0.
 * int16 ADC counts are converted to fp32 exactly while the frames are staged (BASELINE.json config C5). */
int pab_set_input(pab_ctx* ctx, int dtype, float scale);

/*
 * pab_set_post -- post chain after the combination (A8-A13).  Default PAB_RAW.
 *   mode             PAB_RAW | PAB_BANDPASS | PAB_ENVELOPE | PAB_LOG
 *   f_center_hz, f_halfwidth_hz   pass band [f_c - f_hw, f_c + f_hw] of the Hamming-windowed-sinc band-pass, in Hz
 *                    of the axial sampling rate fs_z = c / dz (one row per c/dz seconds of one-way flight)
 *   n_taps_bp        T, 2..256:  y[m] = sum_{t<T} h[t] x[m + T/2 - t], x = 0 outside the image (A12)
 *   n_taps_hilbert   2L+1, odd, 3..255: q[m] = sum_{|t|<=L} g[t] y[m-t], g[t] = 2/(pi t) * Hamming for odd t, 0 for
 *                    even t; env = sqrt(y^2 + q^2) (A9)
 *   dyn_range_db     DR > 0: out = max(20 log10(env / max_frame env), -DR); env = 0 or max = 0 gives -DR (A10)
 */
int pab_set_post(pab_ctx* ctx, int mode, float f_center_hz, float f_halfwidth_hz, int n_taps_bp,
                 int n_taps_hilbert, float dyn_range_db);

/* pab_set_weight -- coherence-factor weighting fused into the beamforming kernel ("can be combined
 * with coherence based real-time weighting factors"; the paper gives no formula: DESIGN.md reading A20 takes the
 * standard coherence factor over all N elements, out-of-record samples counting as zeros).  Default PAB_WEIGHT_NONE.
 * With PAB_WEIGHT_CF a thread carries at most 8 frames (orders 1-3) or 4 frames (orders 4, 5). */
int pab_set_weight(pab_ctx* ctx, int weight);

/* pab_set_interp -- PAB_INTERP_NEAREST switches to the paper's literal eq. (1) (s_i[k + Delta_i] with an
 * integer delay; reading A21): the delayed sample is the nearest RF sample, 0 outside the record.  The
 * signed k-th root is then taken once per RF sample while the frames are staged and the integer delays come from a
 * delay table in device memory (the paper's own arrangement), built here in fp64 with the oracle's
 * expression: n_elem * nx * nz uint16 entries.  On translation-invariant in-range geometries (pitch_m an exact integer
 * multiple q <= 16 of grid.dx, n_elem a multiple of 4) calls of 1..3 frames instead run the single-frame diagonal kernel on a
 * compact table of the same fp64 decisions, one per (column - q * element, row), roots taken per item.  Synchronises the
 * device on the first call.
 * Errors: PAB_ERR_INVALID (n_samp > 65534, or combined with PAB_WEIGHT_CF), PAB_ERR_ALLOC, PAB_ERR_CUDA. */
int pab_set_interp(pab_ctx* ctx, int interp);

/* pab_set_delay_cache -- keep the interpolation tap (integer sample + fraction) of every (pixel, element) pair in
 * device memory, computed once in fp64, instead of recomputing the delay in every call (PAPER.md:190 keeps its
 * delays in GPU global memory; BASELINE.json north_star allows a cached table "where it wins").  It wins most for
 * calls of 1..3 frames on geometries that are not translation invariant, where the in-kernel delay cannot be shared
 * between frames or pairs, and by ~7 % for 16-frame groups.
 * 4 bytes per (pixel, element): 134 MB at 128 elements x 1024 x 256 pixels; when pitch_m is an exact integer
 * multiple q of grid.dx the tap depends on (column - q * element, row) only, and calls of 1..3 frames use a compact
 * table of (nx + q (N-1)) * nz * 8 bytes (2 MB there) instead.  Linear interpolation; coherence-factor weighting
 * (8- and 4-frame groups) and orders 6..8 (4-frame groups) read the table under PAB_CACHE_ALL only (other
 * settings, and geometries whose table block does not fit in shared memory, fall back to the in-kernel delay).
 * In-range geometries only (pab_plan_info.in_range), staged variant.
 * Synchronises the device on the first call.  Errors: PAB_ERR_INVALID, PAB_ERR_ALLOC, PAB_ERR_CUDA. */
int pab_set_delay_cache(pab_ctx* ctx, int mode);

/* pab_set_tuning -- override the plan's blocking (autotuning / experiments); 0 keeps the default of a field.
 *   frames_per_thread 4, 8 or 16;  stages 2..4;  chunk_channels 1..32 (clamped to what fits in shared memory);
 *   host_batch_frames 1..64: frames per piece of pab_beamform_host's copy / compute / copy pipeline.
 * Recomputes the plan (pab_get_plan shows the result).  Synchronises the device.  PAB_ERR_INVALID on bad values. */
int pab_set_tuning(pab_ctx* ctx, int frames_per_thread, int stages, int chunk_channels, int host_batch_frames);

/* pab_set_variant -- force a beamforming kernel variant (testing / benchmarking).  PAB_ERR_INVALID when the
 * staged variant is requested but its plan does not fit in shared memory. */
int pab_set_variant(pab_ctx* ctx, int variant);

/*
 * pab_beamform -- enqueue the whole hot path for n_frames frames on `cuda_stream` and return (never
 * synchronises).
 *   rf_dev     device pointer, [n_frames][n_elem][n_samp], sample index fastest, fp32 or int16 per
 *              pab_set_input; aligned to its element size; read only; caller keeps it alive until the
 *              stream work finishes
 *   n_frames   >= 1; frames are independent; the library batches them internally
 *   order      k = 1..5 (1 = DAS eq. 1, 2 = DMAS eq. 3, 3..5 = eqs. 7, 8, 9); k = 6..8 (row f2: the same
 *              O(N) evaluation of e_k, by its recurrence) with linear interpolation and no weighting only
 *   out_dev    device pointer, [n_frames][nz][nx], x fastest, fp32, 4-byte aligned; fully overwritten
 *   cuda_stream a cudaStream_t passed as void*; NULL = the legacy default stream
 * Exceptions (one device synchronisation each, once per context; skipped while the stream is being captured): under
 * PAB_CACHE_ALL the first call of order 1 or 2 with >= 8 frames, at a row pitch in (1, 8/7] samples, builds a second tap
 * table; with the delay cache off and the automatic variant, the first call of 1..3 frames on a translation-invariant
 * in-range geometry (pitch_m an exact integer multiple q <= 16 of grid.dx, n_elem a multiple of 4) builds the windows of
 * the single-frame diagonal kernel (a few hundred KB; no delay table: that kernel computes one delay per diagonal of
 * (column, element) pairs in the kernel, on the FP64 pipe, and is what such calls then run: pab_plan_info.diagonal = 2).
 * One context must not be used from two streams at once (shared scratch).  The CUDA device that was current at
 * pab_create must be current at the call (PAB_ERR_INVALID otherwise).
 * Errors: PAB_ERR_INVALID (nothing launched), PAB_ERR_CUDA.
 */
int pab_beamform(pab_ctx* ctx, const void* rf_dev, int n_frames, int order, float* out_dev, void* cuda_stream);

/*
 * pab_beamform_host -- the same path from HOST buffers: copies rf_host to the device in pieces of a few frames,
 * runs the kernels and copies the images back on three internal streams with two device buffer sets, so that the
 * copies of successive pieces overlap the kernels; returns after everything has finished.  Pinned host memory
 * is what makes the copies asynchronous; pageable buffers work but serialise.
 *   rf_host   host pointer, same layout and type as rf_dev above (pageable or pinned)
 *   out_host  host pointer, [n_frames][nz][nx] fp32
 */
int pab_beamform_host(pab_ctx* ctx, const void* rf_host, int n_frames, int order, float* out_host);

/*
 * pab_beamform_host_async / pab_host_sync -- the streaming form of pab_beamform_host: enqueues the copies and kernels of
 * the call on the context's internal streams and returns; pab_host_sync waits for everything enqueued so far.
 * Successive calls overlap one another (host-to-device copy of call i + 1, kernels of call i and device-to-host copy of
 * call i - 1 run side by side on two device buffer sets), so a stream of 64-frame batches runs at the rate of its slowest
 * leg -- at C2b the host-to-device copy -- where the blocking call pays its own ramp-up and drain every time.
 *   rf_host, out_host   as for pab_beamform_host, but PINNED (cudaHostAlloc / cudaHostRegister) for the copies to be
 *                       asynchronous, and kept alive and unmodified (rf) / unread (out) until pab_host_sync returns
 * Between the first call and pab_host_sync the context's settings must not change and pab_beamform must not be called on
 * it (shared scratch).  Errors: as pab_beamform_host; an error of the asynchronous work surfaces at pab_host_sync.
 */
int pab_beamform_host_async(pab_ctx* ctx, const void* rf_host, int n_frames, int order, float* out_host);
int pab_host_sync(pab_ctx* ctx);

/* pab_destroy -- free the context and everything it owns.  NULL is a no-op.  Synchronises the device. */
void pab_destroy(pab_ctx* ctx);

/* pab_plan -- host-only: the tiling / staging plan for a geometry (no GPU needed; pab_create uses the
 * same routine).  smem_limit_bytes <= 0 means the sm_100 opt-in limit (232448).  Returns PAB_ERR_INVALID
 * on bad arguments. */
int pab_plan(int n_elem, int n_samp, float fs_hz, float c_m_s, float pitch_m, const pab_grid* grid,
             int smem_limit_bytes, pab_plan_info* plan_out);

/* pab_get_plan -- the plan a context is using. */
int pab_get_plan(const pab_ctx* ctx, pab_plan_info* plan_out);

/* pab_design_bandpass / pab_design_hilbert -- host-only: the FIR taps pab_set_post uploads (fp64 design,
 * rounded to fp32).  h_host[T]; g_host[2L+1] with g_host[t + L] = g[t].  f_lo, f_hi in cycles per row. */
int pab_design_bandpass(int n_taps, double f_lo, double f_hi, float* h_host);
int pab_design_hilbert(int half_len, float* g_host);

/* pab_launch_count -- number of kernels this context has launched since it was created. */
long long pab_launch_count(const pab_ctx* ctx);

/* pipeline stages, for pab_get_profile */
#define PAB_STAGE_INGEST   0   /* a1: int16/fp32 -> staged frame-interleaved fp32                                 */
#define PAB_STAGE_BEAMFORM 1   /* a2..a6, a10: the fused delay + interpolate + power-sum + combination kernel     */
#define PAB_STAGE_POST_FIR 2   /* a7, a8: axial band-pass + Hilbert-FIR envelope + per-frame max                  */
#define PAB_STAGE_POST_LOG 3   /* a9: log compression                                                             */
#define PAB_STAGE_COUNT    4

/*
 * pab_set_profile -- per-launch device timing for measurement: when max_launches > 0
 * every kernel the context launches is bracketed by a pair of CUDA events recorded on the launching stream, up
 * to max_launches launches (later ones are counted by pab_launch_count but not timed); 0 switches it off.
 * Synchronises the device.  pab_get_profile sums the event durations of one stage since the last reset
 * (waits for those launches to finish), returns the sum in milliseconds and the number of timed launches, and
 * with reset != 0 forgets every recorded launch of every stage (read all stages first, reset on the last).
 */
int pab_set_profile(pab_ctx* ctx, int max_launches);
int pab_get_profile(pab_ctx* ctx, int stage, double* total_ms, long long* n_launches, int reset);

/* pab_self_check -- diagnostic for the single-frame diagonal kernel (fp32 input; with the delay cache on: the form with its
 * tap table, pab_plan_info.diagonal == 1; with it off and the automatic variant: the table-free form, == 2; under
 * PAB_INTERP_NEAREST: the form on its table of integer delays): runs one
 * frame through an instantiation that compares every shared-memory gather of its element loop with the staged window of
 * the channel quad it reads from, and returns the number of out-of-window accesses (0 for a correct build).  Stands in
 * for compute-sanitizer's memcheck, which is closed on the GPU pool this library was developed on.  order 1..5 selects
 * the table set (orders 1..3 / 4, 5).  Synchronises the device.  Errors: PAB_ERR_INVALID (no diagonal tables, int16
 * input), PAB_ERR_ALLOC, PAB_ERR_CUDA. */
int pab_self_check(pab_ctx* ctx, const float* rf_dev, int order, long long* violations);

/* pab_measure_peaks -- the microbenchmarks behind the roofline denominators, run on the
 * current device: out_host[0] MUFU (lg2/ex2) lanes per clock per SM, [1] FFMA lanes/clk/SM, [2] packed FFMA2 fp32
 * results/clk/SM, [3] conflict-free LDS.128 bytes/clk/SM (each timed with clock64 inside one 1024-thread CTA per
 * SM), [4] pinned host->device and [5] device->host GB/s of a 64 MiB cudaMemcpyAsync, [6] the SM clock seen during
 * the MUFU loop in MHz, [7] the SM count.  n_out >= 8.  Synchronises the device.  Measurement only: nothing on the
 * hot path calls it.  Errors: PAB_ERR_INVALID, PAB_ERR_DEVICE, PAB_ERR_ALLOC, PAB_ERR_CUDA. */
int pab_measure_peaks(double* out_host, int n_out);

/* Image-quality metrics of the paper's evaluation (SNR eq. 10, CR eq. 11, gCNR eq. 12, FWHM),
 * SURVEY.md section 8(f) row f3, reading A22.  Regions are pixel rectangles. */
typedef struct { int r0, r1, c0, c1; } pab_roi;          /* rows [r0, r1), columns [c0, c1), non-empty, inside the grid */
typedef struct {
    double mu_in, mu_out, sigma_out;                     /* means of the two regions, population std of the background */
    double snr_db;                                       /* 20 log10(mu_in / sigma_out)                       eq. (10) */
    double cr_db;                                        /* 20 log10(mu_in / mu_out)                          eq. (11) */
    double gcnr;                                         /* 1 - sum_bins min(h_in, h_out), amplitudes / max   eq. (12) */
    double fwhm_m;                                       /* half-maximum width on row fwhm_row, metres; NaN if row < 0 */
} pab_metrics;

/*
 * pab_image_metrics -- the metrics of one image on the device.
 *   img_dev    device pointer, [nz][nx] float32 (one frame of the context's grid; non-negative amplitudes, e.g. a
 *              PAB_ENVELOPE output)
 *   target, background   host pointers
 *   n_bins     histogram bins of gCNR, 2..4096
 *   fwhm_row   image row on which FWHM is measured inside the target's columns, or -1
 *   out_host   host pointer, written on success
 * Enqueues on cuda_stream and waits for it (the result goes to the host).  Errors: PAB_ERR_INVALID, PAB_ERR_CUDA.
 */
int pab_image_metrics(pab_ctx* ctx, const float* img_dev, const pab_roi* target, const pab_roi* background, int n_bins,
                      int fwhm_row, pab_metrics* out_host, void* cuda_stream);

/*
 * pab_post_no_alloc -- the post chain of the context (a7..a9: band-pass, Hilbert envelope, and under PAB_LOG the log
 * compression) on images the caller already holds, for callers that must not allocate (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Calls no cudaMalloc / cudaFree and no
 * allocating library routine: the only scratch of the chain, the per-frame envelope maxima, lives in a fixed
 * file-scope device array of PAB_NO_ALLOC_MAX_FRAMES entries (4 KiB, held by every GPU that loads the library until the
 * process exits).  Enqueues one memset and the kernels on `cuda_stream`; never synchronises.
 *   img_dev   device pointer, [n_frames][nz][nx] fp32 beamformed images (what pab_beamform writes under PAB_RAW); read only
 *   n_frames  1..PAB_NO_ALLOC_MAX_FRAMES; more is rejected with PAB_ERR_LIMIT (nothing launched; the message of
 *             pab_last_cuda_error names the limit)
 *   out_dev   device pointer, [n_frames][nz][nx] fp32, caller-owned, must not overlap img_dev; holds what pab_beamform
 *             would have written under the context's post mode
 * The context must be in PAB_ENVELOPE or PAB_LOG mode with filters of 33..64 taps each (after padding to 8).
 * All calls on one GPU share the array, which keeps the last call's values (the entry point clears what it uses on its
 * stream first): calls that overlap on the GPU -- two streams, two contexts, two threads -- race on it.
 * Errors: PAB_ERR_INVALID (null / misaligned / overlapping pointers, mode or filter length not covered, wrong current
 * device), PAB_ERR_LIMIT, PAB_ERR_CUDA.
 */
#define PAB_NO_ALLOC_MAX_FRAMES 1024
int pab_post_no_alloc(pab_ctx* ctx, const float* img_dev, int n_frames, float* out_dev, void* cuda_stream);

/* pab_strerror -- static string for an error code.  pab_last_cuda_error -- the last cudaError_t string seen
 * by this context ("" if none). */
const char* pab_strerror(int code);
const char* pab_last_cuda_error(const pab_ctx* ctx);

/* pab_version -- "pab <major>.<minor> sm_100a". */
const char* pab_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PAB_H_ */
