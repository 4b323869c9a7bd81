// pab_api.cu -- the C ABI of libpab.so (include/pab.h): context, host logic, kernel launches.
#include <cstdio>
#include <cstdlib>
#include <cmath>
#include <cstring>
#include <new>
#include <type_traits>
#include <vector>
#include <cuda_runtime.h>
#include "../../include/pab.h"
#include "pab_plan.h"
#include "pab_types.h"
#include "pab_launch.h"

using namespace pab;

// device buffer sets of the host path (pab_beamform_host*): with three, a whole-batch piece can be copied in, computed and
// copied out at the same time without one leg waiting for the hand-over of the set two pieces back
constexpr int kHostSets = 3;

struct pab_ctx {
    int N = 0, S = 0, Sp = 0;
    float fs = 0, c = 0, pitch = 0;
    pab_grid grid{};
    int dtype = PAB_F32;
    float scale = 1.0f;
    int post_mode = PAB_RAW;
    int n_taps_bp = 0, n_taps_h = 0, TpB = 0, TpH = 0;
    float dyn_range_db = 60.0f;
    PostTaps64 taps64{};             // fast post path (<= 64 taps): taps travel in the kernel parameters
    bool post_fast = false;
    int hilbert_parity = 2;          // 0 / 1: only Hilbert taps of that index parity are non-zero; 2: dense
    int variant = PAB_VARIANT_AUTO;
    int weight = PAB_WEIGHT_NONE;
    int interp = PAB_INTERP_LINEAR;
    int cache_mode = PAB_CACHE_OFF;
    uint32_t* d_taps = nullptr;          // cached interpolation taps, tile-major (pab_set_delay_cache)
    int* d_w0s = nullptr;                // window start of every (tile, element)
    uint32_t* d_taps7 = nullptr;         // the same tables for 56-row tiles (order 1 at row pitches in (1, 8/7] samples)
    int* d_w0s7 = nullptr;
    bool taps7_tried = false;
    uint2* d_compact = nullptr;          // (d, row) tap table when pitch = q dx exactly (translation invariance)
    int cache_q = 0;
    DiagSet diag[2];                     // single-frame diagonal kernel: [0] orders 1..3 (16 pixels per thread), [1] orders 4, 5 (8)
    DiagSet diag_nt[2];                  // the same for the table-free variant (delay cache off): windows only, taps in-kernel
    bool diag_nt_tried = false;
    DiagSet diag_near[2];                // the same kernel for the nearest-sample path (row f4): tables of floor(idx + 1/2), fraction 0
    void* d_metric = nullptr;            // MetricAcc + double[1] + 2 x 4096 histogram bins (row f3), lazy
    unsigned short* d_near = nullptr;    // nearest-sample index table [N][nx][nz] (row f4), built by pab_set_interp
    pab_plan_info plan{};
    PlanTuning tuning{};
    int device = 0, sm_count = 0, smem_optin = 0;
    // device tables
    float2* d_xj = nullptr;
    float2* d_xe = nullptr;
    float4* d_zrow = nullptr;
    float* d_stage = nullptr;        // staged RF of one batch (quad or lin layout)
    size_t stage_bytes = 0;
    float* d_img = nullptr;          // beamformed image of one batch when a post chain is on
    float* d_taps_bp = nullptr;
    float* d_taps_h = nullptr;
    unsigned int* d_max = nullptr;   // [batch] per-frame max of the envelope
    // host-buffer path (lazy)
    void* d_in[kHostSets] = {};
    float* d_out[kHostSets] = {};
    cudaStream_t s_h2d = nullptr, s_run = nullptr, s_d2h = nullptr;
    cudaEvent_t ev_in[kHostSets] = {}, ev_run[kHostSets] = {}, ev_out[kHostSets] = {};
    long long launches = 0;
    long long host_it = 0;               // pieces the host path has enqueued so far (buffer set = host_it & 1)
    // per-launch device timing (pab_set_profile): events 2*slot, 2*slot+1 bracket launch `slot`
    bool profiling = false;
    std::vector<cudaEvent_t> prof_ev;
    std::vector<int> prof_stage;
    int prof_used = 0;
    char err[256] = {0};
};

namespace {

int cuda_fail(pab_ctx* ctx, cudaError_t e, const char* what) {
    if (ctx) snprintf(ctx->err, sizeof ctx->err, "%s: %s", what, cudaGetErrorString(e));
    return e == cudaErrorMemoryAllocation ? PAB_ERR_ALLOC : PAB_ERR_CUDA;
}

#define PAB_CUDA(ctx, call)                                          \
    do {                                                             \
        cudaError_t e_ = (call);                                     \
        if (e_ != cudaSuccess) return cuda_fail((ctx), e_, #call);   \
    } while (0)

size_t elem_size(int dtype) { return dtype == PAB_I16 ? 2 : 4; }

void free_all(pab_ctx* ctx) {
    cudaFree(ctx->d_xj); cudaFree(ctx->d_xe); cudaFree(ctx->d_zrow); cudaFree(ctx->d_stage); cudaFree(ctx->d_img);
    cudaFree(ctx->d_taps_bp); cudaFree(ctx->d_taps_h); cudaFree(ctx->d_max); cudaFree(ctx->d_near); cudaFree(ctx->d_metric); cudaFree(ctx->d_taps); cudaFree(ctx->d_w0s); cudaFree(ctx->d_compact); cudaFree(ctx->d_taps7); cudaFree(ctx->d_w0s7);
    xl_diag_free(&ctx->diag[0]); xl_diag_free(&ctx->diag[1]);
    xl_diag_free(&ctx->diag_nt[0]); xl_diag_free(&ctx->diag_nt[1]);
    xl_diag_free(&ctx->diag_near[0]); xl_diag_free(&ctx->diag_near[1]);
    for (int b = 0; b < kHostSets; ++b) {
        cudaFree(ctx->d_in[b]); cudaFree(ctx->d_out[b]);
        if (ctx->ev_in[b]) cudaEventDestroy(ctx->ev_in[b]);
        if (ctx->ev_run[b]) cudaEventDestroy(ctx->ev_run[b]);
        if (ctx->ev_out[b]) cudaEventDestroy(ctx->ev_out[b]);
    }
    for (cudaEvent_t e : ctx->prof_ev) cudaEventDestroy(e);
    ctx->prof_ev.clear();
    if (ctx->s_h2d) cudaStreamDestroy(ctx->s_h2d);
    if (ctx->s_run) cudaStreamDestroy(ctx->s_run);
    if (ctx->s_d2h) cudaStreamDestroy(ctx->s_d2h);
}

// Calls of 1..3 frames with the delay cache OFF on translation-invariant, in-range geometries (pitch = q dx exactly, q <= 16):
// the diagonal kernel in its table-free form (pab_diag.cuh, TAB = false: one tap per diagonal from delay_tap_f64, shared by
// the 16 or 8 pairs of the diagonal).  It needs no delay table, only the window of every (tile, channel quad), a few
// hundred KB built on the first such call (one device synchronisation, skipped while the stream is being captured).
// Returns whether the set of this order is there.
// pab_plan_info.diagonal: which form of the single-frame diagonal kernel the context's current settings would run
void refresh_diagonal_flag(pab_ctx* ctx) {
    auto has = [](const DiagSet (&d)[2]) { return d[0].smem_bytes > 0 || d[1].smem_bytes > 0; };
    if (ctx->interp == PAB_INTERP_NEAREST) ctx->plan.diagonal = has(ctx->diag_near) ? 1 : 0;
    else if (ctx->cache_mode != PAB_CACHE_OFF) ctx->plan.diagonal = has(ctx->diag) ? 1 : 0;
    else ctx->plan.diagonal = has(ctx->diag_nt) ? 2 : 0;
}

bool ensure_diag_nt(pab_ctx* ctx, int set, cudaStream_t st) {        // set 0: 16 pixels per thread (orders 1..3), 1: 8 pixels
    if (!ctx->diag_nt_tried) {
        cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
        if (cudaStreamIsCapturing(st, &cap) != cudaSuccess || cap != cudaStreamCaptureStatusNone) { cudaGetLastError(); return false; }
        ctx->diag_nt_tried = true;
        const long long q = llround((double)ctx->pitch / (double)ctx->grid.dx);
        if (ctx->plan.in_range && ctx->plan.smem_bytes > 0 && q >= 1 && q <= 16 && (double)ctx->pitch == (double)q * (double)ctx->grid.dx &&
            xl_diag_configure(ctx->smem_optin) == cudaSuccess) {
            cudaError_t e = xl_diag_build(ctx->N, ctx->S, (double)ctx->fs, (double)ctx->c, ctx->grid, (int)q, 4, 3, ctx->smem_optin, 1,
                                          &ctx->diag_nt[0]);
            if (e == cudaSuccess)
                e = xl_diag_build(ctx->N, ctx->S, (double)ctx->fs, (double)ctx->c, ctx->grid, (int)q, 2, 6, ctx->smem_optin, 1, &ctx->diag_nt[1]);
            if (e != cudaSuccess) {          // not fatal: the call keeps the one-frame-per-thread kernels
                cudaGetLastError();
                xl_diag_free(&ctx->diag_nt[0]); xl_diag_free(&ctx->diag_nt[1]);
            } else {
                ctx->launches += 2;
                refresh_diagonal_flag(ctx);
            }
        } else {
            cudaGetLastError();
        }
    }
    return ctx->diag_nt[set].smem_bytes > 0;
}

// Orders 1 and 2 in frame groups are bound by the shared-memory data pipe, and at row pitches in (1, 8/7] samples 64-row
// tiles pay a bank conflict in every quarter-warp (tile_row, pab_pipe.cuh): a second tap-table set for 56-row tiles, when
// it stays below 512 MB.  Built on the first frame-group call of order 1 or 2 under PAB_CACHE_ALL (one device
// synchronisation, skipped while the stream is being captured), so that contexts that never run those orders do not
// carry the second table.
void ensure_taps7(pab_ctx* ctx, cudaStream_t st) {
    if (ctx->taps7_tried) return;
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cap) != cudaSuccess || cap != cudaStreamCaptureStatusNone) { cudaGetLastError(); return; }
    ctx->taps7_tried = true;
    if (!(ctx->plan.zs_per_row > 1.0 && ctx->plan.zs_per_row <= 8.0 / 7.0 + 1e-9)) return;
    const int tiles_x = (ctx->grid.nx + kStgCols - 1) / kStgCols, tiles_z7 = (ctx->grid.nz + 55) / 56;
    const size_t blocks7 = (size_t)tiles_x * tiles_z7 * ctx->N;
    if (tiles_z7 > 65535 || blocks7 * kCacheBlockBytes > (512u << 20)) return;
    cudaError_t e = cudaMalloc(&ctx->d_w0s7, blocks7 * sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&ctx->d_taps7, blocks7 * kCacheBlockBytes);
    if (e == cudaSuccess) {
        CacheGeom G{(double)ctx->fs, (double)ctx->c, (double)ctx->pitch, (double)ctx->grid.x0, (double)ctx->grid.dx,
                    (double)ctx->grid.z0, (double)ctx->grid.dz, ctx->N, ctx->S, ctx->grid.nx, ctx->grid.nz, tiles_x, 56};
        xl_build_delay_cache(G, tiles_z7, ctx->d_taps7, ctx->d_w0s7);
        ctx->launches++;
        e = cudaDeviceSynchronize();
    }
    if (e != cudaSuccess) {          // not fatal: the orders keep the 64-row tables
        cudaGetLastError();
        cudaFree(ctx->d_taps7); cudaFree(ctx->d_w0s7);
        ctx->d_taps7 = nullptr; ctx->d_w0s7 = nullptr;
    }
}

}  // namespace

extern "C" {

const char* pab_version(void) { return "pab 0.1 sm_100a"; }

const char* pab_strerror(int code) {
    switch (code) {
    case PAB_OK: return "ok";
    case PAB_ERR_INVALID: return "invalid argument";
    case PAB_ERR_DEVICE: return "no usable sm_100 CUDA device";
    case PAB_ERR_ALLOC: return "allocation failed";
    case PAB_ERR_CUDA: return "CUDA call failed";
    case PAB_ERR_LIMIT: return "size beyond the fixed maximum of a no-allocation entry point";
    default: return "unknown error code";
    }
}

const char* pab_last_cuda_error(const pab_ctx* ctx) { return ctx ? ctx->err : ""; }
long long pab_launch_count(const pab_ctx* ctx) { return ctx ? ctx->launches : 0; }

int pab_plan(int n_elem, int n_samp, float fs_hz, float c_m_s, float pitch_m, const pab_grid* grid,
             int smem_limit_bytes, pab_plan_info* plan_out) {
    if (!grid || !plan_out) return PAB_ERR_INVALID;
    return plan_geometry(n_elem, n_samp, fs_hz, c_m_s, pitch_m, *grid, smem_limit_bytes, plan_out) ? PAB_OK
                                                                                                    : PAB_ERR_INVALID;
}

int pab_get_plan(const pab_ctx* ctx, pab_plan_info* plan_out) {
    if (!ctx || !plan_out) return PAB_ERR_INVALID;
    *plan_out = ctx->plan;
    return PAB_OK;
}

int pab_design_bandpass(int n_taps, double f_lo, double f_hi, float* h_host) {
    if (!h_host || n_taps < 2 || n_taps > 256 || !(f_lo >= 0) || !(f_hi > f_lo) || !(f_hi <= 0.5)) return PAB_ERR_INVALID;
    design_bandpass(n_taps, f_lo, f_hi, h_host);
    return PAB_OK;
}

int pab_design_hilbert(int half_len, float* g_host) {
    if (!g_host || half_len < 1 || half_len > 127) return PAB_ERR_INVALID;
    design_hilbert(half_len, g_host);
    return PAB_OK;
}

int pab_create(pab_ctx** out, int n_elem, int n_samp, float fs_hz, float c_m_s, float pitch_m, const pab_grid* grid) {
    if (!out || !grid) return PAB_ERR_INVALID;
    pab_plan_info plan;
    if (!plan_geometry(n_elem, n_samp, fs_hz, c_m_s, pitch_m, *grid, 0, &plan)) return PAB_ERR_INVALID;
    if ((long long)n_samp > (1 << 20) || (long long)grid->nx * grid->nz > (1LL << 30)) return PAB_ERR_INVALID;
    int dev = 0, n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev < 1) { cudaGetLastError(); return PAB_ERR_DEVICE; }
    if (cudaGetDevice(&dev) != cudaSuccess) return PAB_ERR_DEVICE;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess || prop.major != 10) return PAB_ERR_DEVICE;

    pab_ctx* ctx = new (std::nothrow) pab_ctx();
    if (!ctx) return PAB_ERR_ALLOC;
    ctx->N = n_elem; ctx->S = n_samp; ctx->Sp = round_up(n_samp, 4);
    ctx->fs = fs_hz; ctx->c = c_m_s; ctx->pitch = pitch_m; ctx->grid = *grid;
    ctx->device = dev; ctx->sm_count = prop.multiProcessorCount; ctx->smem_optin = (int)prop.sharedMemPerBlockOptin;
    plan_geometry(n_elem, n_samp, fs_hz, c_m_s, pitch_m, *grid, ctx->smem_optin, &plan);
    ctx->plan = plan;

    const DelayTables t = make_tables(n_elem, fs_hz, c_m_s, pitch_m, *grid);
    // one batch of staged RF: quad layout, batch rounded up to whole quads (>= the lin layout of one frame)
    ctx->stage_bytes = (size_t)plan.batch_frames * n_elem * (size_t)ctx->Sp * 4;
    int rc = PAB_OK;
    auto fail = [&](cudaError_t e, const char* what) { rc = cuda_fail(ctx, e, what); };
    cudaError_t e;
    if ((e = cudaMalloc(&ctx->d_xj, t.xj.size() * 4)) != cudaSuccess) fail(e, "cudaMalloc xj");
    else if ((e = cudaMalloc(&ctx->d_xe, t.xe.size() * 4)) != cudaSuccess) fail(e, "cudaMalloc xe");
    else if ((e = cudaMalloc(&ctx->d_zrow, t.zrow.size() * 4)) != cudaSuccess) fail(e, "cudaMalloc zrow");
    else if ((e = cudaMalloc(&ctx->d_stage, ctx->stage_bytes)) != cudaSuccess) fail(e, "cudaMalloc stage");
    else if ((e = cudaMalloc(&ctx->d_max, (size_t)plan.batch_frames * 4)) != cudaSuccess) fail(e, "cudaMalloc max");
    else if ((e = cudaMemcpy(ctx->d_xj, t.xj.data(), t.xj.size() * 4, cudaMemcpyHostToDevice)) != cudaSuccess) fail(e, "copy xj");
    else if ((e = cudaMemcpy(ctx->d_xe, t.xe.data(), t.xe.size() * 4, cudaMemcpyHostToDevice)) != cudaSuccess) fail(e, "copy xe");
    else if ((e = cudaMemcpy(ctx->d_zrow, t.zrow.data(), t.zrow.size() * 4, cudaMemcpyHostToDevice)) != cudaSuccess) fail(e, "copy zrow");
    if (rc == PAB_OK) rc = xl_staged_configure(ctx->smem_optin);
    if (rc == PAB_OK && xl_post_configure(ctx->smem_optin) != cudaSuccess) rc = PAB_ERR_CUDA;
    if (rc != PAB_OK) { free_all(ctx); delete ctx; return rc; }
    // set-up of pab_post_no_alloc: the address of its fixed scratch array on this device.  A failure here is reported by
    // that entry point (which retries), not by pab_create.
    if (xl_post_no_alloc_setup(nullptr) != cudaSuccess) cudaGetLastError();
    *out = ctx;
    return PAB_OK;
}

void pab_destroy(pab_ctx* ctx) {
    if (!ctx) return;
    cudaDeviceSynchronize();
    free_all(ctx);
    delete ctx;
}

int pab_set_input(pab_ctx* ctx, int dtype, float scale) {
    if (!ctx || (dtype != PAB_F32 && dtype != PAB_I16) || !(scale == scale) || scale == 0.0f) return PAB_ERR_INVALID;
    ctx->dtype = dtype; ctx->scale = scale;
    return PAB_OK;
}

int pab_set_profile(pab_ctx* ctx, int max_launches) {
    if (!ctx || max_launches < 0 || max_launches > (1 << 20)) return PAB_ERR_INVALID;
    PAB_CUDA(ctx, cudaDeviceSynchronize());
    for (cudaEvent_t e : ctx->prof_ev) cudaEventDestroy(e);
    ctx->prof_ev.clear(); ctx->prof_stage.clear(); ctx->prof_used = 0;
    ctx->profiling = max_launches > 0;
    if (!ctx->profiling) return PAB_OK;
    ctx->prof_ev.resize((size_t)2 * max_launches, nullptr);
    ctx->prof_stage.assign(max_launches, 0);
    for (auto& e : ctx->prof_ev) PAB_CUDA(ctx, cudaEventCreate(&e));
    return PAB_OK;
}

int pab_get_profile(pab_ctx* ctx, int stage, double* total_ms, long long* n_launches, int reset) {
    if (!ctx || stage < 0 || stage >= PAB_STAGE_COUNT || !total_ms || !n_launches) return PAB_ERR_INVALID;
    double ms = 0.0; long long n = 0;
    for (int s = 0; s < ctx->prof_used; ++s) {
        if (ctx->prof_stage[s] != stage) continue;
        PAB_CUDA(ctx, cudaEventSynchronize(ctx->prof_ev[2 * s + 1]));
        float t = 0.0f;
        PAB_CUDA(ctx, cudaEventElapsedTime(&t, ctx->prof_ev[2 * s], ctx->prof_ev[2 * s + 1]));
        ms += t; ++n;
    }
    *total_ms = ms; *n_launches = n;
    if (reset) ctx->prof_used = 0;
    return PAB_OK;
}

int pab_set_tuning(pab_ctx* ctx, int frames_per_thread, int stages, int chunk_channels, int host_batch_frames) {
    if (!ctx || host_batch_frames < 0 || host_batch_frames > 64) return PAB_ERR_INVALID;
    PlanTuning t;
    t.frames_per_thread = frames_per_thread; t.stages = stages; t.chunk_channels = chunk_channels; t.host_batch_frames = host_batch_frames;
    pab_plan_info plan;
    if (!plan_geometry(ctx->N, ctx->S, ctx->fs, ctx->c, ctx->pitch, ctx->grid, ctx->smem_optin, &plan, t)) return PAB_ERR_INVALID;
    PAB_CUDA(ctx, cudaDeviceSynchronize());
    ctx->tuning = t;
    plan.diagonal = ctx->plan.diagonal;
    ctx->plan = plan;
    if (ctx->variant == PAB_VARIANT_STAGED && plan.smem_bytes == 0) ctx->variant = PAB_VARIANT_AUTO;
    return PAB_OK;
}

int pab_set_weight(pab_ctx* ctx, int weight) {
    if (!ctx || (weight != PAB_WEIGHT_NONE && weight != PAB_WEIGHT_CF)) return PAB_ERR_INVALID;
    if (weight == PAB_WEIGHT_CF && ctx->interp == PAB_INTERP_NEAREST) return PAB_ERR_INVALID;
    ctx->weight = weight;
    return PAB_OK;
}

int pab_set_delay_cache(pab_ctx* ctx, int mode) {
    if (!ctx || mode < PAB_CACHE_OFF || mode > PAB_CACHE_ALL) return PAB_ERR_INVALID;
    if (mode != PAB_CACHE_OFF) {
        if (!ctx->plan.in_range || ctx->plan.smem_bytes == 0 || ctx->plan.window_samples > kCacheMaxWindow) return PAB_ERR_INVALID;
        const int tiles_x = (ctx->grid.nx + kStgCols - 1) / kStgCols, tiles_z = (ctx->grid.nz + kStgRows - 1) / kStgRows;
        if (tiles_z > 65535 || ctx->N > 65535) return PAB_ERR_INVALID;
        const size_t blocks = (size_t)tiles_x * tiles_z * ctx->N;
        // translation invariance: pitch = q dx exactly (both are the floats the ABI carries) -> compact (d, row) table,
        // used by the one-frame-per-thread kernel (through L1/L2); the frame-group kernels always take the
        // tile-major table staged by TMA (the compact table's global loads cost them 9 %)
        const long long q = llround((double)ctx->pitch / (double)ctx->grid.dx);
        const bool compact = q >= 1 && q <= 64 && (double)ctx->pitch == (double)q * (double)ctx->grid.dx &&
                             (long long)ctx->grid.nx + q * (ctx->N - 1) <= 65535 &&
                             ((long long)ctx->grid.nx + q * (ctx->N - 1)) * ctx->grid.nz < (1LL << 31);
        const bool need_taps = (mode == PAB_CACHE_ALL || !compact) && !ctx->d_taps;
        const bool need_w0s = !ctx->d_w0s, need_compact = compact && !ctx->d_compact;
        if (need_taps || need_w0s || need_compact) {
            PAB_CUDA(ctx, xl_cached_configure(ctx->smem_optin));
            cudaError_t e = cudaSuccess;
            if (need_w0s) e = cudaMalloc(&ctx->d_w0s, blocks * sizeof(int));
            if (e == cudaSuccess && need_taps) e = cudaMalloc(&ctx->d_taps, blocks * kCacheBlockBytes);
            const int nd = ctx->grid.nx + (int)q * (ctx->N - 1);
            if (e == cudaSuccess && need_compact) e = cudaMalloc(&ctx->d_compact, (size_t)nd * ctx->grid.nz * sizeof(uint2));
            if (e == cudaSuccess) {
                CacheGeom G{(double)ctx->fs, (double)ctx->c, (double)ctx->pitch, (double)ctx->grid.x0, (double)ctx->grid.dx,
                            (double)ctx->grid.z0, (double)ctx->grid.dz, ctx->N, ctx->S, ctx->grid.nx, ctx->grid.nz, tiles_x, kStgRows};
                if (need_taps || need_w0s) {
                    xl_build_delay_cache(G, tiles_z, ctx->d_taps, ctx->d_w0s);
                    ctx->launches++;
                }
                if (need_compact) {
                    xl_build_delay_compact(G, (int)q, nd, ctx->d_compact);
                    ctx->launches++;
                    ctx->cache_q = (int)q;
                }
                e = cudaDeviceSynchronize();
            }
            if (e != cudaSuccess) {
                cudaFree(ctx->d_taps); cudaFree(ctx->d_w0s); cudaFree(ctx->d_compact);
                ctx->d_taps = nullptr; ctx->d_w0s = nullptr; ctx->d_compact = nullptr;
                return cuda_fail(ctx, e, "delay cache");
            }
        }
    }
    // translation-invariant geometries: calls of 1..3 frames take the diagonal kernel (pab_diag.cuh), which shares one
    // tap among the 16 (8 for orders 4, 5) pairs of a diagonal and reads the caller's frame in place
    if (mode != PAB_CACHE_OFF && ctx->d_compact && ctx->diag[0].smem_bytes == 0 && ctx->diag[1].smem_bytes == 0) {
        PAB_CUDA(ctx, xl_diag_configure(ctx->smem_optin));
        cudaError_t e = xl_diag_build(ctx->N, ctx->S, (double)ctx->fs, (double)ctx->c, ctx->grid, ctx->cache_q,
                                      4, 3, ctx->smem_optin, 0, &ctx->diag[0]);
        if (e == cudaSuccess) e = xl_diag_build(ctx->N, ctx->S, (double)ctx->fs, (double)ctx->c, ctx->grid, ctx->cache_q, 2, 6, ctx->smem_optin, 0, &ctx->diag[1]);
        if (e != cudaSuccess) { xl_diag_free(&ctx->diag[0]); xl_diag_free(&ctx->diag[1]); return cuda_fail(ctx, e, "diagonal tables"); }
        ctx->launches += 4;
    }
    ctx->cache_mode = mode;
    refresh_diagonal_flag(ctx);
    return PAB_OK;
}

int pab_self_check(pab_ctx* ctx, const float* rf_dev, int order, long long* violations) {
    if (!ctx || !rf_dev || !violations || order < 1 || order > 5) return PAB_ERR_INVALID;
    // delay cache on: the kernel with its tap table; off: its table-free form (built here if no call has built it yet)
    const bool near = ctx->interp == PAB_INTERP_NEAREST;        // the nearest-sample path: the kernel on its table of integer delays
    if (!near && ctx->cache_mode == PAB_CACHE_OFF && (ctx->variant != PAB_VARIANT_AUTO || !ensure_diag_nt(ctx, order <= 3 ? 0 : 1, 0))) return PAB_ERR_INVALID;
    const DiagSet& D = near ? ctx->diag_near[order <= 3 ? 0 : 1]
                            : ctx->cache_mode == PAB_CACHE_OFF ? ctx->diag_nt[order <= 3 ? 0 : 1] : ctx->diag[order <= 3 ? 0 : 1];
    if (D.smem_bytes == 0 || ctx->dtype != PAB_F32) return PAB_ERR_INVALID;
    float* out = nullptr;
    int* d_viol = nullptr;
    int h = 0;
    cudaError_t e = cudaMalloc(&out, (size_t)ctx->grid.nz * ctx->grid.nx * 4);
    if (e == cudaSuccess) e = cudaMalloc(&d_viol, 4);
    if (e == cudaSuccess) e = cudaMemset(d_viol, 0, 4);
    if (e == cudaSuccess) e = xl_diag_check(order, D, rf_dev, out, ctx->N, ctx->S, ctx->grid.nx, ctx->grid.nz, d_viol, 0);
    if (e == cudaSuccess) { ctx->launches++; e = cudaMemcpy(&h, d_viol, 4, cudaMemcpyDeviceToHost); }
    cudaFree(out); cudaFree(d_viol);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "self check");
    *violations = h;
    return PAB_OK;
}

int pab_set_interp(pab_ctx* ctx, int interp) {
    if (!ctx || (interp != PAB_INTERP_LINEAR && interp != PAB_INTERP_NEAREST)) return PAB_ERR_INVALID;
    if (interp == PAB_INTERP_NEAREST) {
        if (ctx->weight != PAB_WEIGHT_NONE || ctx->S > 65534) return PAB_ERR_INVALID;
        PAB_CUDA(ctx, xl_nearest_configure(ctx->smem_optin));
        if (!ctx->d_near) {
            const int tiles_x = (ctx->grid.nx + kStgCols - 1) / kStgCols, tiles_z = (ctx->grid.nz + kStgRows - 1) / kStgRows;
            const size_t n = (size_t)ctx->N * tiles_x * kStgCols * (size_t)tiles_z * kStgRows;
            PAB_CUDA(ctx, cudaMalloc(&ctx->d_near, n * sizeof(unsigned short)));
            NearestGeom G{(double)ctx->fs, (double)ctx->c, (double)ctx->pitch, (double)ctx->grid.x0, (double)ctx->grid.dx,
                          (double)ctx->grid.z0, (double)ctx->grid.dz, ctx->N, ctx->S, ctx->grid.nx, ctx->grid.nz};
            if (!xl_nearest_table(G, ctx->d_near)) { cudaFree(ctx->d_near); ctx->d_near = nullptr; return PAB_ERR_INVALID; }
            ctx->launches++;
            cudaError_t e = cudaDeviceSynchronize();
            if (e != cudaSuccess) { cudaFree(ctx->d_near); ctx->d_near = nullptr; return cuda_fail(ctx, e, "nearest table"); }
        }
        // Calls of 1..3 frames on translation-invariant in-range geometries: the single-frame diagonal kernel (pab_diag.cuh)
        // with a table of floor(idx + 1/2) and fraction 0, so that its interpolation returns rf[n] exactly and one integer
        // delay serves the 16 (8) pairs of a diagonal; the decision is taken in fp64 by the same expression as the uint16
        // table's.  Not fatal when the sets cannot be had: such calls keep the frame-group kernels.
        if (ctx->diag_near[0].smem_bytes == 0 && ctx->diag_near[1].smem_bytes == 0) {
            const long long q = llround((double)ctx->pitch / (double)ctx->grid.dx);
            if (ctx->plan.in_range && ctx->plan.smem_bytes > 0 && q >= 1 && q <= 16 &&
                (double)ctx->pitch == (double)q * (double)ctx->grid.dx && xl_diag_configure(ctx->smem_optin) == cudaSuccess) {
                cudaError_t e = xl_diag_build(ctx->N, ctx->S, (double)ctx->fs, (double)ctx->c, ctx->grid, (int)q, 4, 3, ctx->smem_optin, 2,
                                              &ctx->diag_near[0]);
                if (e == cudaSuccess)
                    e = xl_diag_build(ctx->N, ctx->S, (double)ctx->fs, (double)ctx->c, ctx->grid, (int)q, 2, 5, ctx->smem_optin, 2, &ctx->diag_near[1]);
                if (e != cudaSuccess) { cudaGetLastError(); xl_diag_free(&ctx->diag_near[0]); xl_diag_free(&ctx->diag_near[1]); }
                else ctx->launches += 4;
            } else {
                cudaGetLastError();
            }
        }
    }
    ctx->interp = interp;
    refresh_diagonal_flag(ctx);
    return PAB_OK;
}

int pab_set_variant(pab_ctx* ctx, int variant) {
    if (!ctx || variant < PAB_VARIANT_AUTO || variant > PAB_VARIANT_STAGED) return PAB_ERR_INVALID;
    if (variant == PAB_VARIANT_STAGED && ctx->plan.smem_bytes == 0) return PAB_ERR_INVALID;
    ctx->variant = variant;
    return PAB_OK;
}

int pab_set_post(pab_ctx* ctx, int mode, float f_center_hz, float f_halfwidth_hz, int n_taps_bp, int n_taps_hilbert,
                 float dyn_range_db) {
    if (!ctx || mode < PAB_RAW || mode > PAB_LOG) return PAB_ERR_INVALID;
    if (mode == PAB_RAW) { ctx->post_mode = PAB_RAW; return PAB_OK; }
    const double fs_z = (double)ctx->c / (double)ctx->grid.dz;      // axial sampling rate, one-way (A13)
    const double f_lo = ((double)f_center_hz - (double)f_halfwidth_hz) / fs_z;
    const double f_hi = ((double)f_center_hz + (double)f_halfwidth_hz) / fs_z;
    if (n_taps_bp < 2 || n_taps_bp > 256 || !(f_lo >= 0) || !(f_hi > f_lo) || !(f_hi <= 0.5)) return PAB_ERR_INVALID;
    if (mode >= PAB_ENVELOPE && (n_taps_hilbert < 3 || n_taps_hilbert > 255 || !(n_taps_hilbert & 1))) return PAB_ERR_INVALID;
    if (mode == PAB_LOG && !(dyn_range_db > 0)) return PAB_ERR_INVALID;
    const int TpB = round_up(n_taps_bp, 8);
    const int TpH = mode >= PAB_ENVELOPE ? round_up(n_taps_hilbert, 8) : 8;
    std::vector<float> hb(TpB, 0.0f), hh(TpH, 0.0f);
    design_bandpass(n_taps_bp, f_lo, f_hi, hb.data());
    if (mode >= PAB_ENVELOPE) design_hilbert((n_taps_hilbert - 1) / 2, hh.data());
    PAB_CUDA(ctx, cudaDeviceSynchronize());
    // the new tap buffers are allocated and filled first and swapped in only on success: a failure leaves the
    // context with its previous post chain intact
    float *nb = nullptr, *nh = nullptr;
    cudaError_t e = cudaMalloc(&nb, TpB * 4);
    if (e == cudaSuccess) e = cudaMalloc(&nh, TpH * 4);
    if (e == cudaSuccess) e = cudaMemcpy(nb, hb.data(), TpB * 4, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(nh, hh.data(), TpH * 4, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { cudaFree(nb); cudaFree(nh); return cuda_fail(ctx, e, "post taps"); }
    if (!ctx->d_img) {
        e = cudaMalloc(&ctx->d_img, (size_t)ctx->plan.batch_frames * ctx->grid.nz * (size_t)ctx->grid.nx * 4);
        if (e != cudaSuccess) { ctx->d_img = nullptr; cudaFree(nb); cudaFree(nh); return cuda_fail(ctx, e, "post scratch"); }
    }
    cudaFree(ctx->d_taps_bp); cudaFree(ctx->d_taps_h);
    ctx->d_taps_bp = nb; ctx->d_taps_h = nh;
    // fast path: both filters fit 64 taps and are long enough for it to pay
    ctx->post_fast = TpB > 32 && TpB <= 64 && (mode < PAB_ENVELOPE || (TpH > 32 && TpH <= 64));
    if (ctx->post_fast) {
        memset(&ctx->taps64, 0, sizeof ctx->taps64);
        PostTaps64& T = ctx->taps64;
        for (int t = 0; t < TpB; ++t) T.hbr[63 - t] = hb[t];
        for (int j = 1; j < 64; ++j) T.hbs[j] = T.hbr[j - 1];
        bool even_zero = true, odd_zero = true;
        if (mode >= PAB_ENVELOPE)
            for (int t = 0; t < TpH; ++t) {
                T.hhr[63 - t] = hh[t];
                if (hh[t] != 0.0f) { if (t & 1) odd_zero = false; else even_zero = false; }
            }
        for (int j = 1; j < 64; ++j) T.hhs[j] = T.hhr[j - 1];
        // type III: the non-zero original parity p sits at reversed parity 1 - p
        const int q = odd_zero ? 1 : 0;
        for (int i = 0; i < 32; ++i) T.hhd[2 * i] = T.hhd[2 * i + 1] = T.hhr[q + 2 * i];
        ctx->hilbert_parity = odd_zero ? 0 : (even_zero ? 1 : 2);
    }
    ctx->post_mode = mode; ctx->n_taps_bp = n_taps_bp; ctx->n_taps_h = n_taps_hilbert;
    ctx->TpB = TpB; ctx->TpH = TpH; ctx->dyn_range_db = dyn_range_db;
    return PAB_OK;
}

int pab_post_no_alloc(pab_ctx* ctx, const float* img_dev, int n_frames, float* out_dev, void* cuda_stream) {
    if (!ctx || !img_dev || !out_dev || n_frames < 1) return PAB_ERR_INVALID;
    if (((uintptr_t)img_dev % 4) != 0 || ((uintptr_t)out_dev % 4) != 0) return PAB_ERR_INVALID;
    if (n_frames > PAB_NO_ALLOC_MAX_FRAMES) {
        snprintf(ctx->err, sizeof ctx->err, "pab_post_no_alloc: n_frames = %d exceeds PAB_NO_ALLOC_MAX_FRAMES = %d (fixed scratch array)",
                 n_frames, PAB_NO_ALLOC_MAX_FRAMES);
        return PAB_ERR_LIMIT;
    }
    if (ctx->post_mode < PAB_ENVELOPE || !ctx->post_fast) return PAB_ERR_INVALID;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != ctx->device) return PAB_ERR_INVALID;
    const int nx = ctx->grid.nx, nz = ctx->grid.nz;
    const size_t bytes = (size_t)n_frames * nz * (size_t)nx * 4;
    const uintptr_t a = (uintptr_t)img_dev, b = (uintptr_t)out_dev;
    if (a < b + bytes && b < a + bytes) return PAB_ERR_INVALID;          // the FIR tiles read their neighbours' rows
    PostParams Q{};
    Q.x = img_dev; Q.out = out_dev;
    Q.TpB = ctx->TpB; Q.shiftB = ctx->n_taps_bp / 2;
    Q.TpH = ctx->TpH; Q.shiftH = (ctx->n_taps_h - 1) / 2;
    Q.nx = nx; Q.nz = nz;
    int launches = 0;
    const cudaError_t e = xl_post_no_alloc(Q, ctx->taps64, ctx->hilbert_parity, n_frames, ctx->post_mode == PAB_LOG, ctx->dyn_range_db,
                                           (cudaStream_t)cuda_stream, &launches);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "pab_post_no_alloc");
    ctx->launches += launches;
    return PAB_OK;
}

int pab_image_metrics(pab_ctx* ctx, const float* img_dev, const pab_roi* target, const pab_roi* background, int n_bins,
                      int fwhm_row, pab_metrics* out_host, void* cuda_stream) {
    if (!ctx || !img_dev || !target || !background || !out_host || n_bins < 2 || n_bins > 4096) return PAB_ERR_INVALID;
    const int nz = ctx->grid.nz, nx = ctx->grid.nx;
    auto bad = [&](const pab_roi* r) { return r->r0 < 0 || r->r1 > nz || r->c0 < 0 || r->c1 > nx || r->r0 >= r->r1 || r->c0 >= r->c1; };
    if (bad(target) || bad(background) || fwhm_row >= nz) return PAB_ERR_INVALID;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t acc_bytes = 64, hist_off = 128, total = hist_off + 2 * 4096 * sizeof(unsigned int);
    if (!ctx->d_metric) PAB_CUDA(ctx, cudaMalloc(&ctx->d_metric, total));
    char* base = (char*)ctx->d_metric;
    MetricAcc* acc = (MetricAcc*)base;
    double* fw = (double*)(base + acc_bytes);
    unsigned int* hist = (unsigned int*)(base + hist_off);
    PAB_CUDA(ctx, cudaMemsetAsync(base, 0, total, st));
    RoiPair R{{target->r0, target->r1, target->c0, target->c1}, {background->r0, background->r1, background->c0, background->c1}};
    ctx->launches += xl_metrics(img_dev, nx, R, acc, hist, n_bins, fwhm_row, fw, st);
    MetricAcc h{};
    double fwh = 0.0;
    std::vector<unsigned int> hh(2 * (size_t)n_bins);
    PAB_CUDA(ctx, cudaMemcpyAsync(&h, acc, sizeof h, cudaMemcpyDeviceToHost, st));
    PAB_CUDA(ctx, cudaMemcpyAsync(&fwh, fw, sizeof fwh, cudaMemcpyDeviceToHost, st));
    PAB_CUDA(ctx, cudaMemcpyAsync(hh.data(), hist, hh.size() * sizeof(unsigned int), cudaMemcpyDeviceToHost, st));
    PAB_CUDA(ctx, cudaStreamSynchronize(st));
    const double n_in = (double)(target->r1 - target->r0) * (target->c1 - target->c0);
    const double n_out = (double)(background->r1 - background->r0) * (background->c1 - background->c0);
    pab_metrics m{};
    m.mu_in = h.sum_in / n_in; m.mu_out = h.sum_out / n_out; m.sigma_out = std::sqrt(h.var_out / n_out);
    m.snr_db = 20.0 * std::log10(m.mu_in / m.sigma_out);
    m.cr_db = 20.0 * std::log10(m.mu_in / m.mu_out);
    double ovl = 0.0;
    for (int b = 0; b < n_bins; ++b) {
        const double a = hh[b] / n_in, o = hh[n_bins + b] / n_out;
        ovl += a < o ? a : o;
    }
    m.gcnr = 1.0 - ovl;
    m.fwhm_m = fwhm_row >= 0 ? fwh * (double)ctx->grid.dx : std::nan("");
    *out_host = m;
    return PAB_OK;
}

}  // extern "C"

#include "pab_run.inl"
