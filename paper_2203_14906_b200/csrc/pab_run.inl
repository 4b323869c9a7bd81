// pab_run.inl -- included by pab_api.cu: batch driver and the two beamform entry points.

namespace {

// One kernel launch: counts it, and brackets it with CUDA events on its stream when profiling is on.
struct Span {
    pab_ctx* c; int stage; cudaStream_t st; int slot = -1;
    Span(pab_ctx* c_, int stage_, cudaStream_t st_) : c(c_), stage(stage_), st(st_) {
        if (c->profiling && c->prof_used < (int)c->prof_ev.size() / 2) {
            slot = c->prof_used++;
            c->prof_stage[slot] = stage;
            cudaEventRecord(c->prof_ev[2 * slot], st);
        }
    }
    ~Span() {
        c->launches++;
        if (slot >= 0) cudaEventRecord(c->prof_ev[2 * slot + 1], st);
    }
};

// One batch (<= plan.batch_frames frames): ingest -> beamform -> post.  rf points at the batch's first frame
// in the caller's layout, out at the batch's first image.
int run_batch(pab_ctx* ctx, const void* rf, int F, int order, float* out, cudaStream_t st) {
    const int F_all = F;                 // frames of the batch (F shrinks to whole quads when the diagonal kernel takes a remainder)
    const int N = ctx->N, S = ctx->S, nx = ctx->grid.nx, nz = ctx->grid.nz;
    const bool post = ctx->post_mode != PAB_RAW;
    BfParams P{};
    P.xj = ctx->d_xj; P.xe = ctx->d_xe; P.zrow = ctx->d_zrow;
    P.N = N; P.S = S; P.Sp = ctx->Sp; P.nx = nx; P.nz = nz;
    P.inv_n = 1.0f / (float)N;
    const int weight = ctx->weight;
    P.out = post ? ctx->d_img : out;
    const bool in_range = ctx->plan.in_range != 0;
    const bool use_staged = ctx->variant == PAB_VARIANT_STAGED ||
                            (ctx->variant == PAB_VARIANT_AUTO && ctx->plan.smem_bytes > 0);

    // table set of the single-frame diagonal kernel: 16 pixels per thread for orders 1..3, 8 for orders 4, 5 and for every order
    // under coherence-factor weighting (more accumulators per pixel)
    const int dset = (order <= 3 && weight == 0) ? 0 : 1;
    if (ctx->interp == PAB_INTERP_NEAREST && F < 4 && use_staged && order <= 5 && ctx->diag_near[order <= 3 ? 0 : 1].smem_bytes > 0) {
        // row f4, calls of 1..3 frames on translation-invariant geometries: the diagonal kernel on its table of integer delays
        // (fraction 0: the interpolation returns rf[n] exactly), straight from the caller's frames; roots per item
        Span sp(ctx, PAB_STAGE_BEAMFORM, st);
        xl_diag(order, ctx->dtype, 0, ctx->diag_near[order <= 3 ? 0 : 1], rf, P.out, F, N, S, nx, nz, ctx->scale, st);
    } else if (ctx->interp == PAB_INTERP_NEAREST) {
        // row f4: rooted quad staging, then the table-driven gather kernel (always the quad layout)
        {
            Span sp(ctx, PAB_STAGE_INGEST, st);
            xl_ingest_root_quad(ctx->dtype, order, rf, ctx->d_stage, F, N, S, ctx->scale, st);
        }
        int nq = (F + 3) / 4, q0 = 0;
        int g0 = ctx->plan.frames_per_thread / 4;
        if (order >= 4 && g0 > 2) g0 = 2;
        for (int g = g0; g >= 1 && nq > 0; g >>= 1) {
            const int groups = nq / g;
            if (groups == 0) continue;
            BfParams R = P;
            R.rf = ctx->d_stage + (size_t)q0 * N * (size_t)S * 4;
            R.out = P.out + (size_t)(4 * q0) * nz * (size_t)nx;
            R.n_frames = F - 4 * q0;
            Span sp(ctx, PAB_STAGE_BEAMFORM, st);
            if (use_staged && xl_nearest_staged_fits(ctx->plan, g, ctx->tuning.stages, ctx->smem_optin))
                xl_nearest_staged(order, g, in_range, R, groups, ctx->plan, ctx->tuning.stages, ctx->tuning.chunk_channels,
                                                  ctx->smem_optin, ctx->sm_count, ctx->d_near, st);
            else xl_nearest_direct(order, g, R, groups, ctx->d_near, st);
            q0 += groups * g;
            nq -= groups * g;
        }
    } else if (F < 4 && ctx->cache_mode != PAB_CACHE_OFF && use_staged && order <= 5 && ctx->diag[dset].smem_bytes > 0) {
        // translation-invariant geometry: the diagonal kernel, straight from the caller's frames (no ingest pass)
        Span sp(ctx, PAB_STAGE_BEAMFORM, st);
        xl_diag(order, ctx->dtype, weight, ctx->diag[dset], rf, P.out, F, N, S, nx, nz, ctx->scale, st);
    } else if (F < 4 && ctx->cache_mode == PAB_CACHE_OFF && ctx->variant == PAB_VARIANT_AUTO && order <= 5 &&
               ensure_diag_nt(ctx, dset, st)) {
        // the same kernel without any delay table: the tap of a diagonal is computed in the kernel (FP64 pipe)
        Span sp(ctx, PAB_STAGE_BEAMFORM, st);
        xl_diag(order, ctx->dtype, weight, ctx->diag_nt[dset], rf, P.out, F, N, S, nx, nz, ctx->scale, st);
    } else if (F < 4) {
        const bool cached = ctx->cache_mode != PAB_CACHE_OFF && use_staged && weight == 0 && order <= 5 &&
                            xl_cached_fits(ctx->plan, 0, ctx->d_compact != nullptr, ctx->smem_optin);
        // lin layout, one frame per thread.  fp32 input with unit scale and 16-byte rows is read in place.
        const bool in_place = ctx->dtype == PAB_F32 && ctx->scale == 1.0f && (S % 4) == 0 &&
                              ((uintptr_t)rf % 16) == 0;
        if (in_place) {
            P.rf = (const float*)rf;
        } else {
            {
                Span sp(ctx, PAB_STAGE_INGEST, st);
                xl_ingest_lin(ctx->dtype, rf, ctx->d_stage, F, N, S, ctx->Sp, ctx->scale, st);
            }
            P.rf = ctx->d_stage;
        }
        P.n_frames = F;
        {
            Span sp(ctx, PAB_STAGE_BEAMFORM, st);
            if (cached) xl_cached(order, 0, 0, P, F, ctx->plan, ctx->tuning.chunk_channels, ctx->smem_optin, ctx->sm_count,
                                      CacheTables{ctx->d_taps, ctx->d_w0s, ctx->d_compact, ctx->cache_q, kStgRows}, st);
            else if (use_staged) xl_staged(order, 0, in_range, weight, P, F, ctx->plan, ctx->tuning.chunk_channels, ctx->smem_optin, ctx->sm_count, st);
            else xl_direct(order, 0, weight, P, F, st);
        }
    } else {
        // A remainder of 1..3 frames would cost a whole padded quad (or, after an odd quad count, a padded 8-frame group):
        // where the single-frame diagonal kernel is available it takes those frames instead, straight from the caller's
        // buffer (measured at C2b order 3: 5 frames 181 -> 138 us, 9 frames 287 -> 215 us).
        const int rem = F & 3;
        const DiagSet* dg = nullptr;
        if (rem != 0 && order <= 5) {
            if (ctx->cache_mode != PAB_CACHE_OFF && use_staged && ctx->diag[dset].smem_bytes > 0) dg = &ctx->diag[dset];
            else if (ctx->cache_mode == PAB_CACHE_OFF && ctx->variant == PAB_VARIANT_AUTO && ensure_diag_nt(ctx, dset, st)) dg = &ctx->diag_nt[dset];
        }
        if (dg) {
            const int Fq = F - rem;
            Span sp(ctx, PAB_STAGE_BEAMFORM, st);
            xl_diag(order, ctx->dtype, weight, *dg, (const char*)rf + (size_t)Fq * N * (size_t)S * elem_size(ctx->dtype),
                    P.out + (size_t)Fq * nz * (size_t)nx, rem, N, S, nx, nz, ctx->scale, st);
            F = Fq;                      // the frame groups below see whole quads only; the post chain still sees every frame
        }
        {
            Span sp(ctx, PAB_STAGE_INGEST, st);
            xl_ingest_quad(ctx->dtype, rf, ctx->d_stage, F, N, S, ctx->scale, st);
        }
        if (ctx->cache_mode == PAB_CACHE_ALL && order <= 2 && weight == 0 && F >= 8) ensure_taps7(ctx, st);
        // quads are consumed in groups of frames_per_thread / 4, then the remainder in halves (4 -> 2 -> 1)
        int nq = (F + 3) / 4, q0 = 0;
        // orders 4 and 5 carry at most 8 frames per thread (16 x 5 accumulators would spill)
        int g0 = ctx->plan.frames_per_thread / 4;
        if (order >= 4 && g0 > 2) g0 = 2;
        if (order >= 6) g0 = 1;
        if (weight != 0) g0 = g0 > (order >= 4 ? 1 : 2) ? (order >= 4 ? 1 : 2) : g0;     // CF: +1..2 accumulators per frame
        for (int g = g0; g >= 1 && nq > 0; g >>= 1) {
            const int groups = nq / g;
            if (groups == 0) continue;
            BfParams R = P;
            R.rf = ctx->d_stage + (size_t)q0 * N * (size_t)S * 4;
            R.out = P.out + (size_t)(4 * q0) * nz * (size_t)nx;
            R.n_frames = F - 4 * q0;
            Span sp(ctx, PAB_STAGE_BEAMFORM, st);
            if (ctx->cache_mode == PAB_CACHE_ALL && use_staged && (order <= 5 || g == 1) &&
                (weight == 0 || xl_cached_weight_ok(order, g, false)) && xl_cached_fits(ctx->plan, g, false, ctx->smem_optin))
                xl_cached(order, g, weight, R, groups, ctx->plan, ctx->tuning.chunk_channels, ctx->smem_optin, ctx->sm_count,
                              (order <= 2 && weight == 0 && g >= 2 && ctx->d_taps7)
                                  ? CacheTables{ctx->d_taps7, ctx->d_w0s7, nullptr, 0, 56}
                                  : CacheTables{ctx->d_taps, ctx->d_w0s, nullptr, 0, kStgRows}, st);
            else if (use_staged) xl_staged(order, g, in_range, weight, R, groups, ctx->plan, ctx->tuning.chunk_channels, ctx->smem_optin, ctx->sm_count, st);
            else xl_direct(order, g, weight, R, groups, st);
            q0 += groups * g;
            nq -= groups * g;
        }
    }
    if (post) {
        PostParams Q{};
        Q.x = ctx->d_img; Q.out = out; Q.frame_max = ctx->d_max;
        Q.taps_bp = ctx->d_taps_bp; Q.taps_h = ctx->d_taps_h;
        Q.TpB = ctx->TpB; Q.shiftB = ctx->n_taps_bp / 2;
        Q.TpH = ctx->TpH; Q.shiftH = (ctx->n_taps_h - 1) / 2;
        Q.nx = nx; Q.nz = nz;
        const bool env = ctx->post_mode >= PAB_ENVELOPE;
        if (env) cudaMemsetAsync(ctx->d_max, 0, (size_t)F_all * 4, st);
        {
            Span sp(ctx, PAB_STAGE_POST_FIR, st);
            if (ctx->post_fast) xl_post64(Q, ctx->taps64, env, ctx->hilbert_parity, F_all, st);
            else xl_post_generic(Q, env, F_all, st);
        }
        if (ctx->post_mode == PAB_LOG) {
            Span sp(ctx, PAB_STAGE_POST_LOG, st);
            xl_post_log(out, ctx->d_max, nx * nz, F_all, ctx->dyn_range_db, st);
        }
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(ctx, e, "kernel launch");
    return PAB_OK;
}

int check_args(pab_ctx* ctx, const void* rf, int n_frames, int order, const float* out) {
    if (!ctx || !rf || !out || n_frames < 1 || order < 1 || order > PAB_MAX_ORDER) return PAB_ERR_INVALID;
    if (order > 5 && (ctx->weight != PAB_WEIGHT_NONE || ctx->interp != PAB_INTERP_LINEAR)) return PAB_ERR_INVALID;
    if (((uintptr_t)rf % elem_size(ctx->dtype)) != 0 || ((uintptr_t)out % 4) != 0) return PAB_ERR_INVALID;
    int dev = -1;                         // the context lives on the device that was current at pab_create
    if (cudaGetDevice(&dev) != cudaSuccess || dev != ctx->device) return PAB_ERR_INVALID;
    return PAB_OK;
}

}  // namespace

extern "C" int pab_beamform(pab_ctx* ctx, const void* rf_dev, int n_frames, int order, float* out_dev, void* cuda_stream) {
    int rc = check_args(ctx, rf_dev, n_frames, order, out_dev);
    if (rc != PAB_OK) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t frame_in = (size_t)ctx->N * ctx->S * elem_size(ctx->dtype);
    const size_t frame_out = (size_t)ctx->grid.nz * ctx->grid.nx;
    for (int f0 = 0; f0 < n_frames; f0 += ctx->plan.batch_frames) {
        const int F = n_frames - f0 < ctx->plan.batch_frames ? n_frames - f0 : ctx->plan.batch_frames;
        rc = run_batch(ctx, (const char*)rf_dev + (size_t)f0 * frame_in, F, order, out_dev + (size_t)f0 * frame_out, st);
        if (rc != PAB_OK) return rc;
    }
    return PAB_OK;
}

namespace {

// Enqueue the host path for one call on the context's three internal streams (H2D, kernels, D2H) with kHostSets device
// buffer sets.  `ctx->host_it` counts pieces over the life of the context, so that the buffer hand-over events order successive
// calls as well as successive pieces of one call.  B: frames per piece; ramp: half pieces at both ends of the call.
int host_enqueue(pab_ctx* ctx, const void* rf_host, int n_frames, int order, float* out_host, int B, bool ramp) {
    const int Bcap = ctx->plan.batch_frames < 64 ? ctx->plan.batch_frames : 64;
    const size_t frame_in = (size_t)ctx->N * ctx->S * elem_size(ctx->dtype);
    const size_t frame_out = (size_t)ctx->grid.nz * ctx->grid.nx * 4;
    if (!ctx->s_h2d) {
        PAB_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->s_h2d, cudaStreamNonBlocking));
        PAB_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->s_run, cudaStreamNonBlocking));
        PAB_CUDA(ctx, cudaStreamCreateWithFlags(&ctx->s_d2h, cudaStreamNonBlocking));
        for (int b = 0; b < kHostSets; ++b) {
            PAB_CUDA(ctx, cudaMalloc(&ctx->d_in[b], (size_t)Bcap * ctx->N * ctx->S * 4));   // sized for fp32
            PAB_CUDA(ctx, cudaMalloc(&ctx->d_out[b], (size_t)Bcap * frame_out));
            PAB_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_in[b], cudaEventDisableTiming));
            PAB_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_run[b], cudaEventDisableTiming));
            PAB_CUDA(ctx, cudaEventCreateWithFlags(&ctx->ev_out[b], cudaEventDisableTiming));
        }
    }
    // H2D of piece b+1 and D2H of piece b-1 overlap the kernels of piece b.
    for (int f0 = 0, F = 0; f0 < n_frames; f0 += F, ++ctx->host_it) {
        F = n_frames - f0 < B ? n_frames - f0 : B;
        if (ramp && (f0 == 0 || n_frames - f0 <= B)) F = (f0 == 0 || n_frames - f0 > B / 2) ? B / 2 : n_frames - f0;
        const long long it = ctx->host_it;
        const int b = (int)(it % kHostSets);
        if (it >= kHostSets) PAB_CUDA(ctx, cudaStreamWaitEvent(ctx->s_h2d, ctx->ev_run[b], 0));   // d_in[b] consumed
        PAB_CUDA(ctx, cudaMemcpyAsync(ctx->d_in[b], (const char*)rf_host + (size_t)f0 * frame_in, (size_t)F * frame_in,
                                      cudaMemcpyHostToDevice, ctx->s_h2d));
        PAB_CUDA(ctx, cudaEventRecord(ctx->ev_in[b], ctx->s_h2d));
        PAB_CUDA(ctx, cudaStreamWaitEvent(ctx->s_run, ctx->ev_in[b], 0));
        if (it >= kHostSets) PAB_CUDA(ctx, cudaStreamWaitEvent(ctx->s_run, ctx->ev_out[b], 0));   // d_out[b] drained
        const int rc = run_batch(ctx, ctx->d_in[b], F, order, ctx->d_out[b], ctx->s_run);
        if (rc != PAB_OK) return rc;
        PAB_CUDA(ctx, cudaEventRecord(ctx->ev_run[b], ctx->s_run));
        PAB_CUDA(ctx, cudaStreamWaitEvent(ctx->s_d2h, ctx->ev_run[b], 0));
        PAB_CUDA(ctx, cudaMemcpyAsync((char*)out_host + (size_t)f0 * frame_out, ctx->d_out[b], (size_t)F * frame_out,
                                      cudaMemcpyDeviceToHost, ctx->s_d2h));
        PAB_CUDA(ctx, cudaEventRecord(ctx->ev_out[b], ctx->s_d2h));
    }
    return PAB_OK;
}

}  // namespace

extern "C" int pab_host_sync(pab_ctx* ctx) {
    if (!ctx) return PAB_ERR_INVALID;
    if (!ctx->s_h2d) return PAB_OK;
    PAB_CUDA(ctx, cudaStreamSynchronize(ctx->s_d2h));
    PAB_CUDA(ctx, cudaStreamSynchronize(ctx->s_run));
    return PAB_OK;
}

extern "C" int pab_beamform_host(pab_ctx* ctx, const void* rf_host, int n_frames, int order, float* out_host) {
    int rc = check_args(ctx, rf_host, n_frames, order, out_host);
    if (rc != PAB_OK) return rc;
    // Host path batches: short calls are cut into 8-frame pieces so that H2D, kernels and D2H of successive pieces
    // overlap inside one call (the call ends with its last piece's kernels and copy, which nothing overlaps: small pieces
    // keep that tail short); long streams use 64-frame pieces (more tiles per launch, negligible ramp).
    const int Bcap = ctx->plan.batch_frames < 64 ? ctx->plan.batch_frames : 64;
    int B = (n_frames >= 256 || Bcap < 8) ? Bcap : 8;
    if (ctx->tuning.host_batch_frames > 0) B = ctx->tuning.host_batch_frames < Bcap ? ctx->tuning.host_batch_frames : Bcap;
    // The first and the last piece are half pieces (when there are enough frames): the pipeline starts computing and
    // starts its last device-to-host copy sooner.
    rc = host_enqueue(ctx, rf_host, n_frames, order, out_host, B, B >= 8 && n_frames >= 4 * B);
    const int rs = pab_host_sync(ctx);           // also after a failed enqueue: nothing of this call stays in flight
    return rc != PAB_OK ? rc : rs;
}

// The streaming form: successive calls overlap each other (the copies of call i + 1 and of call i - 1 run beside the
// kernels of call i), so a call needs no small pieces to hide its own ramp: whole 64-frame pieces, the most efficient launch.
extern "C" int pab_beamform_host_async(pab_ctx* ctx, const void* rf_host, int n_frames, int order, float* out_host) {
    int rc = check_args(ctx, rf_host, n_frames, order, out_host);
    if (rc != PAB_OK) return rc;
    const int Bcap = ctx->plan.batch_frames < 64 ? ctx->plan.batch_frames : 64;
    int B = Bcap;
    if (ctx->tuning.host_batch_frames > 0) B = ctx->tuning.host_batch_frames < Bcap ? ctx->tuning.host_batch_frames : Bcap;
    return host_enqueue(ctx, rf_host, n_frames, order, out_host, B, false);
}
