// pab_tu_post.cu -- translation unit: post chain (a7..a9) and image metrics (row f3).
#include <mutex>
#include "pab_post.cuh"
#include "pab_metrics.cuh"
#include "pab_launch.h"

// Scratch of pab_post_no_alloc: the per-frame envelope maxima (a8 -> a9) live in this fixed array instead of a buffer
// from cudaMalloc.  Every GPU that loads libpab.so holds its 4 KiB until the process exits.  Every call on a device shares
// it (it keeps the last call's values: the entry point clears the frames it uses on its stream before the FIR kernel),
// so two calls that overlap on one GPU race.  In host code the name is a stand-in, not a device address: the kernels get
// the address cudaGetSymbolAddress returns for the current device (xl_post_no_alloc_setup).
static __device__ __align__(256) unsigned int pab_no_alloc_frame_max[PAB_NO_ALLOC_MAX_FRAMES];

namespace pab {

namespace {
constexpr int kNoAllocMaxDevices = 64;
std::mutex g_no_alloc_mutex;
unsigned int* g_no_alloc_ptr[kNoAllocMaxDevices];     // device address of pab_no_alloc_frame_max on device [i], once resolved
}  // namespace

// Once per device, with that device current (pab_create calls it; idempotent): resolves the scratch array's address.
cudaError_t xl_post_no_alloc_setup(unsigned int** ptr_out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kNoAllocMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_no_alloc_mutex);
    if (!g_no_alloc_ptr[dev]) {
        unsigned int* p = nullptr;
        if ((e = cudaGetSymbolAddress((void**)&p, pab_no_alloc_frame_max)) != cudaSuccess) return e;
        g_no_alloc_ptr[dev] = p;
    }
    if (ptr_out) *ptr_out = g_no_alloc_ptr[dev];
    return cudaSuccess;
}

// Band-pass + envelope (+ log) of F <= PAB_NO_ALLOC_MAX_FRAMES frames with the frame maxima in the fixed array.  Q.frame_max
// is ignored.  No allocation: a memset and two (one) launches on st.  Returns the number of kernels through *launches.
cudaError_t xl_post_no_alloc(PostParams Q, const PostTaps64& T, int hpar, int F, bool log, float dr, cudaStream_t st, int* launches) {
    unsigned int* fmax = nullptr;
    cudaError_t e = xl_post_no_alloc_setup(&fmax);
    if (e != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(fmax, 0, (size_t)F * sizeof(unsigned int), st)) != cudaSuccess) return e;
    Q.frame_max = fmax;
    launch_post64(Q, T, true, hpar, F, st);
    if (log) launch_post_log(Q.out, fmax, Q.nx * Q.nz, F, dr, st);
    *launches = log ? 2 : 1;
    return cudaGetLastError();
}

cudaError_t xl_post_configure(int smem_optin) {
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(post_fir_kernel<128, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(post_fir_kernel<128, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_optin)) != cudaSuccess) return e;
    return post64_configure(smem_optin);
}
void xl_post64(const PostParams& Q, const PostTaps64& T, bool env, int hpar, int F, cudaStream_t st) {
    launch_post64(Q, T, env, hpar, F, st);
}
// filters of any length (taps from shared memory): band-pass only, or band-pass + envelope
void xl_post_generic(const PostParams& Q, bool env, int F, cudaStream_t st) {
    constexpr int TZ = 128;
    dim3 grid((Q.nx + 31) / 32, (Q.nz + TZ - 1) / TZ, F);
    if (!env) {
        const size_t sm = ((size_t)(TZ + Q.TpB - 1) * 32 + Q.TpB + Q.TpH) * 4;
        post_fir_kernel<TZ, false><<<grid, 256, sm, st>>>(Q);
    } else {
        const int YR = (TZ + Q.TpH - 1 + 7) & ~7;
        const size_t sm = ((size_t)(YR + Q.TpB - 1) * 32 + (size_t)YR * 32 + Q.TpB + Q.TpH) * 4;
        post_fir_kernel<TZ, true><<<grid, 256, sm, st>>>(Q);
    }
}
void xl_post_log(float* out, const unsigned int* frame_max, int npix, int F, float dr, cudaStream_t st) {
    launch_post_log(out, frame_max, npix, F, dr, st);
}
int xl_metrics(const float* img, int nx, const RoiPair& R, MetricAcc* acc, unsigned int* hist, int n_bins, int fwhm_row,
               double* fw, cudaStream_t st) {
    dim3 grid(32, 2);
    metrics_sum_kernel<<<grid, 256, 0, st>>>(img, nx, R, acc);
    metrics_hist_kernel<<<grid, 256, 0, st>>>(img, nx, R, acc, hist, n_bins);
    if (fwhm_row < 0) return 2;
    metrics_fwhm_kernel<<<1, 32, 0, st>>>(img, nx, fwhm_row, R.t[2], R.t[3], fw);
    return 3;
}

}  // namespace pab
