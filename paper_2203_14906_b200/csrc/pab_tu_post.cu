// pab_tu_post.cu -- translation unit: post chain (a7..a9) and image metrics (row f3).
#include "pab_post.cuh"
#include "pab_metrics.cuh"
#include "pab_launch.h"

namespace pab {

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
