// pab_launch.h -- host entry points of the kernel translation units (csrc/pab_tu_*.cu), called by pab_api.cu.
// libpab.so is compiled as several translation units in parallel (build.py); each kernel family is instantiated
// in exactly one of them, behind these plain functions.
#pragma once
#include "pab_types.h"

namespace pab {

// ---- pab_tu_direct.cu: ingest (a1) and the direct beamforming kernel ----
void xl_ingest_quad(int dtype, const void* rf, float* stage, int F, int N, int S, float scale, cudaStream_t st);
void xl_ingest_lin(int dtype, const void* rf, float* stage, int F, int N, int S, int Sp, float scale, cudaStream_t st);
void xl_direct(int order, int nq, int weight, const BfParams& P, int groups, cudaStream_t st);

// ---- pab_tu_staged.cu: the staged kernel with in-kernel delays ----
int xl_staged_configure(int smem_optin);
void xl_staged(int order, int nq, bool in_range, int weight, const BfParams& P, int groups, const pab_plan_info& plan,
               int chunk_cap, int smem_limit, int sm_count, cudaStream_t st);

// ---- pab_tu_cached.cu: cached interpolation taps ----
cudaError_t xl_cached_configure(int smem_optin);
bool xl_cached_fits(const pab_plan_info& plan, int nq, bool compact, int smem_limit);
bool xl_cached_weight_ok(int order, int nq, bool compact);
void xl_cached(int order, int nq, int weight, const BfParams& P, int groups, const pab_plan_info& plan, int chunk_cap,
               int smem_limit, int sm_count, const CacheTables& T, cudaStream_t st);
void xl_build_delay_cache(const CacheGeom& G, int tiles_z, uint32_t* taps, int* w0s);
void xl_build_delay_compact(const CacheGeom& G, int q, int nd, uint2* compact);

// ---- pab_tu_diag.cu: single frames on translation-invariant geometries ----
cudaError_t xl_diag_configure(int smem_optin);
cudaError_t xl_diag_build(int N, int S, double fs, double c, const pab_grid& g, int q, int npg, int max_order, int smem_limit,
                          int mode, DiagSet* D);      // mode 0: tap table, 1: table-free (windows only), 2: nearest-sample table
void xl_diag_free(DiagSet* D);
cudaError_t xl_diag_check(int order, const DiagSet& D, const float* rf, float* out, int N, int S, int nx, int nz, int* d_viol,
                          cudaStream_t st);
void xl_diag(int order, int dtype, int weight, const DiagSet& D, const void* rf, float* out, int F, int N, int S, int nx, int nz,
             float scale, cudaStream_t st);

// ---- pab_tu_nearest.cu: row f4 ----
cudaError_t xl_nearest_configure(int smem_optin);
bool xl_nearest_table(const NearestGeom& G, unsigned short* table);      // false: grid too large
void xl_ingest_root_quad(int dtype, int order, const void* rf, float* stage, int F, int N, int S, float scale, cudaStream_t st);
bool xl_nearest_staged_fits(const pab_plan_info& plan, int nq, int stages, int smem_limit);
void xl_nearest_staged(int order, int nq, bool in_range, const BfParams& P, int groups, const pab_plan_info& plan, int stages,
                       int chunk_cap, int smem_limit, int sm_count, const unsigned short* table, cudaStream_t st);
void xl_nearest_direct(int order, int nq, const BfParams& P, int groups, const unsigned short* table, cudaStream_t st);

// ---- pab_tu_post.cu: post chain (a7..a9) and image metrics (row f3) ----
cudaError_t xl_post_configure(int smem_optin);
void xl_post64(const PostParams& Q, const PostTaps64& T, bool env, int hpar, int F, cudaStream_t st);
void xl_post_generic(const PostParams& Q, bool env, int F, cudaStream_t st);
// no-allocation post chain (pab_post_no_alloc): frame maxima in a file-scope device array of pab_tu_post.cu
cudaError_t xl_post_no_alloc_setup(unsigned int** ptr_out);
cudaError_t xl_post_no_alloc(PostParams Q, const PostTaps64& T, int hpar, int F, bool log, float dr, cudaStream_t st, int* launches);
void xl_post_log(float* out, const unsigned int* frame_max, int npix, int F, float dr, cudaStream_t st);
int xl_metrics(const float* img, int nx, const RoiPair& R, MetricAcc* acc, unsigned int* hist, int n_bins, int fwhm_row,
               double* fw, cudaStream_t st);        // returns the number of kernels launched

}  // namespace pab
