// pab_tu_cached.cu -- translation unit: the cached-tap beamforming kernel and its table builders.
#include "pab_cache.cuh"
#include "pab_launch.h"

namespace pab {

cudaError_t xl_cached_configure(int smem_optin) { return cached_configure(smem_optin); }
bool xl_cached_fits(const pab_plan_info& plan, int nq, bool compact, int smem_limit) { return cached_fits(plan, nq, compact, smem_limit); }
bool xl_cached_weight_ok(int order, int nq, bool compact) { return cached_weight_ok(order, nq, compact); }
void xl_cached(int order, int nq, int weight, const BfParams& P, int groups, const pab_plan_info& plan, int chunk_cap,
               int smem_limit, int sm_count, const CacheTables& T, cudaStream_t st) {
    launch_cached(order, nq, weight, P, groups, plan, chunk_cap, smem_limit, sm_count, T, st);
}
void xl_build_delay_cache(const CacheGeom& G, int tiles_z, uint32_t* taps, int* w0s) {          // tiles_z = ceil(nz / G.tile_rows)
    delay_cache_kernel<<<dim3(G.tiles_x, tiles_z, G.N), kStgRows * kStgCols>>>(G, taps, w0s);
}
void xl_build_delay_compact(const CacheGeom& G, int q, int nd, uint2* compact) {
    delay_compact_kernel<<<dim3((G.nz + 255) / 256, nd), 256>>>(G, q, compact);
}

}  // namespace pab
