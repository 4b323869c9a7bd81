// pab_tu_nearest.cu -- translation unit: row f4, nearest-sample delays (the literal eq. 1).
#include "pab_nearest.cuh"
#include "pab_launch.h"

namespace pab {

cudaError_t xl_nearest_configure(int smem_optin) { return nearest_configure(smem_optin); }
bool xl_nearest_table(const NearestGeom& G, unsigned short* table) {
    const int tiles_x = (G.nx + kStgCols - 1) / kStgCols, tiles_z = (G.nz + kStgRows - 1) / kStgRows;
    dim3 grid((tiles_z * kStgRows + 255) / 256, tiles_x * kStgCols, G.N);
    if (grid.y > 65535u || grid.z > 65535u) return false;
    nearest_table_kernel<<<grid, 256>>>(G, table);
    return true;
}
void xl_ingest_root_quad(int dtype, int order, const void* rf, float* stage, int F, int N, int S, float scale, cudaStream_t st) {
    if (dtype == PAB_I16) launch_ingest_root_quad<int16_t>(order, rf, stage, F, N, S, scale, st);
    else launch_ingest_root_quad<float>(order, rf, stage, F, N, S, scale, st);
}
bool xl_nearest_staged_fits(const pab_plan_info& plan, int nq, int stages, int smem_limit) {
    return nearest_staged_fits(plan, nq, stages, smem_limit);
}
void xl_nearest_staged(int order, int nq, bool in_range, const BfParams& P, int groups, const pab_plan_info& plan, int stages,
                       int chunk_cap, int smem_limit, int sm_count, const unsigned short* table, cudaStream_t st) {
    launch_nearest_staged(order, nq, in_range, P, groups, plan, stages, chunk_cap, smem_limit, sm_count, table, st);
}
void xl_nearest_direct(int order, int nq, const BfParams& P, int groups, const unsigned short* table, cudaStream_t st) {
    launch_nearest_direct(order, nq, P, groups, table, st);
}

}  // namespace pab
