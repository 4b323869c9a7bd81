// pab_tu_direct.cu -- translation unit: ingest kernels (a1) and the direct beamforming kernel.
#include "pab_kernels.cuh"
#include "pab_launch.h"

namespace pab {

void xl_ingest_quad(int dtype, const void* rf, float* stage, int F, int N, int S, float scale, cudaStream_t st) {
    if (dtype == PAB_I16) launch_ingest_quad<int16_t>(rf, stage, F, N, S, scale, st);
    else launch_ingest_quad<float>(rf, stage, F, N, S, scale, st);
}
void xl_ingest_lin(int dtype, const void* rf, float* stage, int F, int N, int S, int Sp, float scale, cudaStream_t st) {
    if (dtype == PAB_I16) launch_ingest_lin<int16_t>(rf, stage, F, N, S, Sp, scale, st);
    else launch_ingest_lin<float>(rf, stage, F, N, S, Sp, scale, st);
}
void xl_direct(int order, int nq, int weight, const BfParams& P, int groups, cudaStream_t st) {
    launch_direct_nq(order, nq, weight, P, groups, st);
}

}  // namespace pab
