// pab_tu_staged.cu -- translation unit: the staged beamforming kernel with in-kernel delays, in-range geometries
// (no out-of-record masks); pab_tu_staged_gen.cu holds the general instantiations.
#include "pab_staged.cuh"
#include "pab_launch.h"

namespace pab {

bool xl_staged_gen_configure(int smem_optin);
void xl_staged_gen(int order, int nq, int weight, const BfParams& P, int groups, const pab_plan_info& plan, int chunk_cap,
                   int smem_limit, int sm_count, cudaStream_t st);

int xl_staged_configure(int smem_optin) {
    return staged_configure_inr<true>(smem_optin) && xl_staged_gen_configure(smem_optin) ? PAB_OK : PAB_ERR_CUDA;
}
void xl_staged(int order, int nq, bool in_range, int weight, const BfParams& P, int groups, const pab_plan_info& plan,
               int chunk_cap, int smem_limit, int sm_count, cudaStream_t st) {
    if (in_range) launch_staged_t<true>(order, nq, weight, P, groups, plan, chunk_cap, smem_limit, sm_count, st);
    else xl_staged_gen(order, nq, weight, P, groups, plan, chunk_cap, smem_limit, sm_count, st);
}

}  // namespace pab
