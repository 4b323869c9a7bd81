// pab_tu_staged_gen.cu -- translation unit: the staged beamforming kernel, general geometries (pixels whose delay
// falls outside the record are masked, reading A6).
#include "pab_staged.cuh"

namespace pab {

bool xl_staged_gen_configure(int smem_optin) { return staged_configure_inr<false>(smem_optin); }
void xl_staged_gen(int order, int nq, int weight, const BfParams& P, int groups, const pab_plan_info& plan, int chunk_cap,
                   int smem_limit, int sm_count, cudaStream_t st) {
    launch_staged_t<false>(order, nq, weight, P, groups, plan, chunk_cap, smem_limit, sm_count, st);
}

}  // namespace pab
