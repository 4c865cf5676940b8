// rollout_tc.cu -- tcgen05 / TMEM path (placeholder until the tensor-core kernels land).
#include "voila_kernels.h"

namespace voila {

bool tc_supported(const voila_model_desc *, std::string *why) {
    if (why) *why = "tcgen05 path not built yet";
    return false;
}
void *tc_create(const voila_model_desc *, int, std::vector<void *> *, std::string *) { return nullptr; }
void tc_destroy(void *) {}
cudaError_t launch_rollout_tc(void *, const ModelDev &, const RolloutArgs &, cudaStream_t, std::string *,
                              int *) {
    return cudaErrorNotSupported;
}
cudaError_t launch_bu_propose_score_tc(void *, const ModelDev &, const BeliefArgs &, cudaStream_t, int *) {
    return cudaErrorNotSupported;
}

}  // namespace voila
