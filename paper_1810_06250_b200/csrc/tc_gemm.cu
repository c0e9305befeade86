// placeholder until the tcgen05 kernel lands (next commit)
#include "common.cuh"
namespace rms {
rmsynth_status tc_plan_init(rmsynth_plan*) { return RMSYNTH_OK; }
void tc_plan_free(rmsynth_plan*) {}
rmsynth_status tc_execute(const rmsynth_plan*, const float*, const float*, long long, int, float*, float*, float*,
                          float*, float*, float*, int*, cudaStream_t) {
    return fail(RMSYNTH_EUNSUPPORTED, "tensor-core path not built yet");
}
}  // namespace rms
