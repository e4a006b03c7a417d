// farm_sim_tc.cu -- step 4 on the 5th-generation tensor cores (placeholder until the tcgen05 kernel lands).
#include "farm_internal.cuh"
namespace farm {
bool tc_supported(const DevMap &) { return false; }
void *tc_state_create(const DevMap &) { return nullptr; }
void tc_state_destroy(void *) {}
int launch_similarity_tc(const DevMap &, const CallArgs &, uint32_t, cudaStream_t, void *) { return 0; }
}  // namespace farm
