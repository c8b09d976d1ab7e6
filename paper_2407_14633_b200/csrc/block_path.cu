// Placeholder until the block kernels land: fails loudly (no CPU fallback, no silent success).
#include "block_path.h"
#include "negf_internal.h"

namespace negf {
struct BlockPath { int dummy; };
negf_status block_path_create(const negf_config*, const double2*, const double2*, const double2*,
                              const double*, BlockPath** out) {
  *out = nullptr;
  set_error("block > 1 path is not built in this version of libnegf_b200");
  return NEGF_EINVAL;
}
negf_status block_path_self_energy(BlockPath*, const double*, cudaStream_t, ProfHook) { return NEGF_EINVAL; }
negf_status block_path_run(BlockPath*, const double*, double*, double*, cudaStream_t, ProfHook) { return NEGF_EINVAL; }
negf_status block_path_check(BlockPath*) { return NEGF_OK; }
void block_path_plan(BlockPath*, negf_plan_info*) {}
void block_path_destroy(BlockPath*) {}
}  // namespace negf
