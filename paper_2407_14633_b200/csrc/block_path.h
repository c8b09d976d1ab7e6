// Block (real-space, n x n) path: Sancho-Rubio self-energies + block RGF sweeps (configs[2..4]).
#pragma once
#include <cuda_runtime.h>

#include "negf.h"

namespace negf {

struct BlockPath;

struct ProfHook {                 // optional per-kernel timing callbacks (kinds: 0 SR, 1 sweep, 2 reduce)
  void* ctx;
  void (*begin)(void* ctx, int kind);
  void (*end)(void* ctx);
};

negf_status block_path_create(const negf_config* cfg, const double2* z_eq_dev, const double2* w_eq_dev,
                              const double2* z_neq_dev, const double* w_neq_dev, BlockPath** out);
negf_status block_path_self_energy(BlockPath* bp, const double* U_dev, cudaStream_t s, ProfHook hook);
negf_status block_path_run(BlockPath* bp, const double* U_dev, double* n_res, double* T_res,
                           cudaStream_t s, ProfHook hook);
negf_status block_path_check(BlockPath* bp);
void block_path_plan(BlockPath* bp, negf_plan_info* out);
void block_path_destroy(BlockPath* bp);

}  // namespace negf
