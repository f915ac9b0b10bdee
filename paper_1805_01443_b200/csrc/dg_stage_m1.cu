// Stage-kernel variants of DG order 1, local Lax-Friedrichs flux (see dg_stage_launch.cuh).
#include "dg_stage_launch.cuh"
namespace dg {
cudaError_t launch_stage_m1(const StageArgs& A, int eos, int grav, int kind, dim3 grid, cudaStream_t s) {
  return launch_stage_order<1, 0>(A, eos, grav, kind, grid, s);
}
}  // namespace dg
