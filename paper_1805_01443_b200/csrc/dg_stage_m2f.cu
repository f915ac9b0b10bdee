// Stage-kernel variants of DG order 2, HLLC / HLL flux (see dg_stage_launch.cuh).
#include "dg_stage_launch.cuh"
namespace dg {
cudaError_t launch_stage_m2f(const StageArgs& A, int eos, int grav, int kind, dim3 grid, cudaStream_t s) {
  return launch_stage_order<2, 1>(A, eos, grav, kind, grid, s);
}
}  // namespace dg
