// Launch dispatch of the stage kernel for one DG order M: one translation unit per order
// (dg_stage_m1.cu ... dg_stage_m5.cu) so that the 35 variants per order compile in parallel.
#pragma once
#include <cuda_runtime.h>

#include "dg_tables.h"
#include "dg_kernels.cuh"

namespace dg {

// Thread blocks per SM the register allocation aims at; shared memory (4 tiles + tables per block)
// allows exactly this many on a 227 KB SM for M = 5, 4 and is not the limit below.
template <int M> struct StageMinBlocks;
template <> struct StageMinBlocks<1> { static constexpr int value = 16; };
template <> struct StageMinBlocks<2> { static constexpr int value = 8; };
template <> struct StageMinBlocks<3> { static constexpr int value = 5; };
template <> struct StageMinBlocks<4> { static constexpr int value = 3; };
template <> struct StageMinBlocks<5> { static constexpr int value = 2; };

template <int M, int EOS, int GRAV, int KIND>
cudaError_t launch_stage_variant(const StageArgs& A, dim3 grid, cudaStream_t stream) {
  static bool attr_set = false;      // dynamic shared memory above 48 KB must be opted in once
  constexpr size_t smem = stage_smem_bytes<M>();
  auto kern = stage_kernel<M, EOS, GRAV, KIND, StageMinBlocks<M>::value>;
  if (!attr_set) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    attr_set = true;
  }
  kern<<<grid, M * 32, smem, stream>>>(A);
  return cudaGetLastError();
}

template <int M, int EOS, int GRAV>
cudaError_t launch_stage_kind(const StageArgs& A, int kind, dim3 grid, cudaStream_t s) {
  switch (kind) {
    case K_RHS:   return launch_stage_variant<M, EOS, GRAV, K_RHS>(A, grid, s);
    case K_FIRST: return launch_stage_variant<M, EOS, GRAV, K_FIRST>(A, grid, s);
    case K_MID:   return launch_stage_variant<M, EOS, GRAV, K_MID>(A, grid, s);
    case K_LAST:  return launch_stage_variant<M, EOS, GRAV, K_LAST>(A, grid, s);
    case K_LASTD: return launch_stage_variant<M, EOS, GRAV, K_LASTD>(A, grid, s);
    case K_GEN:   return launch_stage_variant<M, EOS, GRAV, K_GEN>(A, grid, s);
    default:      return launch_stage_variant<M, EOS, GRAV, K_GENL>(A, grid, s);
  }
}

template <int M>
cudaError_t launch_stage_order(const StageArgs& A, int eos, int grav, int kind, dim3 grid, cudaStream_t s) {
  if (eos == 0) {
    switch (grav) {
      case G_NONE: return launch_stage_kind<M, 0, G_NONE>(A, kind, grid, s);
      case G_STAR: return launch_stage_kind<M, 0, G_STAR>(A, kind, grid, s);
      default:     return launch_stage_kind<M, 0, G_PLANET>(A, kind, grid, s);
    }
  }
  // the locally isothermal closure is defined through the star (c_s^2 ~ GM/r): gravity is always on
  if (grav == G_PLANET) return launch_stage_kind<M, 1, G_PLANET>(A, kind, grid, s);
  return launch_stage_kind<M, 1, G_STAR>(A, kind, grid, s);
}

// one definition per order, in dg_stage_m<M>.cu
cudaError_t launch_stage_m1(const StageArgs&, int eos, int grav, int kind, dim3 grid, cudaStream_t);
cudaError_t launch_stage_m2(const StageArgs&, int eos, int grav, int kind, dim3 grid, cudaStream_t);
cudaError_t launch_stage_m3(const StageArgs&, int eos, int grav, int kind, dim3 grid, cudaStream_t);
cudaError_t launch_stage_m4(const StageArgs&, int eos, int grav, int kind, dim3 grid, cudaStream_t);
cudaError_t launch_stage_m5(const StageArgs&, int eos, int grav, int kind, dim3 grid, cudaStream_t);

}  // namespace dg
