// Launch dispatch of the stage kernel for one DG order M: one translation unit per order
// (dg_stage_m1.cu ... dg_stage_m5.cu) and numerical flux, so that the 35 variants of each compile in parallel.
#pragma once
#include <cuda_runtime.h>

#include <atomic>

#include "dg_tables.h"
#include "dg_kernels.cuh"
#include "dg_stage_fh.cuh"
#include "dg_stage_m1fv.cuh"

namespace dg {

// Thread blocks per SM the register allocation aims at (order 3: 4 blocks of 160 registers beat 5 of 128, which spill);
// shared memory (4 tiles + tables per block)
// allows exactly this many on a 227 KB SM for M = 5, 4 and is not the limit below.
template <int M> struct StageMinBlocks;
template <> struct StageMinBlocks<1> { static constexpr int value = 16; };
template <> struct StageMinBlocks<2> { static constexpr int value = 8; };
template <> struct StageMinBlocks<3> { static constexpr int value = 4; };
template <> struct StageMinBlocks<4> { static constexpr int value = 3; };
template <> struct StageMinBlocks<5> { static constexpr int value = 2; };

// Orders whose default stage kernel is the one with the face-helper warp (dg_stage_fh.cuh).  Order 5: M worker warps
// of 168 registers leave the schedulers unevenly filled.  Order 3: 4 blocks of 3 + 1 warps at 128 registers, 4 % faster
// than 4 blocks of 3 warps at 160, and another 4 % since the workers evaluate the segment's first S face themselves.
// Order 4: 3 blocks of 4 + 1 warps at 136 registers (24-40 B of spills), +2 % at 1024^2 and +0.4 % at 2048^2 (A/B in
// one process).  Order 2 with a third warp (6 blocks, 96 registers) is 17-25 % slower and keeps dg::stage_kernel.
template <int M> struct StageFaceHelper { static constexpr bool value = M >= 3; };

constexpr int kMaxDevices = 64;

template <int M, int EOS, int GRAV, int KIND, int FLUX>
cudaError_t launch_stage_variant_fh(const StageArgs& A, dim3 grid, cudaStream_t stream) {
  static std::atomic<bool> attr_set[kMaxDevices];
  constexpr size_t smem = stage_fh_smem_bytes<M>();
  auto kern = stage_kernel_fh<M, EOS, GRAV, KIND, StageMinBlocks<M>::value, FLUX>;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  const bool cached = dev >= 0 && dev < kMaxDevices;
  if (!cached || !attr_set[dev].load(std::memory_order_acquire)) {
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (cached) attr_set[dev].store(true, std::memory_order_release);
  }
  kern<<<grid, (M + 1) * 32, smem, stream>>>(A);
  return cudaGetLastError();
}

template <int M, int EOS, int GRAV, int KIND, int FLUX>
cudaError_t launch_stage_variant(const StageArgs& A, dim3 grid, cudaStream_t stream) {
  if constexpr (M == 1) {                        // order 1: the register-only kernel (dg_stage_m1fv.cuh), one warp per segment of rows
    if (A.impl != 1) {
      stage_kernel_m1<EOS, GRAV, KIND, FLUX><<<dim3((A.g.nx + M1_OWN - 1) / M1_OWN, (grid.y + M1_WARPS - 1) / M1_WARPS), M1_WARPS * 32, 0, stream>>>(A);
      return cudaGetLastError();
    }
  }
  // (the sub-steps of the general schemes, K_GEN, gather up to five more arrays in the epilogue and run faster on the
  // M-warp kernel: Cash-Karp with the limiter 6.7 ms per 1024^2 order-5 step against 8.2)
  if constexpr (StageFaceHelper<M>::value) {
    if (A.impl == 2 || (A.impl == 0 && KIND != K_GEN)) return launch_stage_variant_fh<M, EOS, GRAV, KIND, FLUX>(A, grid, stream);
  }
  // dynamic shared memory above 48 KB is opted in once per device (the attribute belongs to the device's context):
  // one flag per device ordinal, set after the call succeeded; racing threads at worst both make the (idempotent) call
  static std::atomic<bool> attr_set[kMaxDevices];
  constexpr size_t smem = stage_smem_bytes<M>();
  auto kern = stage_kernel<M, EOS, GRAV, KIND, StageMinBlocks<M>::value, FLUX>;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  const bool cached = dev >= 0 && dev < kMaxDevices;
  if (!cached || !attr_set[dev].load(std::memory_order_acquire)) {
    e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (cached) attr_set[dev].store(true, std::memory_order_release);
  }
  kern<<<grid, StageWarps<M, KIND>::threads, smem, stream>>>(A);
  return cudaGetLastError();
}

template <int M, int EOS, int GRAV, int FLUX>
cudaError_t launch_stage_kind(const StageArgs& A, int kind, dim3 grid, cudaStream_t s) {
  switch (kind) {
    case K_RHS:   return launch_stage_variant<M, EOS, GRAV, K_RHS, FLUX>(A, grid, s);
    case K_FIRST: return launch_stage_variant<M, EOS, GRAV, K_FIRST, FLUX>(A, grid, s);
    case K_MID:   return launch_stage_variant<M, EOS, GRAV, K_MID, FLUX>(A, grid, s);
    case K_LAST:  return launch_stage_variant<M, EOS, GRAV, K_LAST, FLUX>(A, grid, s);
    case K_LASTD: return launch_stage_variant<M, EOS, GRAV, K_LASTD, FLUX>(A, grid, s);
    case K_GEN:   return launch_stage_variant<M, EOS, GRAV, K_GEN, FLUX>(A, grid, s);
    default:      return launch_stage_variant<M, EOS, GRAV, K_GENL, FLUX>(A, grid, s);
  }
}

template <int M, int FLUX>
cudaError_t launch_stage_order(const StageArgs& A, int eos, int grav, int kind, dim3 grid, cudaStream_t s) {
  if (eos == 0) {
    switch (grav) {
      case G_NONE: return launch_stage_kind<M, 0, G_NONE, FLUX>(A, kind, grid, s);
      case G_STAR: return launch_stage_kind<M, 0, G_STAR, FLUX>(A, kind, grid, s);
      default:     return launch_stage_kind<M, 0, G_PLANET, FLUX>(A, kind, grid, s);
    }
  }
  // the locally isothermal closure is defined through the star (c_s^2 ~ GM/r): gravity is always on
  if (grav == G_PLANET) return launch_stage_kind<M, 1, G_PLANET, FLUX>(A, kind, grid, s);
  return launch_stage_kind<M, 1, G_STAR, FLUX>(A, kind, grid, s);
}

// one definition per order and numerical flux (0: local Lax-Friedrichs, 1: HLLC / HLL), in dg_stage_m<M>.cu
// and dg_stage_m<M>f.cu
#define DG_DECLARE_STAGE(name) \
  cudaError_t name(const StageArgs&, int eos, int grav, int kind, dim3 grid, cudaStream_t)
DG_DECLARE_STAGE(launch_stage_m1); DG_DECLARE_STAGE(launch_stage_m2); DG_DECLARE_STAGE(launch_stage_m3);
DG_DECLARE_STAGE(launch_stage_m4); DG_DECLARE_STAGE(launch_stage_m5);
DG_DECLARE_STAGE(launch_stage_m1f); DG_DECLARE_STAGE(launch_stage_m2f); DG_DECLARE_STAGE(launch_stage_m3f);
DG_DECLARE_STAGE(launch_stage_m4f); DG_DECLARE_STAGE(launch_stage_m5f);
#undef DG_DECLARE_STAGE

}  // namespace dg
