// dg_torque_static (include/dg.h): the torque of Eq.(6), for callers that may not allocate device
// memory at all -- code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc.  No context, no
// workspace: the caller passes the modal state and the output, both DEVICE; the only scratch the computation needs, the
// per-block partial sums of the reduction, lives in a file-scope __device__ array of fixed size.
//
// Same operation as torque_kernel / torque_finish_kernel (dg_limit.cuh) behind dg_torque, which read the context's
// nodal state and keep their partial sums in the caller's workspace.  This variant reads the cell average straight
// from the external layout (mode (0,0) of the orthonormal basis IS the cell average), so it needs no
// basis tables either.  Sums are taken in a fixed order: the result does not depend on scheduling.
//
// The scratch array:
//   * 2 doubles per thread block, DG_STATIC_MAX_BLOCKS blocks = 1 MiB of device memory on every GPU that loads the
//     library, from the load to the end of the process;
//   * its name is a host-side stand-in in host code, not a device address: the address the kernels get comes from
//     cudaGetSymbolAddress, taken once per device with that device current (static_setup below);
//   * shared by every call on a device and never cleared: a call overwrites exactly the 2 x nblocks slots its own
//     finish kernel reads, so nothing has to start at zero -- but two calls that overlap on the GPU (different streams,
//     no ordering between them) race on it.  Order them.
#include <cuda_runtime.h>

#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>

#include "../../include/dg.h"

namespace {

constexpr int kMaxBlocks = DG_STATIC_MAX_BLOCKS;
constexpr int kTile = 32;                        // a thread block covers 32 x 32 cells
constexpr int kWarps = 8;
constexpr int kMaxDevices = 64;
constexpr unsigned FULL = 0xffffffffu;

static __device__ __align__(256) double g_static_scratch[2 * kMaxBlocks];

std::atomic<double*> g_scratch_ptr[kMaxDevices];  // device address of g_static_scratch on each device ordinal

thread_local char g_err[256] = "";

int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof g_err, fmt, ap);
  va_end(ap);
  return code;
}

// Device address of the scratch array on the current device: looked up once per device, then cached.
int static_setup(double** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail(DG_ECUDA, "dg_static_setup: cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= kMaxDevices) return fail(DG_EINVAL, "dg_static_setup: device ordinal %d beyond %d", dev, kMaxDevices - 1);
  double* p = g_scratch_ptr[dev].load(std::memory_order_acquire);
  if (!p) {
    e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_static_scratch);
    if (e != cudaSuccess || !p)
      return fail(DG_ECUDA, "dg_static_setup: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
    g_scratch_ptr[dev].store(p, std::memory_order_release);   // (racing threads store the same address)
  }
  if (out) *out = p;
  return DG_OK;
}

// One thread block per 32 x 32 cells: warp w takes rows w, w + 8, w + 16, w + 24 of the block, lane = cell along x.
// U is the external layout [ny][nx][4][m][m]; the density's cell average is coefficient 0 of the cell's cdof doubles.
// Per cell: M_n = average density x area, a += G M_n (r_n - r_p) / (|r_n - r_p|^2 + eps_p^2)^(3/2).
__global__ void __launch_bounds__(kWarps * 32)
torque_static_kernel(const double* __restrict__ U, double* __restrict__ partial, int nx, int ny, int cdof,
                     double x0, double y0, double dx, double dy, double gm, double xp, double yp, double eps2p) {
  __shared__ double sx[kWarps], sy[kWarps];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int i = blockIdx.x * kTile + lane;
  double ax = 0.0, ay = 0.0;
#pragma unroll
  for (int k = 0; k < kTile / kWarps; ++k) {
    const int j = blockIdx.y * kTile + k * kWarps + w;
    if (j < ny && i < nx) {
      const double rho = __ldg(U + ((size_t)j * nx + i) * cdof);
      const double Mn = rho * dx * dy;
      const double ddx = x0 + (i + 0.5) * dx - xp, ddy = y0 + (j + 0.5) * dy - yp;
      const double r2 = fma(ddx, ddx, fma(ddy, ddy, eps2p));
      const double f = gm * Mn / (r2 * sqrt(r2));
      ax = fma(f, ddx, ax);
      ay = fma(f, ddy, ay);
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    ax += __shfl_xor_sync(FULL, ax, o);
    ay += __shfl_xor_sync(FULL, ay, o);
  }
  if (lane == 0) { sx[w] = ax; sy[w] = ay; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double tx = 0.0, ty = 0.0;
#pragma unroll
    for (int k = 0; k < kWarps; ++k) { tx += sx[k]; ty += sy[k]; }
    const size_t b = (size_t)blockIdx.y * gridDim.x + blockIdx.x;
    partial[2 * b] = tx;
    partial[2 * b + 1] = ty;
  }
}

// out[0] = Gamma_z = x_p a_y - y_p a_x, out[1] = a_x, out[2] = a_y
__global__ void __launch_bounds__(256)
torque_static_finish_kernel(const double* __restrict__ partial, int nblocks, double xp, double yp, double* __restrict__ out) {
  __shared__ double sx[256], sy[256];
  double ax = 0.0, ay = 0.0;
  for (int b = threadIdx.x; b < nblocks; b += 256) { ax += partial[2 * b]; ay += partial[2 * b + 1]; }
  sx[threadIdx.x] = ax;
  sy[threadIdx.x] = ay;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) { sx[threadIdx.x] += sx[threadIdx.x + o]; sy[threadIdx.x] += sy[threadIdx.x + o]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    out[0] = xp * sy[0] - yp * sx[0];
    out[1] = sx[0];
    out[2] = sy[0];
  }
}

}  // namespace

extern "C" {

int dg_static_setup(void) { return static_setup(nullptr); }

const char* dg_static_last_error(void) { return g_err; }

int dg_torque_static(const dg_params* p, const double* U, double t, double* out, void* cuda_stream) {
  if (!p || !U || !out) return fail(DG_EINVAL, "dg_torque_static: null argument");
  if (reinterpret_cast<uintptr_t>(U) % sizeof(double) || reinterpret_cast<uintptr_t>(out) % sizeof(double))
    return fail(DG_EINVAL, "dg_torque_static: U and out must be 8-byte aligned");
  if (p->nx < 1 || p->ny < 1 || p->order < 1 || p->order > 5 || !(p->x1 > p->x0) || !(p->y1 > p->y0) || !std::isfinite(t))
    return fail(DG_EINVAL, "dg_torque_static: bad parameters (nx %d, ny %d, order %d)", p->nx, p->ny, p->order);
  const long long bx = (p->nx + kTile - 1) / kTile, by = (p->ny + kTile - 1) / kTile;
  if (bx * by > kMaxBlocks)
    return fail(DG_ENOSPC, "dg_torque_static: %d x %d cells need %lld blocks of 32 x 32 cells, the static scratch holds "
                "DG_STATIC_MAX_BLOCKS = %d (use dg_torque, whose scratch is in the caller's workspace)",
                p->nx, p->ny, bx * by, kMaxBlocks);
  double* scratch = nullptr;
  int e = static_setup(&scratch);
  if (e) return e;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const double ang = p->omega_planet * t + p->phase0;        // the planet's fixed circular orbit
  const double xp = p->r_planet * std::cos(ang), yp = p->r_planet * std::sin(ang);
  const double dx = (p->x1 - p->x0) / p->nx, dy = (p->y1 - p->y0) / p->ny;
  const dim3 grid((unsigned)bx, (unsigned)by);
  torque_static_kernel<<<grid, kWarps * 32, 0, s>>>(U, scratch, p->nx, p->ny, 4 * p->order * p->order, p->x0, p->y0, dx, dy,
                                                    p->gm_star, xp, yp, p->eps_planet * p->eps_planet);
  torque_static_finish_kernel<<<1, 256, 0, s>>>(scratch, (int)(bx * by), xp, yp, out);
  const cudaError_t ce = cudaGetLastError();
  if (ce != cudaSuccess) return fail(DG_ECUDA, "dg_torque_static: launch: %s", cudaGetErrorString(ce));
  return DG_OK;
}

}  // extern "C"
