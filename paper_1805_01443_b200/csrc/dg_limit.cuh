// sm_100a kernels of the rows SURVEY.md 8(f) marks NEXT-1 and NEXT-3:
//   limit_kernel   positivity-preserving limiter (step (iii)(d) PAPER.md:150; Zhang & Shu
//                  2010) on the lane-blocked nodal state, in place; FINAL also applies the wave-killing
//                  relaxation and reduces the CFL wave speed
//   torque_kernel  specific torque on the planet, Eq.(6)
//
// Limiter in nodal form.  The points of Zhang & Shu's set S_K are (Gauss_m in x) x (Lobatto_nh in y)
// and (Lobatto_nh in x) x (Gauss_m in y), plus the m x m Gauss points of the volume integral (the
// nodal values themselves: DESIGN.md reading L2).  Thread (warp w, lane) holds column xi_w of its cell in
// registers and reads line eta_w of the same cell from the shared-memory copy of the tile, so the
// values at its 2 nh points are two 1-D interpolations Lh[k][.] (Gauss nodes -> Lobatto nodes).
// Scaling the non-constant modes by theta is, on nodal values, u <- ubar + theta (u - ubar).
#pragma once
#include <cstdint>

#include "dg_kernels.cuh"

namespace dg {

constexpr int MAXNH = 4;

struct LimDev {
  int nh;                        // Lobatto points: smallest rule exact for degree N_p (2 nh - 3 >= N_p)
  double Lh[MAXNH][MAXM];        // Lh[k][r] = l_r(xh_k): Lagrange basis of the Gauss nodes at the Lobatto nodes
  double w[MAXM];                // Gauss weights (cell average)
};

struct LimitArgs {
  double* q;                     // state, limited in place
  const double* q0;              // initial state (FINAL with damping)
  unsigned long long* wmax;      // FINAL: CFL wave-speed maximum
  double eps;                    // floor for density and pressure
  DampArgs D;                    // FINAL: wave-killing zones (all off: no relaxation)
  int rows;
  Geom g;
  Phys ph;
  LimDev LT;
};

template <int M>
constexpr size_t limit_smem_bytes() {
  return ((size_t)4 * M * M * 32 + (size_t)4 * M * 32 + (size_t)2 * M * 32) * sizeof(double);
}

// the parameter t in [0,1] at which the segment ubar + t (s - ubar) meets the surface p = eps_p
// (ideal gas: rho p/(gamma-1) = E rho - |m|^2/2 is a quadratic g(t) = A t^2 + B t + C with
// g(0) >= 0 > g(1); the crossing is the root 2C / (sqrt(B^2 - 4AC) - B) for either sign of A)
__device__ __forceinline__ double segment_root(const double (&ub)[4], const double (&s)[4], double e1) {
  const double dr = s[0] - ub[0], dmx = s[1] - ub[1], dmy = s[2] - ub[2], dE = s[3] - ub[3];
  const double A = dE * dr - 0.5 * (dmx * dmx + dmy * dmy);
  const double B = ub[3] * dr + ub[0] * dE - (ub[1] * dmx + ub[2] * dmy) - e1 * dr;
  const double C = ub[3] * ub[0] - 0.5 * (ub[1] * ub[1] + ub[2] * ub[2]) - e1 * ub[0];
  const double disc = B * B - 4.0 * A * C;
  const double den = sqrt(fmax(disc, 0.0)) - B;
  double t = den > 0.0 ? 2.0 * C / den : 0.0;
  if (!(t >= 0.0)) t = 0.0;
  return fmin(t, 1.0);
}

template <int M, int EOS, bool FINAL>
__global__ void __launch_bounds__(M * 32)
limit_kernel(const __grid_constant__ LimitArgs A) {
  constexpr int C = 4 * M * M;
  constexpr int BS = C * 32;
  extern __shared__ __align__(16) double lsm[];
  double* tile = lsm;                            // [v][r][q][lane]
  double* sAvg = tile + BS;                      // [v][q][lane]
  double* sMin = sAvg + 4 * M * 32;              // [w][lane]  density minima
  double* sT = sMin + M * 32;                    // [w][lane]  pressure step parameters

  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int ib = blockIdx.x;
  const int i = ib * 32 + lane;
  const Geom& g = A.g;
  const LimDev& LT = A.LT;
  const bool valid = i < g.nx;
  const int j0 = blockIdx.y * A.rows, j1 = min(g.ny, j0 + A.rows);
  const size_t row_stride = (size_t)g.nbx * BS;
  const double xc = g.x0 + (i + 0.5) * g.dx;
  const bool damp_on = FINAL && A.D.on;
  double spmax = 0.0;

  auto cfl_of_row = [&](int j) {                 // warp 0: wave speed of row j from sAvg (row a10)
    double avg[4];
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      double s = 0.0;
#pragma unroll
      for (int qq = 0; qq < M; ++qq) s += sAvg[(v * M + qq) * 32 + lane];
      avg[v] = s;
    }
    double sp = 0.0;
    if (valid) {
      const double yc = g.y0 + (j + 0.5) * g.dy;
      const double rinv = 1.0 / avg[0];
      const double vx = avg[1] * rinv, vy = avg[2] * rinv;
      double c;
      if (EOS == 0) c = sqrt(A.ph.gamma * A.ph.gm1 * (avg[3] - 0.5 * (avg[1] * vx + avg[2] * vy)) * rinv);
      else          c = sqrt(A.ph.h2gm * rsqrt(fma(xc, xc, fma(yc, yc, A.ph.eps2s))));
      sp = (fabs(vx) + c) * g.inv_dx + (fabs(vy) + c) * g.inv_dy;
      if (!(sp >= 0.0)) sp = __longlong_as_double(0x7ff0000000000000LL);
    }
    spmax = fmax(spmax, sp);
  };

  double un[4][M];                               // next row's column, in flight during this row
  {
    const double* p = A.q + (size_t)j0 * row_stride + (size_t)ib * BS + lane;
#pragma unroll
    for (int v = 0; v < 4; ++v)
#pragma unroll
      for (int r = 0; r < M; ++r) un[v][r] = p[((v * M + r) * M + w) * 32];
  }

  for (int j = j0; j < j1; ++j) {
    double* p = A.q + (size_t)j * row_stride + (size_t)ib * BS + lane;
    double uc[4][M];
#pragma unroll
    for (int v = 0; v < 4; ++v)
#pragma unroll
      for (int r = 0; r < M; ++r) uc[v][r] = un[v][r];
    if (j + 1 < j1) {
      const double* pn = p + row_stride;
#pragma unroll
      for (int v = 0; v < 4; ++v)
#pragma unroll
        for (int r = 0; r < M; ++r) un[v][r] = pn[((v * M + r) * M + w) * 32];
    }
    if (FINAL && w == 0 && j > j0) cfl_of_row(j - 1);   // sAvg of the previous row (synchronised at its end)
    __syncthreads();                             // previous row's readers of tile / sAvg are done
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      double s = 0.0;
#pragma unroll
      for (int r = 0; r < M; ++r) {
        tile[((v * M + r) * M + w) * 32 + lane] = uc[v][r];
        s = fma(LT.w[r], uc[v][r], s);
      }
      sAvg[(v * M + w) * 32 + lane] = 0.25 * LT.w[w] * s;
    }
    __syncthreads();
    double ul[4][M];                             // line eta_w
#pragma unroll
    for (int v = 0; v < 4; ++v)
#pragma unroll
      for (int q = 0; q < M; ++q) ul[v][q] = tile[((v * M + w) * M + q) * 32 + lane];
    double ub[4];
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      double s = 0.0;
#pragma unroll
      for (int q = 0; q < M; ++q) s += sAvg[(v * M + q) * 32 + lane];
      ub[v] = s;
    }
    // step 1: density minimum over this thread's 2 nh points and its column's m nodes
    double rmin = ub[0];
#pragma unroll
    for (int r = 0; r < M; ++r) rmin = fmin(rmin, uc[0][r]);
    for (int k = 0; k < LT.nh; ++k) {
      double a = 0.0, b = 0.0;
#pragma unroll
      for (int r = 0; r < M; ++r) {
        a = fma(LT.Lh[k][r], uc[0][r], a);
        b = fma(LT.Lh[k][r], ul[0][r], b);
      }
      rmin = fmin(rmin, fmin(a, b));
    }
    sMin[w * 32 + lane] = rmin;
    __syncthreads();
#pragma unroll
    for (int ww = 0; ww < M; ++ww) rmin = fmin(rmin, sMin[ww * 32 + lane]);
    const double eps_rho = fmin(A.eps, ub[0]);
    double th1 = 1.0;
    if (rmin < eps_rho) th1 = (ub[0] - eps_rho) / (ub[0] - rmin);
    // step 2: pressure (ideal gas), with the density already limited
    double th2 = 1.0;
    if (EOS == 0) {
      const double pbar = A.ph.gm1 * (ub[3] - 0.5 * (ub[1] * ub[1] + ub[2] * ub[2]) / ub[0]);
      const double eps_p = fmin(A.eps, pbar);
      const double e1 = eps_p / A.ph.gm1;
      double tmin = 1.0;
      for (int k = 0; k < LT.nh; ++k) {
#pragma unroll
        for (int set = 0; set < 2; ++set) {
          double s[4];
#pragma unroll
          for (int v = 0; v < 4; ++v) {
            double a = 0.0;
#pragma unroll
            for (int r = 0; r < M; ++r) a = fma(LT.Lh[k][r], set == 0 ? uc[v][r] : ul[v][r], a);
            s[v] = a;
          }
          s[0] = fma(th1, s[0] - ub[0], ub[0]);
          const double pr = A.ph.gm1 * (s[3] - 0.5 * (s[1] * s[1] + s[2] * s[2]) / s[0]);
          if (pr < eps_p) tmin = fmin(tmin, segment_root(ub, s, e1));
        }
      }
#pragma unroll
      for (int r = 0; r < M; ++r) {               // the column's own nodes
        double s[4] = {fma(th1, uc[0][r] - ub[0], ub[0]), uc[1][r], uc[2][r], uc[3][r]};
        const double pr = A.ph.gm1 * (s[3] - 0.5 * (s[1] * s[1] + s[2] * s[2]) / s[0]);
        if (pr < eps_p) tmin = fmin(tmin, segment_root(ub, s, e1));
      }
      sT[w * 32 + lane] = tmin;
      __syncthreads();
#pragma unroll
      for (int ww = 0; ww < M; ++ww) th2 = fmin(th2, sT[ww * 32 + lane]);
    }
    // apply to this thread's column; FINAL: wave-killing relaxation and the CFL partial averages
    const bool changed = th1 < 1.0 || th2 < 1.0;
    double f0 = 0.0, ft = 1.0;
    bool damp = false;
    if (damp_on) {
      const double yc = g.y0 + (j + 0.5) * g.dy;
      damp = damp_factors(A.D, sqrt(xc * xc + yc * yc), f0, ft);
    }
    const double* p0 = A.q0 + (size_t)j * row_stride + (size_t)ib * BS + lane;
    // (every thread read sAvg before the barrier that follows the sMin exchange: it may be rewritten now)
    if (FINAL && damp && A.D.mode == 1) {
      // wave-killing of density, velocities and temperature: node by node over this thread's column
#pragma unroll
      for (int r = 0; r < M; ++r) {
        double u[4], u0[4];
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          const double th = v == 0 ? th1 * th2 : th2;
          u[v] = changed ? fma(th, uc[v][r] - ub[v], ub[v]) : uc[v][r];
          u0[v] = __ldg(p0 + ((v * M + r) * M + w) * 32);
        }
        damp_node_primitive(f0, ft, A.D.gm1, u, u0);
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          uc[v][r] = u[v];
          if (valid) p[((v * M + r) * M + w) * 32] = u[v];
        }
      }
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        double avg = 0.0;
#pragma unroll
        for (int r = 0; r < M; ++r) avg = fma(LT.w[r], uc[v][r], avg);
        sAvg[(v * M + w) * 32 + lane] = 0.25 * LT.w[w] * avg;
      }
    } else {
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        const double th = v == 0 ? th1 * th2 : th2;
        double avg = 0.0;
#pragma unroll
        for (int r = 0; r < M; ++r) {
          const int e = ((v * M + r) * M + w) * 32;
          double val = uc[v][r];
          if (changed) val = fma(th, val - ub[v], ub[v]);
          if (damp) val = fma(f0, __ldg(p0 + e), ft * val);
          if (valid && (changed || damp)) p[e] = val;
          if (FINAL) avg = fma(LT.w[r], val, avg);
        }
        if (FINAL) sAvg[(v * M + w) * 32 + lane] = 0.25 * LT.w[w] * avg;
      }
    }
    if (FINAL) __syncthreads();                  // sAvg of this row complete (read by warp 0 next iteration)
  }
  if (FINAL && w == 0) {
    cfl_of_row(j1 - 1);
    unsigned long long bits = (unsigned long long)__double_as_longlong(spmax);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const unsigned long long other = __shfl_xor_sync(FULL, bits, o);
      bits = other > bits ? other : bits;
    }
    if (lane == 0) atomicMax(A.wmax, bits);
  }
}

// ---------------------------------------------------------------------------------------------
// Torque on the planet, Eq.(6): Gamma_z = x_p a_y - y_p a_x with
//   a = sum_n G M_n (r_n - r_p) / (|r_n - r_p|^2 + eps_p^2)^(3/2),
// M_n = cell average of the density x cell area, r_n = the cell centre.  One warp per 32-cell tile;
// per-block partial sums land in `partial` (2 doubles per block) and torque_finish_kernel adds them
// in a fixed order, so the result does not depend on scheduling.
// ---------------------------------------------------------------------------------------------
template <int M>
__global__ void __launch_bounds__(128)
torque_kernel(const double* __restrict__ Q, double* __restrict__ partial, Geom g, DevTables T,
              double gm, double xp, double yp, double eps2p) {
  constexpr int C = 4 * M * M;
  __shared__ double sx[4], sy[4];
  const int lane = threadIdx.x & 31, wj = threadIdx.x >> 5;
  const int j = blockIdx.y * 4 + wj;
  const int ib = blockIdx.x;
  const int i = ib * 32 + lane;
  double ax = 0.0, ay = 0.0;
  if (j < g.ny && i < g.nx) {
    const double* cell = Q + ((size_t)j * g.nbx + ib) * C * 32 + lane;
    double s = 0.0;
#pragma unroll
    for (int r = 0; r < M; ++r) {
      double sr = 0.0;
#pragma unroll
      for (int q = 0; q < M; ++q) sr = fma(T.w[q], __ldg(cell + (r * M + q) * 32), sr);
      s = fma(T.w[r], sr, s);
    }
    const double Mn = 0.25 * s * g.dx * g.dy;
    const double ddx = g.x0 + (i + 0.5) * g.dx - xp, ddy = g.y0 + (j + 0.5) * g.dy - yp;
    const double r2 = fma(ddx, ddx, fma(ddy, ddy, eps2p));
    const double k = gm * Mn / (r2 * sqrt(r2));
    ax = k * ddx;
    ay = k * ddy;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    ax += __shfl_xor_sync(FULL, ax, o);
    ay += __shfl_xor_sync(FULL, ay, o);
  }
  if (lane == 0) { sx[wj] = ax; sy[wj] = ay; }
  __syncthreads();
  if (threadIdx.x == 0) {
    const size_t b = (size_t)blockIdx.y * gridDim.x + blockIdx.x;
    partial[2 * b] = (sx[0] + sx[1]) + (sx[2] + sx[3]);
    partial[2 * b + 1] = (sy[0] + sy[1]) + (sy[2] + sy[3]);
  }
}

// out[0] = Gamma_z, out[1] = a_x, out[2] = a_y
__global__ void __launch_bounds__(256)
torque_finish_kernel(const double* __restrict__ partial, int nblocks, double xp, double yp, double* out) {
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

}  // namespace dg
