// sm_100a kernels of the DG Euler hot path.
//
// Device data layout ("lane-blocked nodal"):
//   Q[j][ib][v][r][q][lane]      j  = cell row, ib = block of 32 consecutive cells along x,
//                                 v  = variable, (r,q) = Gauss-Legendre node (eta index, xi index),
//                                 lane = cell inside the block = the thread's lane.
// Every global and shared access of a warp is then 32 consecutive doubles (256 B): perfectly
// coalesced / conflict-free without any staging, and the x-neighbours of a cell are the
// neighbouring lanes (face data travels by warp shuffle).
//
// Stage kernel: one thread block = M warps marches over `rows` consecutive cell rows of one
// 32-cell column block.  For each row:
//   X phase  warp r owns the eta-line r of all 32 cells: traces at xi = -1/+1, flux F at the M nodes
//            of the line, x-derivative contraction (register blocked, tables in the constant bank),
//            LLF flux on the W/E faces (neighbour data by shuffle), x-lifting -> shared memory.
//   Y phase  warp q owns the xi-column q: the same along y with G, plus the gravity source, plus the
//            S/N faces (row below carried in registers while marching, row above read ahead), then
//            the RK combine (and damping) and the store of u^(s).
#pragma once
#include <cstdint>

namespace dg {

constexpr unsigned FULL = 0xffffffffu;

// Kernel variants are compile-time so that the unrolled node loops are straight-line code (runtime
// flags inside them split basic blocks and stop the scheduler from interleaving the nodes' chains).
enum : int {          // KIND: what the epilogue of the stage does
  K_RHS   = 0,        // write N = L(u)                                   (dg_rhs)
  K_FIRST = 1,        // u + dt N                                         (stage 1: alpha = 0, u^n not read)
  K_MID   = 2,        // a u^n + b (u + dt N)
  K_LAST  = 3,        // K_MID + fused CFL wave-speed reduction
  K_LASTD = 4,        // K_LAST + wave-killing relaxation
  K_COUNT = 5,
};
enum : int { G_NONE = 0, G_STAR = 1, G_PLANET = 2 };   // GRAV: gravity source terms present

struct DevTables {            // kernel-parameter (constant bank) copy of the tables
  double xi[MAXM], w[MAXM];
  double Dx[MAXM][MAXM];      // Dh[q'][q]/dx
  double Dy[MAXM][MAXM];      // Dh[r'][r]/dy
  double lxp[MAXM], lxm[MAXM], lyp[MAXM], lym[MAXM];   // lift vectors / dx, / dy
  double Ip[MAXM], Im[MAXM];  // interpolation to xi = +1 / -1
};

struct ConvTables { double B[MAXM][MAXM], P[MAXM][MAXM]; };

struct Phys {
  double gamma, gm1;          // eos 0
  double h2gm;                // eos 1: h^2 GM
  double gm, eps2s;           // star
  double qgm, xp, yp, eps2p;  // planet at the stage time
};

struct Geom {
  double x0, y0, dx, dy, hdx, hdy, inv_dx, inv_dy;
  int nx, ny, nbx, bc;
};

struct StageArgs {
  const double* qprev;        // u^(s-1)
  const double* qn;           // u^n
  double* qout;               // u^(s)   (or N when F_RHS_ONLY)
  const double* q0;           // initial state (damping)
  const double* btrW; const double* btrE; const double* btrS; const double* btrN;  // bc 2 traces
  unsigned long long* wmax;   // CFL wave-speed maximum (bit pattern of a non-negative double)
  double a, b, dt;
  double damp_r0, damp_inv_w, damp_tau0;
  int rows;
  Geom g;
  Phys ph;
  DevTables T;
};

// ---------------------------------------------------------------------------------------------
// fp64 special functions without slow paths: MUFU seed (~20 bits) + 2 Newton steps (measured max
// relative error 1.1e-16 / 1.4e-16 on B200).  Arguments are positive and normal here.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ double rcp_fast(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-x, r, 1.0);             // r <- r (1 + e + e^2), e ~ 1e-6
  return fma(r, fma(e, e, e), r);
}
__device__ __forceinline__ double rsqrt_fast(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-(x * y), y, 1.0);        // y <- y (1 + e/2 + 3 e^2/8), e ~ 1e-6
  return fma(y, e * fma(0.375, e, 0.5), y);
}
__device__ __forceinline__ double sqrt_fast(double x) { return x * rsqrt_fast(x); }

// ---------------------------------------------------------------------------------------------
// Point-wise physics (rows a2, a3, a6)
// ---------------------------------------------------------------------------------------------
// Euler flux in direction DIR of the conservative state u (Eq.(1)) with the closure
// Eq.(2) PAPER.md:45-49 (EOS 0) or p = c_s^2 rho (EOS 1: cs2 and c = sqrt(cs2) are passed in).
// LAM: also the signal speed |v_n| + c.
template <int EOS, int DIR, bool LAM>
__device__ __forceinline__ void euler_flux(const Phys& ph, const double (&u)[4], double cs2, double ciso,
                                           double (&F)[4], double& lam) {
  const double rinv = rcp_fast(u[0]);
  const double vx = u[1] * rinv, vy = u[2] * rinv;
  double pr;
  if (EOS == 0) pr = ph.gm1 * (u[3] - 0.5 * fma(u[1], vx, u[2] * vy));
  else          pr = cs2 * u[0];
  const double vn = DIR == 0 ? vx : vy;
  F[0] = u[1 + DIR];
  F[1] = DIR == 0 ? fma(u[1], vn, pr) : u[1] * vn;
  F[2] = DIR == 1 ? fma(u[2], vn, pr) : u[2] * vn;
  F[3] = (u[3] + pr) * vn;
  if (LAM) {
    const double c = EOS == 0 ? sqrt_fast(ph.gamma * pr * rinv) : ciso;
    lam = fabs(vn) + c;
  }
}

// Local Lax-Friedrichs flux from the two sides' states, fluxes and speeds.
// Each interior face is evaluated exactly once (by the cell on its left / below) and handed to the
// other cell, so the interface flux is single valued to the last bit.
__device__ __forceinline__ void llf(const double (&UL)[4], const double (&FL)[4], double lamL,
                                    const double (&UR)[4], const double (&FR)[4], double lamR,
                                    double (&H)[4]) {
  const double hl = 0.5 * fmax(lamL, lamR);
#pragma unroll
  for (int v = 0; v < 4; ++v) H[v] = fma(-hl, UR[v] - UL[v], 0.5 * (FL[v] + FR[v]));
}

// ---------------------------------------------------------------------------------------------
// Traces of a cell (node stride `s` doubles: 32 inside a tile, 1 inside the edge buffer)
// ---------------------------------------------------------------------------------------------
template <int M>
__device__ __forceinline__ void line_trace(const double* cell, int stride, int r,
                                           const double (&I)[MAXM], double (&out)[4]) {
#pragma unroll
  for (int v = 0; v < 4; ++v) {
    double s = 0.0;
#pragma unroll
    for (int q = 0; q < M; ++q) s = fma(I[q], cell[((v * M + r) * M + q) * stride], s);
    out[v] = s;
  }
}
template <int M>
__device__ __forceinline__ void column_trace(const double* cell, int stride, int q,
                                             const double (&I)[MAXM], double (&out)[4]) {
#pragma unroll
  for (int v = 0; v < 4; ++v) {
    double s = 0.0;
#pragma unroll
    for (int r = 0; r < M; ++r) s = fma(I[r], cell[((v * M + r) * M + q) * stride], s);
    out[v] = s;
  }
}

__device__ __forceinline__ double shfl_up1(double x) { return __shfl_up_sync(FULL, x, 1); }
__device__ __forceinline__ double shfl_dn1(double x) { return __shfl_down_sync(FULL, x, 1); }

// ---------------------------------------------------------------------------------------------
// TMA (bulk async copy) + mbarrier helpers: one contiguous 32-cell tile per copy
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// ---------------------------------------------------------------------------------------------
// The fused RK-stage kernel (rows a2..a12 of SURVEY.md 8(a); a1/a4's basis change is folded into
// the tables, see dg_tables.h).
//
// Shared memory of one thread block (M warps, one 32-cell column block, `rows` rows):
//   tiles[3]  ring of u^(s-1) tiles (rows j-1 | j | j+1 | j+2 rotating), each one contiguous
//             4 M^2 x 32 doubles in HBM -> filled by ONE cp.async.bulk (TMA) each, mbarrier-tracked;
//             the copy for row j+2 is in flight while row j is computed
//   sN        x-direction part of N for the row in flight ([v][r][q][lane]; transposes ownership
//             from eta-lines to xi-columns)
//   sRi       1/sqrt(x^2+y^2+eps^2) at the row's volume nodes (shared by c_s^2 and the star gravity)
//   sEdge[2]  the two x-neighbour cells outside the block, prefetched one row ahead
// ---------------------------------------------------------------------------------------------
constexpr int NST = 3;

template <int M>
constexpr size_t stage_smem_bytes() {
  // tiles + sN + sRi + sEdge + mbarriers
  return ((size_t)(NST + 1) * 4 * M * M * 32 + (size_t)M * M * 32 + (size_t)4 * 4 * M * M) * sizeof(double) + 64;
}

template <int M, int EOS, int GRAV, int KIND, int MINB>
__global__ void __launch_bounds__(M * 32, MINB)
stage_kernel(const __grid_constant__ StageArgs A) {
  constexpr bool grav = GRAV != G_NONE;
  constexpr bool need_ri = EOS == 1 || grav;
  constexpr bool use_un = KIND >= K_MID;
  constexpr bool do_cfl = KIND >= K_LAST;
  constexpr bool do_damp = KIND == K_LASTD;
  constexpr int C = 4 * M * M;                   // doubles per cell
  constexpr int BS = C * 32;                     // doubles per 32-cell tile
  constexpr int NT = M * 32;
  constexpr uint32_t TILE_BYTES = BS * sizeof(double);
  extern __shared__ __align__(128) double smem[];
  double* tiles = smem;
  double* sN = tiles + NST * BS;
  double* sRi = sN + BS;                         // [r][q][lane]
  double* sEdge = sRi + M * M * 32;              // [slot][side][C]
  uint64_t* mbar = reinterpret_cast<uint64_t*>(sEdge + 4 * C);

  const int tid = threadIdx.x;
  const int lane = tid & 31;
  const int w = tid >> 5;                        // eta-line (X phase) / xi-column (Y phase)
  const int ib = blockIdx.x;
  const int i = ib * 32 + lane;
  const Geom& g = A.g;
  const DevTables& T = A.T;
  const bool valid = i < g.nx;
  const int last_lane = min(31, g.nx - 1 - ib * 32);
  const int j0 = blockIdx.y * A.rows;
  const int j1 = min(g.ny, j0 + A.rows);
  const size_t row_stride = (size_t)g.nbx * BS;

  const double xc = g.x0 + (i + 0.5) * g.dx;
  const double xW = g.x0 + i * g.dx, xE = g.x0 + (i + 1) * g.dx;
  const double xq_col = xc + g.hdx * T.xi[w];    // x of this thread's column (Y phase)

  // x-neighbour cells outside this block: (cell index, or -1 when there is none)
  const int iLn = ib > 0 ? ib * 32 - 1 : (g.bc == 0 ? g.nx - 1 : -1);
  const int iRn = ib * 32 + 32 < g.nx ? ib * 32 + 32 : (g.bc == 0 ? 0 : -1);
  const double* edgeL = iLn >= 0 ? A.qprev + (size_t)(iLn >> 5) * BS + (iLn & 31) : nullptr;
  const double* edgeR = iRn >= 0 ? A.qprev + (size_t)(iRn >> 5) * BS + (iRn & 31) : nullptr;
  constexpr int NE = (2 * C + NT - 1) / NT;      // edge elements per thread
  auto edge_load = [&](int jj, double (&e)[NE]) {
#pragma unroll
    for (int k = 0; k < NE; ++k) {
      const int idx = tid + k * NT;
      e[k] = 0.0;
      if (idx < 2 * C) {
        const double* src = idx < C ? edgeL : edgeR;
        const int el = idx < C ? idx : idx - C;
        if (src) e[k] = __ldg(src + (size_t)jj * row_stride + el * 32);
      }
    }
  };
  auto edge_store = [&](int slot, const double (&e)[NE]) {
#pragma unroll
    for (int k = 0; k < NE; ++k) {
      const int idx = tid + k * NT;
      if (idx < 2 * C) sEdge[slot * 2 * C + idx] = e[k];
    }
  };

  // tile t holds row j0-1+t (wrapped for periodic domains; absent outside a non-periodic domain)
  auto tile_row = [&](int t) -> int {
    const int jj = j0 - 1 + t;
    if (jj < 0) return g.bc == 0 ? g.ny - 1 : -1;
    if (jj >= g.ny) return g.bc == 0 ? 0 : -1;
    return jj;
  };
  auto tile_issue = [&](int t) {
    const int jr = tile_row(t);
    if (tid == 0 && jr >= 0) {
      uint64_t* bar = mbar + t % NST;
      mbar_expect_tx(bar, TILE_BYTES);
      bulk_g2s(tiles + (t % NST) * BS, A.qprev + jr * row_stride + (size_t)ib * BS, TILE_BYTES, bar);
    }
  };
  // k-th copy into a slot completes mbarrier phase k; tile 0 is the only one that can be absent
  // and still be followed by later copies into its slot (non-periodic bottom row)
  const int skip0 = tile_row(0) < 0 ? 1 : 0;
  auto tile_wait = [&](int t) {
    if (tile_row(t) >= 0) mbar_wait(mbar + t % NST, (uint32_t)((t / NST - (t % NST == 0 ? skip0 : 0)) & 1));
  };

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NST; ++s) mbar_init(mbar + s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  tile_issue(0);
  tile_issue(1);
  tile_issue(2);
  {
    double e[NE];
    edge_load(j0, e);
    edge_store(j0 & 1, e);
  }

  // numerical flux through the south face of the row about to be processed, column q = w
  double HS[4];
  bool have_HS = false;
  double spmax = 0.0;                            // running CFL wave-speed maximum of this lane (warp 0)
  double bU[4], bG[4], bLam = 0.0;               // north-face data of the row below (first row only)
  bool have_below = false;
  {
    tile_wait(0);
    const double yS = g.y0 + j0 * g.dy;
    double cs2 = 0.0, ciso = 0.0;
    if (EOS == 1) {
      cs2 = A.ph.h2gm * rsqrt_fast(fma(xq_col, xq_col, fma(yS, yS, A.ph.eps2s)));
      ciso = sqrt_fast(cs2);
    }
    if (tile_row(0) >= 0) {
      column_trace<M>(tiles + lane, 32, w, T.Ip, bU);
      have_below = true;
    } else if (g.bc == 2) {
#pragma unroll
      for (int v = 0; v < 4; ++v) bU[v] = __ldg(A.btrS + ((size_t)(ib * 4 + v) * M + w) * 32 + lane);
      have_below = true;
    }
    if (have_below) euler_flux<EOS, 1, true>(A.ph, bU, cs2, ciso, bG, bLam);
  }
  __syncthreads();                               // tile 0's slot may be refilled; sEdge[j0&1] visible

  for (int j = j0; j < j1; ++j) {
    const int t = j - j0 + 1;                    // tile index of row j
    if (j + 1 < j1) tile_issue(t + 2);           // row j+2 -> the slot row j-1 has just left
    const double* tu = tiles + (t % NST) * BS + lane;
    const double yc = g.y0 + (j + 0.5) * g.dy;
    double enext[NE];
    const bool more = j + 1 < j1;
    if (more) edge_load(j + 1, enext);

    // fused CFL wave speed of the row finished in the previous iteration (row a10).
    // Partial cell averages were parked in sN[v][r=0][q][lane], which only this warp rewrites.
    if (do_cfl && w == 0 && j > j0) {
      double avg[4];
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        double s = 0.0;
#pragma unroll
        for (int qq = 0; qq < M; ++qq) s += sN[((v * M + 0) * M + qq) * 32 + lane];
        avg[v] = s;
      }
      double sp = 0.0;
      if (valid) {
        const double ycp = g.y0 + (j - 0.5) * g.dy;
        const double rinv = 1.0 / avg[0];
        const double vx = avg[1] * rinv, vy = avg[2] * rinv;
        double c;
        if (EOS == 0) c = sqrt(A.ph.gamma * A.ph.gm1 * (avg[3] - 0.5 * (avg[1] * vx + avg[2] * vy)) * rinv);
        else          c = sqrt(A.ph.h2gm * rsqrt(fma(xc, xc, fma(ycp, ycp, A.ph.eps2s))));
        sp = (fabs(vx) + c) * g.inv_dx + (fabs(vy) + c) * g.inv_dy;
        if (!(sp >= 0.0)) sp = __longlong_as_double(0x7ff0000000000000LL);   // NaN -> +inf
      }
      spmax = fmax(spmax, sp);                   // per lane; reduced once after the last row
    }

    tile_wait(t);
    // =========================== X phase: eta-line r = w ===========================
    {
      const int r = w;
      const double yr = yc + g.hdy * T.xi[r];
      const double y2e = fma(yr, yr, A.ph.eps2s);
      double acc[4][M];
#pragma unroll
      for (int v = 0; v < 4; ++v)
#pragma unroll
        for (int q = 0; q < M; ++q) acc[v][q] = 0.0;
      double UW[4] = {0, 0, 0, 0}, UE[4] = {0, 0, 0, 0};
#pragma unroll
      for (int q = 0; q < M; ++q) {
        double u[4];
#pragma unroll
        for (int v = 0; v < 4; ++v) u[v] = tu[((v * M + r) * M + q) * 32];
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          UW[v] = fma(T.Im[q], u[v], UW[v]);
          UE[v] = fma(T.Ip[q], u[v], UE[v]);
        }
        double cs2 = 0.0;
        if (need_ri) {
          const double xq = xc + g.hdx * T.xi[q];
          const double ri = rsqrt_fast(fma(xq, xq, y2e));
          sRi[(r * M + q) * 32 + lane] = ri;
          if (EOS == 1) cs2 = A.ph.h2gm * ri;
        }
        double F[4], dummy;
        euler_flux<EOS, 0, false>(A.ph, u, cs2, 0.0, F, dummy);
#pragma unroll
        for (int v = 0; v < 4; ++v)
#pragma unroll
          for (int qq = 0; qq < M; ++qq) acc[v][qq] = fma(T.Dx[qq][q], F[v], acc[v][qq]);
      }
      // own W/E face states, fluxes, speeds; c_s at the E face is the right neighbour's W value
      double cs2W = 0.0, cW = 0.0, cs2E = 0.0, cE = 0.0;
      if (EOS == 1) {
        cs2W = A.ph.h2gm * rsqrt_fast(fma(xW, xW, y2e));
        cW = sqrt_fast(cs2W);
        cs2E = shfl_dn1(cs2W);
        cE = shfl_dn1(cW);
        if (lane == 31) {
          cs2E = A.ph.h2gm * rsqrt_fast(fma(xE, xE, y2e));
          cE = sqrt_fast(cs2E);
        }
      }
      double FWo[4], FEo[4], lamWo, lamEo;
      euler_flux<EOS, 0, true>(A.ph, UW, cs2W, cW, FWo, lamWo);
      euler_flux<EOS, 0, true>(A.ph, UE, cs2E, cE, FEo, lamEo);
      double UR[4], FR[4], lamR;
#pragma unroll
      for (int v = 0; v < 4; ++v) { UR[v] = shfl_dn1(UW[v]); FR[v] = shfl_dn1(FWo[v]); }
      lamR = shfl_dn1(lamWo);
      if (lane == last_lane) {                   // right neighbour is outside this block
        if (edgeR) {
          line_trace<M>(sEdge + (j & 1) * 2 * C + C, 1, r, T.Im, UR);
        } else if (g.bc == 1) {
#pragma unroll
          for (int v = 0; v < 4; ++v) UR[v] = UE[v];
        } else {
#pragma unroll
          for (int v = 0; v < 4; ++v) UR[v] = __ldg(A.btrE + ((size_t)j * 4 + v) * M + r);
        }
        euler_flux<EOS, 0, true>(A.ph, UR, cs2E, cE, FR, lamR);
      }
      double HE[4], HW[4];
      llf(UE, FEo, lamEo, UR, FR, lamR, HE);
#pragma unroll
      for (int v = 0; v < 4; ++v) HW[v] = shfl_up1(HE[v]);
      if (lane == 0) {                           // left neighbour is outside this block
        double UL[4], FL[4], lamL;
        if (edgeL) {
          line_trace<M>(sEdge + (j & 1) * 2 * C, 1, r, T.Ip, UL);
        } else if (g.bc == 1) {
#pragma unroll
          for (int v = 0; v < 4; ++v) UL[v] = UW[v];
        } else {
#pragma unroll
          for (int v = 0; v < 4; ++v) UL[v] = __ldg(A.btrW + ((size_t)j * 4 + v) * M + r);
        }
        euler_flux<EOS, 0, true>(A.ph, UL, cs2W, cW, FL, lamL);
        llf(UL, FL, lamL, UW, FWo, lamWo, HW);
      }
#pragma unroll
      for (int v = 0; v < 4; ++v)
#pragma unroll
        for (int qq = 0; qq < M; ++qq)
          sN[((v * M + r) * M + qq) * 32 + lane] =
              fma(T.lxm[qq], HW[v], fma(-T.lxp[qq], HE[v], acc[v][qq]));
    }
    __syncthreads();

    // =========================== Y phase: xi-column q = w ===========================
    {
      const int q = w;
      const double xq = xq_col;
      const double* __restrict__ qn = A.qn + j * row_stride + (size_t)ib * BS + lane;
      double un[4][M];
      if (use_un) {
#pragma unroll
        for (int v = 0; v < 4; ++v)
#pragma unroll
          for (int rr = 0; rr < M; ++rr) un[v][rr] = __ldg(qn + ((v * M + rr) * M + q) * 32);
      }
      double acc[4][M];
#pragma unroll
      for (int v = 0; v < 4; ++v)
#pragma unroll
        for (int r = 0; r < M; ++r) acc[v][r] = 0.0;
      double UN[4] = {0, 0, 0, 0};
      const bool first = !have_HS;
#pragma unroll
      for (int r = 0; r < M; ++r) {
        double u[4];
#pragma unroll
        for (int v = 0; v < 4; ++v) u[v] = tu[((v * M + r) * M + q) * 32];
#pragma unroll
        for (int v = 0; v < 4; ++v) UN[v] = fma(T.Ip[r], u[v], UN[v]);
        // gravity (row a3); the isothermal sound speed shares the star's 1/r_s
        double cs2 = 0.0, gx = 0.0, gy = 0.0;
        if (need_ri) {
          const double yr = yc + g.hdy * T.xi[r];
          const double ri = sRi[(r * M + q) * 32 + lane];
          if (EOS == 1) cs2 = A.ph.h2gm * ri;
          if (grav) {
            const double k = -A.ph.gm * ri * ri * ri;
            gx = k * xq;
            gy = k * yr;
            if (GRAV == G_PLANET) {
              const double ddx = xq - A.ph.xp, ddy = yr - A.ph.yp;
              const double rpi = rsqrt_fast(fma(ddx, ddx, fma(ddy, ddy, A.ph.eps2p)));
              const double kp = -A.ph.qgm * rpi * rpi * rpi;
              gx = fma(kp, ddx, gx);
              gy = fma(kp, ddy, gy);
            }
          }
        }
        double G[4], dummy;
        euler_flux<EOS, 1, false>(A.ph, u, cs2, 0.0, G, dummy);
#pragma unroll
        for (int v = 0; v < 4; ++v)
#pragma unroll
          for (int rr = 0; rr < M; ++rr) acc[v][rr] = fma(T.Dy[rr][r], G[v], acc[v][rr]);
        if (grav) {
          acc[1][r] = fma(u[0], gx, acc[1][r]);
          acc[2][r] = fma(u[0], gy, acc[2][r]);
          acc[3][r] = fma(u[1], gx, fma(u[2], gy, acc[3][r]));
        }
      }
      // south face: carried from the previous row, or built once at the start of the segment
      if (first) {
        double US[4];
        column_trace<M>(tu, 32, q, T.Im, US);
        const double yS = g.y0 + j * g.dy;
        double cs2 = 0.0, ciso = 0.0;
        if (EOS == 1) {
          cs2 = A.ph.h2gm * rsqrt_fast(fma(xq, xq, fma(yS, yS, A.ph.eps2s)));
          ciso = sqrt_fast(cs2);
        }
        double GSo[4], lamSo;
        euler_flux<EOS, 1, true>(A.ph, US, cs2, ciso, GSo, lamSo);
        if (!have_below) {                       // transmissive bottom boundary
#pragma unroll
          for (int v = 0; v < 4; ++v) { bU[v] = US[v]; bG[v] = GSo[v]; }
          bLam = lamSo;
        }
        llf(bU, bG, bLam, US, GSo, lamSo, HS);
        have_HS = true;
      }
      // north face: own trace against the S trace of the row above (tile t+1)
      const double yN = g.y0 + (j + 1) * g.dy;
      double cs2N = 0.0, cN = 0.0;
      if (EOS == 1) {
        cs2N = A.ph.h2gm * rsqrt_fast(fma(xq, xq, fma(yN, yN, A.ph.eps2s)));
        cN = sqrt_fast(cs2N);
      }
      double GNo[4], lamNo;
      euler_flux<EOS, 1, true>(A.ph, UN, cs2N, cN, GNo, lamNo);
      double aU[4], aG[4], aLam;
      if (tile_row(t + 1) >= 0) {
        tile_wait(t + 1);
        column_trace<M>(tiles + ((t + 1) % NST) * BS + lane, 32, q, T.Im, aU);
        euler_flux<EOS, 1, true>(A.ph, aU, cs2N, cN, aG, aLam);
      } else if (g.bc == 1) {
#pragma unroll
        for (int v = 0; v < 4; ++v) { aU[v] = UN[v]; aG[v] = GNo[v]; }
        aLam = lamNo;
      } else {
#pragma unroll
        for (int v = 0; v < 4; ++v) aU[v] = __ldg(A.btrN + ((size_t)(ib * 4 + v) * M + q) * 32 + lane);
        euler_flux<EOS, 1, true>(A.ph, aU, cs2N, cN, aG, aLam);
      }
      double HN[4];
      llf(UN, GNo, lamNo, aU, aG, aLam, HN);

      // wave-killing factors of this cell (row a12): out <- f0 u0 + ft out
      double f0 = 0.0, ft = 1.0;
      bool damp = false;
      if (do_damp) {
        const double rc = sqrt(xc * xc + yc * yc);
        if (rc > A.damp_r0) {
          const double s = (rc - A.damp_r0) * A.damp_inv_w;
          const double R = fmin(1.0, s * s);
          if (R > 0.0) {
            const double tau = A.damp_tau0 / R;
            const double inv = 1.0 / (tau + A.dt);
            damp = true;
            f0 = A.dt * inv;
            ft = tau * inv;
          }
        }
      }
      // modal update in nodal form + RK combination (rows a8, a9) and store
      double* __restrict__ qo = A.qout + j * row_stride + (size_t)ib * BS + lane;
      const double* __restrict__ q0 = A.q0 + j * row_stride + (size_t)ib * BS + lane;
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        double avg = 0.0;
#pragma unroll
        for (int rr = 0; rr < M; ++rr) {
          const int e = ((v * M + rr) * M + q) * 32;
          const double n = sN[e + lane] + fma(T.lym[rr], HS[v], fma(-T.lyp[rr], HN[v], acc[v][rr]));
          double out;
          if (KIND == K_RHS) {
            out = n;
          } else {
            out = fma(A.dt, n, tu[e]);
            if (use_un) out = fma(A.a, un[v][rr], A.b * out);
            if (do_damp && damp) out = fma(f0, __ldg(q0 + e), ft * out);
          }
          if (valid) qo[e] = out;
          if (do_cfl) avg = fma(T.w[rr], out, avg);
        }
        if (do_cfl) sN[((v * M + 0) * M + q) * 32 + lane] = 0.25 * T.w[q] * avg;
      }
#pragma unroll
      for (int v = 0; v < 4; ++v) HS[v] = HN[v];   // this row's N face is the next row's S face
      if (more) edge_store((j + 1) & 1, enext);
    }
    __syncthreads();
  }
  // CFL wave speed of the last row of the segment, then one reduction per thread block
  if (do_cfl && w == 0) {
    double avg[4];
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      double s = 0.0;
#pragma unroll
      for (int qq = 0; qq < M; ++qq) s += sN[((v * M + 0) * M + qq) * 32 + lane];
      avg[v] = s;
    }
    double sp = 0.0;
    if (valid) {
      const double ycp = g.y0 + (j1 - 0.5) * g.dy;
      const double rinv = 1.0 / avg[0];
      const double vx = avg[1] * rinv, vy = avg[2] * rinv;
      double c;
      if (EOS == 0) c = sqrt(A.ph.gamma * A.ph.gm1 * (avg[3] - 0.5 * (avg[1] * vx + avg[2] * vy)) * rinv);
      else          c = sqrt(A.ph.h2gm * rsqrt(fma(xc, xc, fma(ycp, ycp, A.ph.eps2s))));
      sp = (fabs(vx) + c) * g.inv_dx + (fabs(vy) + c) * g.inv_dy;
      if (!(sp >= 0.0)) sp = __longlong_as_double(0x7ff0000000000000LL);
    }
    // non-negative doubles order like their bit patterns
    unsigned long long bits = (unsigned long long)__double_as_longlong(fmax(spmax, sp));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const unsigned long long other = __shfl_xor_sync(FULL, bits, o);
      bits = other > bits ? other : bits;
    }
    if (lane == 0) atomicMax(A.wmax, bits);
  }
}

template <int EOS>
__device__ __forceinline__ double cs2_iso(const Phys& ph, double x, double y) {
  return EOS == 1 ? ph.h2gm * rsqrt(fma(x, x, fma(y, y, ph.eps2s))) : 0.0;
}

// ---------------------------------------------------------------------------------------------
// Stand-alone CFL reduction (row a10) on the nodal state: cell averages by the m x m rule.
// ---------------------------------------------------------------------------------------------
template <int M, int EOS>
__global__ void __launch_bounds__(128)
cfl_kernel(const double* __restrict__ Q, unsigned long long* wmax, Geom g, Phys ph, DevTables T) {
  const int lane = threadIdx.x & 31;
  const int j = blockIdx.y * 4 + (threadIdx.x >> 5);
  const int ib = blockIdx.x;
  const int i = ib * 32 + lane;
  constexpr int C = 4 * M * M;
  double sp = 0.0;
  if (j < g.ny && i < g.nx) {
    const double* cell = Q + ((size_t)j * g.nbx + ib) * C * 32 + lane;
    double avg[4];
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      double s = 0.0;
#pragma unroll
      for (int r = 0; r < M; ++r) {
        double sr = 0.0;
#pragma unroll
        for (int q = 0; q < M; ++q) sr = fma(T.w[q], __ldg(cell + ((v * M + r) * M + q) * 32), sr);
        s = fma(T.w[r], sr, s);
      }
      avg[v] = 0.25 * s;
    }
    const double rinv = 1.0 / avg[0];
    const double vx = avg[1] * rinv, vy = avg[2] * rinv;
    double c;
    if (EOS == 0) c = sqrt(ph.gamma * ph.gm1 * (avg[3] - 0.5 * (avg[1] * vx + avg[2] * vy)) * rinv);
    else          c = sqrt(cs2_iso<EOS>(ph, g.x0 + (i + 0.5) * g.dx, g.y0 + (j + 0.5) * g.dy));
    sp = (fabs(vx) + c) * g.inv_dx + (fabs(vy) + c) * g.inv_dy;
    if (!(sp >= 0.0)) sp = __longlong_as_double(0x7ff0000000000000LL);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) sp = fmax(sp, __shfl_xor_sync(FULL, sp, o));
  if (lane == 0) atomicMax(wmax, (unsigned long long)__double_as_longlong(sp));
}

// ---------------------------------------------------------------------------------------------
// Layout / basis conversion at the boundary of the library (rows a1 and a4's projection):
//   modal U[j][i][v][b][a]  <->  nodal Q[j][ib][v][r][q][lane]
// ---------------------------------------------------------------------------------------------
template <int M>
__global__ void __launch_bounds__(32)
modal_to_nodal_kernel(const double* __restrict__ U, double* __restrict__ Q, int nx, int nbx,
                      const __grid_constant__ ConvTables CT) {
  constexpr int C = 4 * M * M;
  __shared__ double buf[32 * (C + 1)];
  const int lane = threadIdx.x, ib = blockIdx.x, j = blockIdx.y;
  const int ncell = min(32, nx - ib * 32);
  const double* src = U + ((size_t)j * nx + (size_t)ib * 32) * C;
  for (int k = lane; k < ncell * C; k += 32) buf[(k / C) * (C + 1) + (k % C)] = __ldg(src + k);
  __syncwarp();
  double* dst = Q + ((size_t)j * nbx + ib) * C * 32 + lane;
  const double* mine = buf + lane * (C + 1);
#pragma unroll 1
  for (int v = 0; v < 4; ++v) {
    double t[M][M];                                  // t[b][q] = sum_a B[q][a] U[b][a]
#pragma unroll
    for (int b = 0; b < M; ++b)
#pragma unroll
      for (int q = 0; q < M; ++q) {
        double s = 0.0;
#pragma unroll
        for (int a = 0; a < M; ++a) s = fma(CT.B[q][a], lane < ncell ? mine[(v * M + b) * M + a] : 0.0, s);
        t[b][q] = s;
      }
#pragma unroll
    for (int r = 0; r < M; ++r)
#pragma unroll
      for (int q = 0; q < M; ++q) {
        double s = 0.0;
#pragma unroll
        for (int b = 0; b < M; ++b) s = fma(CT.B[r][b], t[b][q], s);
        // padding lanes hold a benign constant state (rho = E = 1, no momentum)
        if (lane >= ncell) s = (v == 0 || v == 3) ? 1.0 : 0.0;
        dst[((v * M + r) * M + q) * 32] = s;
      }
  }
}

template <int M>
__global__ void __launch_bounds__(32)
nodal_to_modal_kernel(const double* __restrict__ Q, double* __restrict__ U, int nx, int nbx,
                      const __grid_constant__ ConvTables CT) {
  constexpr int C = 4 * M * M;
  __shared__ double buf[32 * (C + 1)];
  const int lane = threadIdx.x, ib = blockIdx.x, j = blockIdx.y;
  const int ncell = min(32, nx - ib * 32);
  const double* src = Q + ((size_t)j * nbx + ib) * C * 32 + lane;
  double* mine = buf + lane * (C + 1);
#pragma unroll 1
  for (int v = 0; v < 4; ++v) {
    double t[M][M];                                  // t[r][a] = sum_q P[q][a] u[r][q]
#pragma unroll
    for (int r = 0; r < M; ++r) {
      double u[M];
#pragma unroll
      for (int q = 0; q < M; ++q) u[q] = __ldg(src + ((v * M + r) * M + q) * 32);
#pragma unroll
      for (int a = 0; a < M; ++a) {
        double s = 0.0;
#pragma unroll
        for (int q = 0; q < M; ++q) s = fma(CT.P[q][a], u[q], s);
        t[r][a] = s;
      }
    }
#pragma unroll
    for (int b = 0; b < M; ++b)
#pragma unroll
      for (int a = 0; a < M; ++a) {
        double s = 0.0;
#pragma unroll
        for (int r = 0; r < M; ++r) s = fma(CT.P[r][b], t[r][a], s);
        mine[(v * M + b) * M + a] = s;
      }
  }
  __syncwarp();
  double* dst = U + ((size_t)j * nx + (size_t)ib * 32) * C;
  for (int k = lane; k < ncell * C; k += 32) dst[k] = buf[(k / C) * (C + 1) + (k % C)];
}

// Traces of the initial state on the domain boundary (bc 2, row a11):
//   btrW[j][v][r], btrE[j][v][r]            (x = x0 / x1 faces)
//   btrS[ib][v][q][lane], btrN[ib][v][q][lane]   (y = y0 / y1 faces)
template <int M>
__global__ void boundary_trace_kernel(const double* __restrict__ Q0, double* btrW, double* btrE,
                                      double* btrS, double* btrN, Geom g, DevTables T) {
  constexpr int C = 4 * M * M;
  constexpr size_t BS = (size_t)C * 32;
  const size_t row_stride = (size_t)g.nbx * BS;
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int nside = g.ny * 4 * M;
  if (t < nside) {
    const int r = t % M, v = (t / M) % 4, j = t / (4 * M);
    const int il = g.nx - 1;
    const double* cw = Q0 + j * row_stride;
    const double* ce = Q0 + j * row_stride + (size_t)(il >> 5) * BS + (il & 31);
    double sw = 0.0, se = 0.0;
    for (int q = 0; q < M; ++q) {
      sw = fma(T.Im[q], cw[((v * M + r) * M + q) * 32], sw);
      se = fma(T.Ip[q], ce[((v * M + r) * M + q) * 32], se);
    }
    btrW[t] = sw;
    btrE[t] = se;
  }
  const int ntop = g.nbx * 4 * M * 32;
  if (t < ntop) {
    const int lane = t & 31, q = (t >> 5) % M, v = (t / (32 * M)) % 4, ib = t / (32 * M * 4);
    const double* cs = Q0 + ib * BS + lane;
    const double* cn = Q0 + (size_t)(g.ny - 1) * row_stride + ib * BS + lane;
    double ss = 0.0, sn = 0.0;
    for (int r = 0; r < M; ++r) {
      ss = fma(T.Im[r], cs[((v * M + r) * M + q) * 32], ss);
      sn = fma(T.Ip[r], cn[((v * M + r) * M + q) * 32], sn);
    }
    btrS[t] = ss;
    btrN[t] = sn;
  }
}

// Stand-alone wave-killing relaxation (row a12), used where it cannot ride on the last
// stage (dg_step_debug).  In place: Q <- (dt Q0 + tau Q)/(tau + dt) for cells with R(r) > 0.
template <int M>
__global__ void __launch_bounds__(128)
damp_kernel(double* __restrict__ Q, const double* __restrict__ Q0, Geom g, double dt, double r0,
            double inv_w, double tau0) {
  const int lane = threadIdx.x & 31;
  const int j = blockIdx.y * 4 + (threadIdx.x >> 5);
  const int ib = blockIdx.x;
  const int i = ib * 32 + lane;
  constexpr int C = 4 * M * M;
  if (j >= g.ny || i >= g.nx) return;
  const double xc = g.x0 + (i + 0.5) * g.dx, yc = g.y0 + (j + 0.5) * g.dy;
  const double rc = sqrt(xc * xc + yc * yc);
  if (!(rc > r0)) return;
  const double s = (rc - r0) * inv_w;
  const double R = fmin(1.0, s * s);
  if (!(R > 0.0)) return;
  const double tau = tau0 / R;
  const size_t base = ((size_t)j * g.nbx + ib) * C * 32 + lane;
#pragma unroll 4
  for (int e = 0; e < C; ++e) Q[base + e * 32] = (dt * Q0[base + e * 32] + tau * Q[base + e * 32]) / (tau + dt);
}

}  // namespace dg
