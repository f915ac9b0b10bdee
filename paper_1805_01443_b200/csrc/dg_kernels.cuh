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
// Compile-time variants: EOS (ideal gas / locally isothermal), GRAV (none / star / star + planet), KIND (what
// the epilogue does: rhs only, SSP stages, Butcher-form sub-steps of SURVEY.md 8(f) NEXT-2), FLUX (local
// Lax-Friedrichs / HLLC-HLL, NEXT-4).  At a halo edge of a strip decomposition the out-of-strip row is
// fetched from a halo row like any other tile (StageArgs::haloS / haloN).
//
// Why 2 thread blocks of 5 warps per SM at M = 5: 4 tile-sized buffers of 25.6 KB + tables = 114 KB of shared
// memory per block, and 168 registers is the most that lets 10 warps reside (registers are handed out to
// warps in groups of four: 12 x 168 x 32 <= 64 Ki).
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
  K_GEN   = 5,        // sub-step of a general explicit scheme (Appendix A) in state form
                      //   (dg_tables.h): K_MID plus earlier stage states, out = a u^n + b u + sum_j kc[j] kin[j] + beta N
  K_GENL  = 6,        // K_GEN of the last sub-step: fused CFL reduction, wave-killing if enabled
  K_COUNT = 7,
};
constexpr int MAXK = 5;   // earlier stage states a general sub-step can combine (Cash-Karp's last: 4)
enum : int { G_NONE = 0, G_STAR = 1, G_PLANET = 2 };   // GRAV: gravity source terms present

struct DevTables {            // kernel-parameter (constant bank) copy of the tables
  double xi[MAXM], w[MAXM];
  double Dx[MAXM][MAXM];      // beta Dh[q'][q]/dx
  double Dy[MAXM][MAXM];      // beta Dh[r'][r]/dy
  double lxp[MAXM], lxm[MAXM], lyp[MAXM], lym[MAXM];   // (beta/2) lift vectors / dx, / dy (kernels carry 2 x LLF flux)
  double Ip[MAXM], Im[MAXM];  // interpolation to xi = +1 / -1
};

struct ConvTables { double B[MAXM][MAXM], P[MAXM][MAXM]; };

struct Phys {
  double gamma, gm1;          // eos 0
  double h2gm;                // eos 1: h^2 GM
  double gmb, eps2s;          // star: beta GM (beta = the stage's factor of N, folded in on the host)
  double qgmb, xp, yp, eps2p; // planet at the stage time: beta q GM
};

struct Geom {
  double x0, y0, dx, dy, hdx, hdy, inv_dx, inv_dy;
  int nx, ny, nbx, bc;
};

// Wave-killing zones (row a12): outer zone r > r0 (full strength from r1 outwards) and,
// for the paper's own disc, an inner zone r < in_r0 (full strength from in_r1 inwards).  Per cell, with
// the ramp R = min(1, ((r - r_d)/(r_b - r_d))^2) and tau = 2 pi sqrt(r_d^3/GM)/R:  Q <- f0 Q0 + ft Q,
// f0 = dt/(tau + dt), ft = tau/(tau + dt).
struct DampArgs {
  double r0, inv_w, tau0;          // outer: r_d, 1/(r_b - r_d), 2 pi sqrt(r_d^3/GM); off: r0 = +inf, on = 0
  double in_r0, in_inv_w, in_tau0; // inner: r_d, 1/(r_d - r_b), 2 pi sqrt(r_d^3/GM); off: in_r0 = 0
  int on;                          // any zone enabled
  int mode;                        // 0: relax the conservative state; 1: density, velocities, temperature
  double gm1;                      // gamma - 1 (mode 1: T = p/rho with p from Eq.(2))
  double dt;
};
__device__ __forceinline__ double rcp_fast(double x);
__device__ __forceinline__ bool damp_factors(const DampArgs& D, double rc, double& f0, double& ft) {
  double s, tau0;
  if (rc > D.r0) {                               // r0 = +inf when the outer zone is off
    s = (rc - D.r0) * D.inv_w;
    tau0 = D.tau0;
  } else if (rc < D.in_r0) {                     // in_r0 = 0 when the inner zone is off
    s = (D.in_r0 - rc) * D.in_inv_w;
    tau0 = D.in_tau0;
  } else {
    return false;
  }
  const double R = fmin(1.0, s * s);
  if (!(R > 0.0)) return false;
  const double tau = tau0 * rcp_fast(R);          // slow-path-free (relative error 1.1e-16)
  const double inv = rcp_fast(tau + D.dt);
  f0 = D.dt * inv;
  ft = tau * inv;
  return true;
}

struct StageArgs {
  const double* qprev;        // u^(s-1)
  const double* qn;           // u^n
  double* qout;               // u^(s)   (or N when F_RHS_ONLY)
  const double* q0;           // initial state (damping)
  const double* btrW; const double* btrE; const double* btrS; const double* btrN;  // bc 2 traces
  const double* haloS; const double* haloN;   // strip decomposition along y: the neighbour strips' boundary rows
                                              // of the array qprev ([nbx][4 M^2 x 32], same layout), or null
  unsigned long long* wmax;   // CFL wave-speed maximum (bit pattern of a non-negative double)
  double a, b, dt;            // out = a u^n + b u^(s-1) + beta N; beta = b dt is folded into T and ph
  DampArgs D;
  int rows;
  // rows a launch covers: thread blocks y < nblkA march over [rowA0, rowA1) in segments of `rows` rows, the others
  // over [rowB0, rowB1).  A whole-domain launch is region A = [0, ny); a strip of a decomposed domain launches its
  // interior rows while the halo exchange is in flight and the few rows next to the halos afterwards.
  int rowA0, rowA1, nblkA, rowB0, rowB1;
  // K_GEN / K_GENL: the earlier stage states the sub-step combines (besides u^n and its input) and their
  // coefficients
  const double* kin[MAXK];
  double kc[MAXK];
  double* zout;               // if set: also store a u^n + b u + beta N, the value before the kin terms are added
                              // (limiter runs keep these instead of stage states: the limiter changes the states)
  int nk;
  int impl;                   // host-side choice of the kernel: 0 default, 1 dg::stage_kernel, 2 dg::stage_kernel_fh (dg_stage_fh.cuh)
  int gen_pf;                 // L2 prefetch of the epilogue's inputs: 0 none, 1 row start, 2 a row ahead (evicted before use: 1.7x DRAM reads), 3 at the x/y phase boundary
  Geom g;
  Phys ph;
  DevTables T;
};

// Wave-killing of "the density, velocities and temperature" (damp_mode 1) at one node: Q <- f0 Q0 + ft Q
// for Q = rho, v_x, v_y, T = p/rho (p from Eq.(2) of the carried energy), then the conservative state of the
// relaxed fields.  u: the node's current state (in/out), u0: the initial state's.
__device__ __forceinline__ void damp_node_primitive(double f0, double ft, double gm1, double (&u)[4], const double (&u0)[4]) {
  const double ri0 = 1.0 / u0[0], ri = 1.0 / u[0];
  const double v0x = u0[1] * ri0, v0y = u0[2] * ri0, vx_ = u[1] * ri, vy_ = u[2] * ri;
  const double T0 = gm1 * (u0[3] - 0.5 * (u0[1] * v0x + u0[2] * v0y)) * ri0;
  const double T1 = gm1 * (u[3] - 0.5 * (u[1] * vx_ + u[2] * vy_)) * ri;
  const double rho = fma(f0, u0[0], ft * u[0]);
  const double vx = fma(f0, v0x, ft * vx_), vy = fma(f0, v0y, ft * vy_);
  const double T = fma(f0, T0, ft * T1);
  u[0] = rho;
  u[1] = rho * vx;
  u[2] = rho * vy;
  u[3] = rho * (T / gm1 + 0.5 * (vx * vx + vy * vy));
}

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
// same for either sign of x (the MUFU seed carries the sign)
__device__ __forceinline__ double rcp_fast_signed(double x) { return copysign(rcp_fast(fabs(x)), x); }
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

// Local Lax-Friedrichs flux from the two sides' states, fluxes and speeds,
// TIMES TWO: (FL + FR) - max(lamL, lamR) (UR - UL); the 1/2 lives in the lifting tables.
// Each interior face is evaluated exactly once (by the cell on its left / below) and handed to the
// other cell, so the interface flux is single valued to the last bit.
__device__ __forceinline__ void llf2(const double (&UL)[4], const double (&FL)[4], double lamL,
                                     const double (&UR)[4], const double (&FR)[4], double lamR,
                                     double (&H)[4]) {
  const double lam = fmax(lamL, lamR);
#pragma unroll
  for (int v = 0; v < 4; ++v) H[v] = fma(-lam, UR[v] - UL[v], FL[v] + FR[v]);
}

// What a Riemann solver needs from one side of a face besides U and F.  FLUX 0 (local Lax-Friedrichs): the
// signal speed |v_n| + c; FLUX 1 (HLLC for the ideal gas, HLL for the isothermal closure; SURVEY.md 8(f)
// NEXT-4): normal velocity, sound speed and pressure.
template <int FLUX> struct Wave;
template <> struct Wave<0> { double lam; };
template <> struct Wave<1> { double vn, c, pr; };

template <int EOS, int DIR, int FLUX>
__device__ __forceinline__ void face_flux(const Phys& ph, const double (&u)[4], double cs2, double ciso,
                                          double (&F)[4], Wave<FLUX>& w) {
  if constexpr (FLUX == 0) {
    euler_flux<EOS, DIR, true>(ph, u, cs2, ciso, F, w.lam);
  } else {
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
    w.vn = vn;
    w.c = EOS == 0 ? sqrt_fast(ph.gamma * pr * rinv) : ciso;
    w.pr = pr;
  }
}

// Numerical flux TIMES TWO through a face with normal +DIR (the 1/2 lives in the lifting tables), left state
// first.  FLUX 1: Davis wave speeds S_L = min(v_L - c_L, v_R - c_R), S_R = max(v_L + c_L, v_R + c_R); HLL
// (S_R F_L - S_L F_R + S_L S_R (U_R - U_L))/(S_R - S_L) for the isothermal closure; HLLC (Toro, Spruce &
// Speares 1994) with the contact speed S* and the star state of the upwind side for the ideal gas.
template <int FLUX, int EOS, int DIR>
__device__ __forceinline__ void riemann2(const double (&UL)[4], const double (&FL)[4], const Wave<FLUX>& wL,
                                         const double (&UR)[4], const double (&FR)[4], const Wave<FLUX>& wR,
                                         double (&H)[4]) {
  if constexpr (FLUX == 0) {
    llf2(UL, FL, wL.lam, UR, FR, wR.lam, H);
  } else {
    const double SL = fmin(wL.vn - wL.c, wR.vn - wR.c), SR = fmax(wL.vn + wL.c, wR.vn + wR.c);
    if (SL >= 0.0) {
#pragma unroll
      for (int v = 0; v < 4; ++v) H[v] = 2.0 * FL[v];
    } else if (SR <= 0.0) {
#pragma unroll
      for (int v = 0; v < 4; ++v) H[v] = 2.0 * FR[v];
    } else if (EOS == 1) {
      const double k = 2.0 * rcp_fast(SR - SL);
#pragma unroll
      for (int v = 0; v < 4; ++v) H[v] = k * (SR * FL[v] - SL * FR[v] + SL * SR * (UR[v] - UL[v]));
    } else {
      constexpr int n = 1 + DIR, tg = 2 - DIR;
      const double mL = UL[0] * (SL - wL.vn), mR = UR[0] * (SR - wR.vn);
      const double Ss = (wR.pr - wL.pr + UL[n] * (SL - wL.vn) - UR[n] * (SR - wR.vn)) * rcp_fast_signed(mL - mR);
      const bool left = Ss >= 0.0;
      const double S = left ? SL : SR, vK = left ? wL.vn : wR.vn, pK = left ? wL.pr : wR.pr;
      double U[4], F[4];
#pragma unroll
      for (int v = 0; v < 4; ++v) { U[v] = left ? UL[v] : UR[v]; F[v] = left ? FL[v] : FR[v]; }
      const double rinv = rcp_fast(U[0]);
      const double m = U[0] * (S - vK);                       // rho_K (S_K - v_K)
      const double fac = m * rcp_fast_signed(S - Ss);
      double Us[4];
      Us[0] = fac;
      Us[n] = fac * Ss;
      Us[tg] = fac * (U[tg] * rinv);
      Us[3] = fac * (U[3] * rinv + (Ss - vK) * (Ss + pK * rcp_fast_signed(m)));
#pragma unroll
      for (int v = 0; v < 4; ++v) H[v] = 2.0 * fma(S, Us[v] - U[v], F[v]);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Trace of a cell at eta = -1/+1 (node stride `s` doubles: 32 inside a tile)
// ---------------------------------------------------------------------------------------------
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

// A read-only global load the compiler may not move: issued where it is written (a prefetch into registers
// for a later row), not sunk to its first use.
__device__ __forceinline__ double ldg_here(const double* p) {
  double v;
  asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(v) : "l"(p));
  return v;
}

__device__ __forceinline__ double shfl_up1(double x) { return __shfl_up_sync(FULL, x, 1); }
__device__ __forceinline__ double shfl_dn1(double x) { return __shfl_down_sync(FULL, x, 1); }
__device__ __forceinline__ Wave<0> shfl_dn1(const Wave<0>& w) { return Wave<0>{shfl_dn1(w.lam)}; }
__device__ __forceinline__ Wave<1> shfl_dn1(const Wave<1>& w) {
  return Wave<1>{shfl_dn1(w.vn), shfl_dn1(w.c), shfl_dn1(w.pr)};
}

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

__device__ __forceinline__ void bulk_prefetch_l2(const void* src, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
// orders earlier generic-proxy accesses of shared memory before later async-proxy (TMA) writes
__device__ __forceinline__ void fence_proxy_async() {
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// ---------------------------------------------------------------------------------------------
// The fused RK-stage kernel (rows a2..a12 of SURVEY.md 8(a); a1/a4's basis change is folded into
// the tables, see dg_tables.h).  Writes
//     out = a u^n + b u^(s-1) + beta N(u^(s-1)),     beta = b dt,
// with beta (and the 1/2 of the Lax-Friedrichs average) folded into the derivative / lifting tables
// and the gravity constants on the host; K_RHS: a = b = 0, beta = 1.
//
// Shared memory of one thread block (M warps, one 32-cell column block, `rows` rows):
//   tiles[3]  ring of u^(s-1) tiles (rows j-1 | j | j+1 | j+2 rotating), each one contiguous
//             4 M^2 x 32 doubles in HBM -> filled by ONE cp.async.bulk (TMA) each, mbarrier-tracked;
//             the copy for row j+2 is in flight while row j is computed
//   sN        first the landing buffer of the row's u^n tile (TMA, issued as soon as the previous
//             row has let go of it), then a u^n + the x-direction part of beta N
//             ([v][r][q][lane]; transposes ownership from eta-lines to xi-columns)
//   sRi       1/sqrt(x^2+y^2+eps^2) at the row's volume nodes (shared by c_s^2 and the star gravity)
//   sAvg      partial cell averages of the row just written (fused CFL reduction, row a10)
// ---------------------------------------------------------------------------------------------
constexpr int NST = 3;
// Depth of the tile ring per order.  Deeper rings for the low orders (8 slots at order 1, 5 at order 2, whose rows are
// short and tiles small) were measured and changed nothing (1024^2 / 2048^2: order 1 0.33 / 0.42 of the copy
// bandwidth either way, order 2 0.58 / 0.68 against 0.61 / 0.71): those orders are bound by the latency of one
// warp's row, not by the prefetch distance.
template <int M> struct StageRing { static constexpr int value = NST; };

template <int M>
constexpr size_t stage_smem_bytes() {
  // tiles + sN + sRi + sAvg + mbarriers
  return ((size_t)(StageRing<M>::value + 1) * 4 * M * M * 32 + (size_t)M * M * 32 + (size_t)4 * M * 32) * sizeof(double) + 128;
}

// Warps per thread block: M workers, plus -- at M = 5, in the stages that carry the fused CFL reduction -- one helper
// warp that issues the TMA copies / prefetches and does that reduction.  It costs no occupancy there (registers are
// allocated to warps in groups of four, so 2 x 6 warps of 168 registers fit exactly like 2 x 5) and takes ~150
// instructions per row off worker warp 0's critical path: last stage 0.645 ms instead of 0.670 at 1024^2.  In the
// stages without the reduction the extra warp only costs (+2 % measured), so they keep M warps.
template <int M, int KIND> struct StageWarps {
  static constexpr int helper = (M == 5 && (KIND == K_LAST || KIND == K_LASTD || KIND == K_GENL)) ? 1 : 0;
  static constexpr int threads = (M + helper) * 32;
};

template <int M, int EOS, int GRAV, int KIND, int MINB, int FLUX = 0>
__global__ void __launch_bounds__((StageWarps<M, KIND>::threads), MINB)
stage_kernel(const __grid_constant__ StageArgs A) {
  constexpr bool grav = GRAV != G_NONE;
  constexpr bool need_ri = EOS == 1 || grav;
  constexpr bool gen = KIND == K_GEN || KIND == K_GENL;
  constexpr bool add_u = KIND != K_RHS;
  constexpr bool use_un = KIND == K_MID || KIND == K_LAST || KIND == K_LASTD || gen;
  constexpr bool do_cfl = KIND == K_LAST || KIND == K_LASTD || KIND == K_GENL;
  constexpr bool do_damp = KIND == K_LASTD || KIND == K_GENL;    // K_GENL: only if the zone is enabled
  constexpr int NS = StageRing<M>::value;        // slots of the tile ring
  constexpr int C = 4 * M * M;                   // doubles per cell
  constexpr int BS = C * 32;                     // doubles per 32-cell tile
  constexpr uint32_t TILE_BYTES = BS * sizeof(double);
  extern __shared__ __align__(128) double smem[];
  double* tiles = smem;
  double* sN = tiles + NS * BS;
  double* sRi = sN + BS;                         // [r][q][lane]
  double* sAvg = sRi + M * M * 32;               // [v][q][lane]
  uint64_t* mbar = reinterpret_cast<uint64_t*>(sAvg + 4 * M * 32);   // [NS] tiles, [NS] u^n

  const int tid = threadIdx.x;
  const int lane = tid & 31;
  const int w = tid >> 5;                        // eta-line (X phase) / xi-column (Y phase)
  constexpr bool HELPER = StageWarps<M, KIND>::helper != 0;
  constexpr int ISSUER = HELPER ? M * 32 : 0;    // the thread that issues copies and prefetches
  constexpr int CFLW = HELPER ? M : 0;           // the warp that does the fused CFL reduction
  const bool worker = w < M;
  const int ib = blockIdx.x;
  const int i = ib * 32 + lane;
  const Geom& g = A.g;
  const DevTables& T = A.T;
  const bool valid = i < g.nx;
  const int last_lane = min(31, g.nx - 1 - ib * 32);
  const bool regA = (int)blockIdx.y < A.nblkA;
  const int j0 = regA ? A.rowA0 + (int)blockIdx.y * A.rows : A.rowB0 + ((int)blockIdx.y - A.nblkA) * A.rows;
  const int j1 = min(regA ? A.rowA1 : A.rowB1, j0 + A.rows);
  const size_t row_stride = (size_t)g.nbx * BS;

  const double xc = g.x0 + (i + 0.5) * g.dx;
  const double xW = g.x0 + i * g.dx, xE = g.x0 + (i + 1) * g.dx;
  const double xq_col = xc + g.hdx * T.xi[worker ? w : 0];    // x of this thread's column (Y phase)

  // x-neighbour cells outside this block: (cell index, or -1 when there is none).  Lanes 0..7 of
  // warp r fetch line r of those two cells straight from L2 (their own blocks are loading the same
  // rows at about the same time): lane = side * 4 + v.
  const int iLn = ib > 0 ? ib * 32 - 1 : (g.bc == 0 ? g.nx - 1 : -1);
  const int iRn = ib * 32 + 32 < g.nx ? ib * 32 + 32 : (g.bc == 0 ? 0 : -1);
  const bool haveL = iLn >= 0, haveR = iRn >= 0;
  const double* edge_src = nullptr;
  if (lane < 8 && worker) {
    const int ic = lane < 4 ? iLn : iRn;
    if (ic >= 0) edge_src = A.qprev + (size_t)(ic >> 5) * BS + (ic & 31) + (size_t)(((lane & 3) * M + w) * M) * 32;
  }

  // tile t holds row j0-1+t: wrapped for periodic domains; the neighbour strip's row (-2 south, -3 north) when
  // the domain is one strip of a decomposition along y; absent (-1) outside a non-periodic domain
  auto tile_row = [&](int t) -> int {
    const int jj = j0 - 1 + t;
    if (jj < 0) return A.haloS ? -2 : (g.bc == 0 ? g.ny - 1 : -1);
    if (jj >= g.ny) return A.haloN ? -3 : (g.bc == 0 ? 0 : -1);
    return jj;
  };
  auto tile_issue = [&](int t) {                 // thread 0 only
    const int jr = tile_row(t);
    if (jr != -1) {
      uint64_t* bar = mbar + t % NS;
      const double* src = jr >= 0 ? A.qprev + jr * row_stride : (jr == -2 ? A.haloS : A.haloN);
      mbar_expect_tx(bar, TILE_BYTES);
      bulk_g2s(tiles + (t % NS) * BS, src + (size_t)ib * BS, TILE_BYTES, bar);
    }
  };
  // k-th copy into a slot completes mbarrier phase k; tile 0 is the only one that can be absent
  // and still be followed by later copies into its slot (non-periodic bottom row)
  const int skip0 = tile_row(0) == -1 ? 1 : 0;
  auto tile_wait = [&](int t) {
    if (tile_row(t) != -1) mbar_wait(mbar + t % NS, (uint32_t)((t / NS - (t % NS == 0 ? skip0 : 0)) & 1));
  };
  auto un_issue = [&](int j) {                   // thread 0 only; u^n tile of row j -> sN
    mbar_expect_tx(mbar + NS, TILE_BYTES);
    bulk_g2s(sN, A.qn + (size_t)j * row_stride + (size_t)ib * BS, TILE_BYTES, mbar + NS);
  };
  // the last stage also reads the initial state where the wave-killing zone is active: pull that
  // tile into L2 ahead of its use (cheap test on the tile's farthest corner)
  auto prefetch_q0 = [&](int j) {                // thread 0 only
    const double xl = g.x0 + ib * 32 * g.dx, xr = g.x0 + (ib * 32 + 32) * g.dx;
    const double yl = g.y0 + j * g.dy, yr = g.y0 + (j + 1) * g.dy;
    const double xa = fmax(fabs(xl), fabs(xr)), ya = fmax(fabs(yl), fabs(yr));
    bool want = xa * xa + ya * ya > A.D.r0 * A.D.r0;
    if (A.D.in_r0 > 0.0 && !want) {              // inner zone: the tile's nearest point to the origin
      const double xn = (xl <= 0.0 && xr >= 0.0) ? 0.0 : fmin(fabs(xl), fabs(xr));
      const double yn = (yl <= 0.0 && yr >= 0.0) ? 0.0 : fmin(fabs(yl), fabs(yr));
      want = xn * xn + yn * yn < A.D.in_r0 * A.D.in_r0;
    }
    if (want) bulk_prefetch_l2(A.q0 + (size_t)j * row_stride + (size_t)ib * BS, TILE_BYTES);
  };

  // general sub-steps read earlier stage states in the epilogue: pull the row's tiles into L2 ahead
  auto prefetch_gen = [&](int j) {               // issuing thread only
    const size_t off = (size_t)j * row_stride + (size_t)ib * BS;
    for (int k = 0; k < A.nk; ++k) bulk_prefetch_l2(A.kin[k] + off, TILE_BYTES);
  };

  if (tid == ISSUER) {
#pragma unroll
    for (int s = 0; s <= NS; ++s) mbar_init(mbar + s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  constexpr int PFD = NS - 2;                    // rows ahead at which the u^n tile is pulled into L2
  if (tid == ISSUER) {
#pragma unroll
    for (int s = 0; s < NS; ++s)
      if (s <= j1 - j0 + 1) tile_issue(s);       // tiles 0 .. rows + 1 are all a segment needs
    if (use_un) un_issue(j0);
    if (use_un) {
#pragma unroll
      for (int d = 1; d < PFD; ++d)
        if (j0 + d < j1) bulk_prefetch_l2(A.qn + (size_t)(j0 + d) * row_stride + (size_t)ib * BS, TILE_BYTES);
    }
    if (do_damp) prefetch_q0(j0);
    if (gen && A.gen_pf) prefetch_gen(j0);
  }

  // line r = w of the two out-of-block x-neighbours, fetched one row ahead (lanes 0..7)
  double eraw[M];
#pragma unroll
  for (int q = 0; q < M; ++q) eraw[q] = edge_src ? __ldg(edge_src + (size_t)j0 * row_stride + q * 32) : 0.0;

  // numerical flux (x2) through the south face of the segment's first row, column q = w: the only
  // face whose two sides are both evaluated here; afterwards a row's N flux is the next row's S flux
  double HS[4];
  double spmax = 0.0;                            // running CFL wave-speed maximum of this lane (warp CFLW)
  if (worker) {
    const double yS = g.y0 + j0 * g.dy;
    double cs2 = 0.0, ciso = 0.0;
    if (EOS == 1) {
      cs2 = A.ph.h2gm * rsqrt_fast(fma(xq_col, xq_col, fma(yS, yS, A.ph.eps2s)));
      ciso = sqrt_fast(cs2);
    }
    double US[4], GSo[4], bU[4], bG[4];
    Wave<FLUX> lamSo, bLam;
    tile_wait(1);
    column_trace<M>(tiles + BS + lane, 32, w, T.Im, US);
    face_flux<EOS, 1, FLUX>(A.ph, US, cs2, ciso, GSo, lamSo);
    if (tile_row(0) != -1) {
      tile_wait(0);
      column_trace<M>(tiles + lane, 32, w, T.Ip, bU);
      face_flux<EOS, 1, FLUX>(A.ph, bU, cs2, ciso, bG, bLam);
    } else if (g.bc == 2) {
#pragma unroll
      for (int v = 0; v < 4; ++v) bU[v] = __ldg(A.btrS + ((size_t)(ib * 4 + v) * M + w) * 32 + lane);
      face_flux<EOS, 1, FLUX>(A.ph, bU, cs2, ciso, bG, bLam);
    } else {                                     // transmissive bottom boundary
#pragma unroll
      for (int v = 0; v < 4; ++v) { bU[v] = US[v]; bG[v] = GSo[v]; }
      bLam = lamSo;
    }
    riemann2<FLUX, EOS, 1>(bU, bG, bLam, US, GSo, lamSo, HS);
  }
  __syncthreads();                               // tile 0's slot may be refilled

  for (int j = j0; j < j1; ++j) {
    const int t = j - j0 + 1;                    // tile index of row j
    const bool more = j + 1 < j1;
    if (tid == ISSUER) {
      fence_proxy_async();                       // the slots about to be refilled were read through the generic proxy
      if (t - 1 + NS <= j1 - j0 + 1) tile_issue(t - 1 + NS);   // -> the slot row j-1 has just left (NS = 3: row j+2)
      if (use_un && j > j0) un_issue(j);         // sN is free again
      if (use_un && j + PFD < j1)                // so that a later row's copy comes from L2
        bulk_prefetch_l2(A.qn + (size_t)(j + PFD) * row_stride + (size_t)ib * BS, TILE_BYTES);
      if (do_damp && more) prefetch_q0(j + 1);
      if (gen && A.gen_pf == 2 && more) prefetch_gen(j + 1);
      if (gen && A.gen_pf == 1 && j > j0) prefetch_gen(j);
    }
    const double* tu = tiles + (t % NS) * BS + lane;
    const double yc = g.y0 + (j + 0.5) * g.dy;

    // fused CFL wave speed of the row finished in the previous iteration (row a10)
    if (do_cfl && w == CFLW && j > j0) {
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
        const double ycp = g.y0 + (j - 0.5) * g.dy;
        const double rinv = rcp_fast(avg[0]);    // slow-path-free: this warp is the row's critical path
        const double vx = avg[1] * rinv, vy = avg[2] * rinv;
        double c;
        if (EOS == 0) c = sqrt_fast(A.ph.gamma * A.ph.gm1 * (avg[3] - 0.5 * (avg[1] * vx + avg[2] * vy)) * rinv);
        else          c = sqrt_fast(A.ph.h2gm * rsqrt_fast(fma(xc, xc, fma(ycp, ycp, A.ph.eps2s))));
        sp = (fabs(vx) + c) * g.inv_dx + (fabs(vy) + c) * g.inv_dy;
        if (!(sp >= 0.0)) sp = __longlong_as_double(0x7ff0000000000000LL);   // NaN -> +inf
      }
      spmax = fmax(spmax, sp);                   // per lane; reduced once after the last row
    }

    // =========================== X phase: eta-line r = w ===========================
    double enext[M];                             // next row's edge lines: in flight during this whole row
#pragma unroll
    for (int q = 0; q < M; ++q)
      enext[q] = (edge_src && more) ? ldg_here(edge_src + (size_t)(j + 1) * row_stride + q * 32) : 0.0;
    if (worker) {
      const int r = w;
      // (no wait for tile t here: this warp has seen its mbarrier phase complete already -- as tile t of the S face in
      // the prologue, or as the row above in the previous row's Y phase; a second try_wait costs ~100 cycles per row)
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
      // traces of the two out-of-block neighbours: lane side*4+v reduces its line; lane 0 picks up the
      // left one (lanes 0..3), the last lane the right one (lanes 4..7)
      double etr = 0.0;
#pragma unroll
      for (int q = 0; q < M; ++q) etr = fma(lane < 4 ? T.Ip[q] : T.Im[q], eraw[q], etr);
      double UX[4];
#pragma unroll
      for (int v = 0; v < 4; ++v) UX[v] = __shfl_sync(FULL, etr, (lane == 0 ? 0 : 4) + v);
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
      double FWo[4], FEo[4];
      Wave<FLUX> lamWo, lamEo;
      face_flux<EOS, 0, FLUX>(A.ph, UW, cs2W, cW, FWo, lamWo);
      face_flux<EOS, 0, FLUX>(A.ph, UE, cs2E, cE, FEo, lamEo);
      double UR[4], FR[4];
      Wave<FLUX> lamR;
#pragma unroll
      for (int v = 0; v < 4; ++v) { UR[v] = shfl_dn1(UW[v]); FR[v] = shfl_dn1(FWo[v]); }
      lamR = shfl_dn1(lamWo);
      if (last_lane == 0) {                      // a one-cell block: lane 0 needs both neighbours
#pragma unroll
        for (int v = 0; v < 4; ++v) UR[v] = __shfl_sync(FULL, etr, 4 + v);
      } else if (lane == last_lane) {
#pragma unroll
        for (int v = 0; v < 4; ++v) UR[v] = UX[v];
      }
      if (lane == last_lane) {                   // right neighbour is outside this block
        if (!haveR) {
          if (g.bc == 1) {
#pragma unroll
            for (int v = 0; v < 4; ++v) UR[v] = UE[v];
          } else {
#pragma unroll
            for (int v = 0; v < 4; ++v) UR[v] = __ldg(A.btrE + ((size_t)j * 4 + v) * M + r);
          }
        }
        face_flux<EOS, 0, FLUX>(A.ph, UR, cs2E, cE, FR, lamR);
      }
      double HE[4], HW[4];
      riemann2<FLUX, EOS, 0>(UE, FEo, lamEo, UR, FR, lamR, HE);
#pragma unroll
      for (int v = 0; v < 4; ++v) HW[v] = shfl_up1(HE[v]);
      if (lane == 0) {                           // left neighbour is outside this block
        double UL[4], FL[4];
        Wave<FLUX> lamL;
        if (haveL) {
#pragma unroll
          for (int v = 0; v < 4; ++v) UL[v] = UX[v];
        } else if (g.bc == 1) {
#pragma unroll
          for (int v = 0; v < 4; ++v) UL[v] = UW[v];
        } else {
#pragma unroll
          for (int v = 0; v < 4; ++v) UL[v] = __ldg(A.btrW + ((size_t)j * 4 + v) * M + r);
        }
        face_flux<EOS, 0, FLUX>(A.ph, UL, cs2W, cW, FL, lamL);
        riemann2<FLUX, EOS, 0>(UL, FL, lamL, UW, FWo, lamWo, HW);
      }
      // a u^n (landed in sN) + x-part of beta N
      if (use_un) mbar_wait(mbar + NS, (uint32_t)((t - 1) & 1));
#pragma unroll
      for (int v = 0; v < 4; ++v)
#pragma unroll
        for (int qq = 0; qq < M; ++qq) {
          double* p = sN + ((v * M + r) * M + qq) * 32 + lane;
          double val = fma(T.lxm[qq], HW[v], fma(-T.lxp[qq], HE[v], acc[v][qq]));
          if (use_un) val = fma(A.a, *p, val);
          *p = val;
        }
    }
    __syncthreads();

    if (gen && A.gen_pf == 3 && tid == (HELPER ? ISSUER : 32 % (M * 32))) prefetch_gen(j);
    // =========================== Y phase: xi-column q = w ===========================
    if (worker) {
      const int q = w;
      const double xq = xq_col;
      double acc[4][M];
#pragma unroll
      for (int v = 0; v < 4; ++v)
#pragma unroll
        for (int r = 0; r < M; ++r) acc[v][r] = 0.0;
      // wave-killing factors of this cell (row a12): out <- f0 u0 + ft out
      double f0 = 0.0, ft = 1.0;
      bool damp = false;
      if (do_damp && (KIND != K_GENL || A.D.on))
        damp = damp_factors(A.D, sqrt_fast(fma(xc, xc, yc * yc) + 1e-300), f0, ft);   // + tiny: a centre at the origin
      // the initial state of the damped cells: for M <= 4 requested here and used in the epilogue (the
      // loads have the whole Y phase to land); at M = 5 the 20 extra live doubles cost more than they
      // save (measured: 0.668 vs 0.637 ms for the last stage), so there the loads stay in the epilogue
      constexpr bool early_q0 = do_damp && M <= 4;
      double z0[4][M];
      if (early_q0) {
        const double* __restrict__ q0e = A.q0 + j * row_stride + (size_t)ib * BS + lane;
#pragma unroll
        for (int v = 0; v < 4; ++v)
#pragma unroll
          for (int rr = 0; rr < M; ++rr) z0[v][rr] = damp ? __ldg(q0e + ((v * M + rr) * M + q) * 32) : 0.0;
      }
      double UN[4] = {0, 0, 0, 0};
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
            const double k = -A.ph.gmb * ri * ri * ri;
            gx = k * xq;
            gy = k * yr;
            if (GRAV == G_PLANET) {
              const double ddx = xq - A.ph.xp, ddy = yr - A.ph.yp;
              const double rpi = rsqrt_fast(fma(ddx, ddx, fma(ddy, ddy, A.ph.eps2p)));
              const double kp = -A.ph.qgmb * rpi * rpi * rpi;
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
        if (add_u) {                             // + b u^(s-1)  (b = 1 in the first stage)
#pragma unroll
          for (int v = 0; v < 4; ++v) acc[v][r] = KIND == K_FIRST ? acc[v][r] + u[v] : fma(A.b, u[v], acc[v][r]);
        }
      }
      // north face: own trace against the S trace of the row above (tile t+1)
      const double yN = g.y0 + (j + 1) * g.dy;
      double cs2N = 0.0, cN = 0.0;
      if (EOS == 1) {
        cs2N = A.ph.h2gm * rsqrt_fast(fma(xq, xq, fma(yN, yN, A.ph.eps2s)));
        cN = sqrt_fast(cs2N);
      }
      double GNo[4];
      Wave<FLUX> lamNo;
      face_flux<EOS, 1, FLUX>(A.ph, UN, cs2N, cN, GNo, lamNo);
      double aU[4], aG[4];
      Wave<FLUX> aLam;
      if (tile_row(t + 1) != -1) {
        tile_wait(t + 1);
        column_trace<M>(tiles + ((t + 1) % NS) * BS + lane, 32, q, T.Im, aU);
        face_flux<EOS, 1, FLUX>(A.ph, aU, cs2N, cN, aG, aLam);
      } else if (g.bc == 1) {
#pragma unroll
        for (int v = 0; v < 4; ++v) { aU[v] = UN[v]; aG[v] = GNo[v]; }
        aLam = lamNo;
      } else {
#pragma unroll
        for (int v = 0; v < 4; ++v) aU[v] = __ldg(A.btrN + ((size_t)(ib * 4 + v) * M + q) * 32 + lane);
        face_flux<EOS, 1, FLUX>(A.ph, aU, cs2N, cN, aG, aLam);
      }
      double HN[4];
      riemann2<FLUX, EOS, 1>(UN, GNo, lamNo, aU, aG, aLam, HN);

      // modal update in nodal form + RK combination (rows a8, a9) and store
      const size_t cell_off = j * row_stride + (size_t)ib * BS + lane;
      double* __restrict__ qo = A.qout + cell_off;
#pragma unroll
      for (int v = 0; v < 4; ++v) {
        double avg = 0.0;
        // general sub-step: the earlier stage states of this variable's column, all requested before the first
        // use (independent loads in flight together; slots >= nk are predicated off)
        double gk[MAXK][M];
        if (gen) {
#pragma unroll
          for (int k = 0; k < MAXK; ++k)
#pragma unroll
            for (int rr = 0; rr < M; ++rr)
              gk[k][rr] = k < A.nk ? __ldg(A.kin[k] + cell_off + ((v * M + rr) * M + q) * 32) : 0.0;
        }
#pragma unroll
        for (int rr = 0; rr < M; ++rr) {
          const int e = ((v * M + rr) * M + q) * 32;
          double out = sN[e + lane] + acc[v][rr];
          out = fma(T.lym[rr], HS[v], fma(-T.lyp[rr], HN[v], out));
          if (gen) {
            if (KIND == K_GEN && A.zout && valid) A.zout[cell_off + e] = out;
#pragma unroll
            for (int k = 0; k < MAXK; ++k) out = fma(A.kc[k], gk[k][rr], out);   // kc = 0 beyond nk
          }
          if (do_damp && damp) out = fma(f0, early_q0 ? z0[v][rr] : __ldg(A.q0 + cell_off + e), ft * out);
          if (valid) qo[e] = out;
          if (do_cfl) avg = fma(T.w[rr], out, avg);
        }
        if (do_cfl) sAvg[(v * M + q) * 32 + lane] = 0.25 * T.w[q] * avg;
      }
#pragma unroll
      for (int v = 0; v < 4; ++v) HS[v] = HN[v];   // this row's N face is the next row's S face
    }
#pragma unroll
    for (int q = 0; q < M; ++q) eraw[q] = enext[q];   // consumed only now: the loads had the whole row to land
    __syncthreads();
  }
  // CFL wave speed of the last row of the segment, then one reduction per thread block
  if (do_cfl && w == CFLW) {
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
damp_kernel(double* __restrict__ Q, const double* __restrict__ Q0, Geom g, DampArgs D) {
  const int lane = threadIdx.x & 31;
  const int j = blockIdx.y * 4 + (threadIdx.x >> 5);
  const int ib = blockIdx.x;
  const int i = ib * 32 + lane;
  constexpr int C = 4 * M * M;
  if (j >= g.ny || i >= g.nx) return;
  const double xc = g.x0 + (i + 0.5) * g.dx, yc = g.y0 + (j + 0.5) * g.dy;
  double f0, ft;
  if (!damp_factors(D, sqrt(xc * xc + yc * yc), f0, ft)) return;
  const size_t base = ((size_t)j * g.nbx + ib) * C * 32 + lane;
  if (D.mode == 1) {
#pragma unroll 1
    for (int n = 0; n < M * M; ++n) {
      double u[4], u0[4];
#pragma unroll
      for (int v = 0; v < 4; ++v) { u[v] = Q[base + (v * M * M + n) * 32]; u0[v] = Q0[base + (v * M * M + n) * 32]; }
      damp_node_primitive(f0, ft, D.gm1, u, u0);
#pragma unroll
      for (int v = 0; v < 4; ++v) Q[base + (v * M * M + n) * 32] = u[v];
    }
    return;
  }
#pragma unroll 4
  for (int e = 0; e < C; ++e) Q[base + e * 32] = fma(f0, Q0[base + e * 32], ft * Q[base + e * 32]);
}

}  // namespace dg
