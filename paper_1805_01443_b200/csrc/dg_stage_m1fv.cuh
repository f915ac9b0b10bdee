// Stage kernel of DG order 1 (one mode, one node per cell: a first-order finite-volume update), the same operator as
// dg::stage_kernel<1, ...> evaluates (rows a2..a12 of SURVEY.md 8(a); the volume integral vanishes because the basis
// function is constant) but laid out for what order 1 is: 32 B of state per cell and ~200 fp64 operations.
//
// dg::stage_kernel gives an order-1 tile row to ONE warp that walks through the tile ring, two mbarrier waits, a
// shared-memory hand-over between its own X and Y phase and the divergent tile-edge code: the path is bound by
// instruction issue per cell.  Here everything lives in registers and there is no divergent code in the row loop:
//   * a warp owns 30 cells of a row (lanes 1..30) and marches over `rows` rows; lanes 0 and 31 carry the two cells next
//     to them (wrapped, copied or frozen at the domain boundary as the boundary condition says), so that every lane
//     finds its x-neighbour by shuffle and no lane is special -- 2 lanes in 32 repeat a neighbour warp's loads and
//     fluxes, in exchange for a row loop without tile-edge branches (they cost every warp ~90 of ~490 instructions);
//   * each y-face is evaluated once and carried to the next row in registers, each x-face once (by the lane on its
//     left, same instructions on the same operands in the two warps that share a face), so the interface flux stays
//     single valued to the last bit;
//   * rows come by plain loads issued two rows ahead; the three row buffers and the two y-face fluxes rotate by
//     renaming (the loop body is written three times), not by register moves;
//   * c_s at an E face is the right neighbour's c_s at its W face (shuffle), nothing goes through shared memory, there
//     is no barrier, and what does not change along the march is set up once.
// 4 warps per block, each with its own segment of rows.
#pragma once
#include "dg_kernels.cuh"

namespace dg {

constexpr int M1_WARPS = 4;
constexpr int M1_OWN = 30;                       // cells per warp and row (lanes 1..M1_OWN)

template <int EOS, int GRAV, int KIND, int FLUX = 0>
__global__ void __launch_bounds__(M1_WARPS * 32, 4)
stage_kernel_m1(const __grid_constant__ StageArgs A) {
  constexpr bool grav = GRAV != G_NONE;
  constexpr bool gen = KIND == K_GEN || KIND == K_GENL;
  constexpr bool add_u = KIND != K_RHS;
  constexpr bool use_un = KIND == K_MID || KIND == K_LAST || KIND == K_LASTD || gen;
  constexpr bool do_cfl = KIND == K_LAST || KIND == K_LASTD || KIND == K_GENL;
  constexpr bool do_damp = KIND == K_LASTD || KIND == K_GENL;    // K_GENL: only if the zone is enabled
  constexpr int BS = 4 * 32;                     // doubles per 32-cell tile of the state arrays

  const int lane = threadIdx.x & 31;
  const int seg = (int)blockIdx.y * M1_WARPS + (int)(threadIdx.x >> 5);   // this warp's segment of rows
  const Geom& g = A.g;
  const int nsegB = A.rowB1 > A.rowB0 ? (A.rowB1 - A.rowB0 + A.rows - 1) / A.rows : 0;
  if (seg >= A.nblkA + nsegB) return;
  const bool regA = seg < A.nblkA;
  const int j0 = regA ? A.rowA0 + seg * A.rows : A.rowB0 + (seg - A.nblkA) * A.rows;
  const int j1 = min(regA ? A.rowA1 : A.rowB1, j0 + A.rows);
  const size_t row_stride = (size_t)g.nbx * BS;

  // the cell at this lane's position (ic: -1 and nx are just outside the domain) and the cell whose state it reads
  const int ic = (int)blockIdx.x * M1_OWN - 1 + lane;
  const bool own = lane >= 1 && lane <= M1_OWN && ic < g.nx;
  int is = ic;
  if (ic < 0) is = g.bc == 0 ? g.nx - 1 : 0;                       // periodic: wrapped; else the cell inside (bc 1: its copy)
  else if (ic >= g.nx) is = (g.bc == 0 && ic == g.nx) ? 0 : g.nx - 1;
  const size_t col = (size_t)(is >> 5) * BS + (is & 31);
  // bc 2: the lane just outside the domain holds the trace of the initial state beyond that edge, btrW / btrE [j][v]
  const bool frozen = g.bc == 2 && (ic == -1 || ic == g.nx);
  const double* btrX = ic < 0 ? A.btrW : A.btrE;

  // what does not change along the march
  const double xc = g.x0 + (ic + 0.5) * g.dx;
  const double xW = g.x0 + ic * g.dx;
  const double lxm = A.T.lxm[0], lxp = A.T.lxp[0], lym = A.T.lym[0], lyp = A.T.lyp[0];

  // source of row jj of the array qprev.  Outside the rows of the domain: wrapped for periodic domains; the neighbour
  // strip's row when the domain is one strip of a decomposition along y; else the boundary condition as a row of its
  // own -- bc 2: the trace of the initial state beyond that edge (btrS / btrN have the layout of a row), bc 1: the row
  // inside (its copy)
  auto row_ptr = [&](int jj) -> const double* {
    if (jj < 0) return (A.haloS ? A.haloS : g.bc == 0 ? A.qprev + (size_t)(g.ny - 1) * row_stride : g.bc == 2 ? A.btrS : A.qprev) + col;
    if (jj >= g.ny) return (A.haloN ? A.haloN : g.bc == 0 ? A.qprev : g.bc == 2 ? A.btrN : A.qprev + (size_t)(g.ny - 1) * row_stride) + col;
    return A.qprev + (size_t)jj * row_stride + col;
  };
  // (one load per variable with a per-lane stride: a second, predicated load into the same registers for the frozen
  // lanes would wait for the first one to land -- a write-after-write dependency -- and make the prefetch synchronous)
  const int vs = frozen ? 1 : 32;
  auto load_row = [&](int jj, double (&u)[4]) {
    const double* p = frozen ? btrX + (size_t)min(max(jj, 0), g.ny - 1) * 4 : row_ptr(jj);
#pragma unroll
    for (int v = 0; v < 4; ++v) u[v] = ldg_here(p + v * vs);
  };
  auto cs_at = [&](double x, double y, double& cs2, double& c) {
    cs2 = 0.0; c = 0.0;
    if (EOS == 1) {
      cs2 = A.ph.h2gm * rsqrt_fast(fma(x, x, fma(y, y, A.ph.eps2s)));
      c = sqrt_fast(cs2);
    }
  };
  // numerical flux (x2) through the y-face at height yF between the states lo (below) and hi (above)
  auto y_flux = [&](const double (&lo)[4], const double (&hi)[4], double yF, double (&H)[4]) {
    double cs2, c, GL[4], GH[4];
    cs_at(xc, yF, cs2, c);
    Wave<FLUX> wl, wh;
    face_flux<EOS, 1, FLUX>(A.ph, lo, cs2, c, GL, wl);
    face_flux<EOS, 1, FLUX>(A.ph, hi, cs2, c, GH, wh);
    riemann2<FLUX, EOS, 1>(lo, GL, wl, hi, GH, wh, H);
  };
  double spmax = 0.0;

  // One row: cur = row j, nxt = row j+1 (requested a row ago), far = row j+2 (requested here); HS / HN = the numerical
  // flux (x2) through the row's S face (from the row below) and N face (evaluated here, the next row's HS).
  auto row = [&](int j, const double (&cur)[4], const double (&nxt)[4], double (&far)[4], const double (&HS)[4], double (&HN)[4]) {
    // requests for later rows and for the other arrays of this cell, before the arithmetic
    if (j + 2 <= j1) load_row(j + 2, far);       // (row j1 is only the last row's N neighbour)
    const size_t cell_off = (size_t)j * row_stride + col;
    double un[4], z0[4], gk[MAXK][4];
    const double yc = g.y0 + (j + 0.5) * g.dy;
    double f0 = 0.0, ft = 1.0;
    bool damp = false;
    if (do_damp && (KIND != K_GENL || A.D.on))
      damp = damp_factors(A.D, sqrt_fast(fma(xc, xc, yc * yc) + 1e-300), f0, ft);
    if (use_un) {
#pragma unroll
      for (int v = 0; v < 4; ++v) un[v] = __ldg(A.qn + cell_off + v * 32);
    }
    if (do_damp) {
#pragma unroll
      for (int v = 0; v < 4; ++v) z0[v] = damp ? __ldg(A.q0 + cell_off + v * 32) : 0.0;
    }
    if (gen) {
#pragma unroll
      for (int k = 0; k < MAXK; ++k)
#pragma unroll
        for (int v = 0; v < 4; ++v) gk[k][v] = k < A.nk ? __ldg(A.kin[k] + cell_off + v * 32) : 0.0;
    }
    const double (&u)[4] = cur;

    // ---- W/E faces: each face once, by the lane on its left, handed to the lane on its right ----
    double cs2W, cW;
    cs_at(xW, yc, cs2W, cW);
    const double cs2E = EOS == 1 ? shfl_dn1(cs2W) : 0.0, cE = EOS == 1 ? shfl_dn1(cW) : 0.0;
    double FWo[4], FEo[4];
    Wave<FLUX> wWo, wEo;
    face_flux<EOS, 0, FLUX>(A.ph, u, cs2W, cW, FWo, wWo);
    face_flux<EOS, 0, FLUX>(A.ph, u, cs2E, cE, FEo, wEo);
    double UR[4], FR[4];
#pragma unroll
    for (int v = 0; v < 4; ++v) { UR[v] = shfl_dn1(u[v]); FR[v] = shfl_dn1(FWo[v]); }
    const Wave<FLUX> wR = shfl_dn1(wWo);
    double HE[4], HW[4];
    riemann2<FLUX, EOS, 0>(u, FEo, wEo, UR, FR, wR, HE);
#pragma unroll
    for (int v = 0; v < 4; ++v) HW[v] = shfl_up1(HE[v]);

    // ---- gravity source (row a3) ----
    double src1 = 0.0, src2 = 0.0, src3 = 0.0;
    if (grav) {
      const double ri = rsqrt_fast(fma(xc, xc, fma(yc, yc, A.ph.eps2s)));
      const double k = -A.ph.gmb * ri * ri * ri;
      double gx = k * xc, gy = k * yc;
      if (GRAV == G_PLANET) {
        const double ddx = xc - A.ph.xp, ddy = yc - A.ph.yp;
        const double rpi = rsqrt_fast(fma(ddx, ddx, fma(ddy, ddy, A.ph.eps2p)));
        const double kp = -A.ph.qgmb * rpi * rpi * rpi;
        gx = fma(kp, ddx, gx);
        gy = fma(kp, ddy, gy);
      }
      src1 = u[0] * gx;
      src2 = u[0] * gy;
      src3 = fma(u[1], gx, u[2] * gy);
    }
    const double src[4] = {0.0, src1, src2, src3};

    // ---- N face against the row above (the top of a non-periodic domain is a row like any other: row_ptr) ----
    y_flux(u, nxt, g.y0 + (j + 1) * g.dy, HN);

    // ---- update (rows a8, a9): a u^n + b u + beta N, beta folded into the lifting constants and the gravity ----
    double res[4];
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      double out = fma(lxm, HW[v], fma(-lxp, HE[v], src[v]));
      out = fma(lym, HS[v], fma(-lyp, HN[v], out));
      if (add_u) out = KIND == K_FIRST ? out + u[v] : fma(A.b, u[v], out);
      if (use_un) out = fma(A.a, un[v], out);
      if (gen) {
        if (KIND == K_GEN && A.zout && own) A.zout[cell_off + v * 32] = out;
#pragma unroll
        for (int k = 0; k < MAXK; ++k) out = fma(A.kc[k], gk[k][v], out);   // kc = 0 beyond nk
      }
      if (do_damp && damp) out = fma(f0, z0[v], ft * out);
      if (own) A.qout[cell_off + v * 32] = out;
      res[v] = out;
    }
    if (do_cfl) {                                // fused CFL wave speed (row a10): the state is its own average
      double sp = 0.0;
      if (own) {
        const double rinv = rcp_fast(res[0]);
        const double vx = res[1] * rinv, vy = res[2] * rinv;
        double c;
        if (EOS == 0) c = sqrt_fast(A.ph.gamma * A.ph.gm1 * (res[3] - 0.5 * (res[1] * vx + res[2] * vy)) * rinv);
        else          c = sqrt_fast(A.ph.h2gm * rsqrt_fast(fma(xc, xc, fma(yc, yc, A.ph.eps2s))));
        sp = (fabs(vx) + c) * g.inv_dx + (fabs(vy) + c) * g.inv_dy;
        if (!(sp >= 0.0)) sp = __longlong_as_double(0x7ff0000000000000LL);   // NaN -> +inf
      }
      spmax = fmax(spmax, sp);
    }
  };

  double ra[4], rb[4], rc[4], Ha[4], Hb[4];
  load_row(j0, ra);
  {
    double below[4];
    load_row(j0 - 1, below);
    load_row(j0 + 1, rb);
    y_flux(below, ra, g.y0 + j0 * g.dy, Ha);     // S face of the first row: the only y-face fetched from both sides
  }
  // six rows per trip: the three row buffers rotate with period 3, the two face fluxes with period 2
  for (int j = j0; j < j1; j += 6) {
    row(j, ra, rb, rc, Ha, Hb);
    if (j + 1 < j1) row(j + 1, rb, rc, ra, Hb, Ha);
    if (j + 2 < j1) row(j + 2, rc, ra, rb, Ha, Hb);
    if (j + 3 < j1) row(j + 3, ra, rb, rc, Hb, Ha);
    if (j + 4 < j1) row(j + 4, rb, rc, ra, Ha, Hb);
    if (j + 5 < j1) row(j + 5, rc, ra, rb, Hb, Ha);
  }
  if (do_cfl) {
    unsigned long long bits = (unsigned long long)__double_as_longlong(spmax);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const unsigned long long other = __shfl_xor_sync(FULL, bits, o);
      bits = other > bits ? other : bits;
    }
    if (lane == 0) atomicMax(A.wmax, bits);
  }
}

}  // namespace dg
