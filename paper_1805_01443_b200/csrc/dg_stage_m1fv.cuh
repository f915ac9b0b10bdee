// Stage kernel of DG order 1 (one mode, one node per cell: a first-order finite-volume update), the same operator as
// dg::stage_kernel<1, ...> evaluates (rows a2..a12 of SURVEY.md 8(a); the volume integral vanishes because the basis
// function is constant) but laid out for what order 1 is: 32 B of state per cell and ~170 fp64 operations.
//
// dg::stage_kernel gives an order-1 tile row to ONE warp that walks through the tile ring, two mbarrier waits, a
// shared-memory hand-over between its own X and Y phase and the divergent tile-edge code: ~400 instructions per row in
// one dependent chain, and the path is bound by instruction issue per cell.  Here a warp still owns one 32-cell
// column block and marches over `rows` rows -- each y-face is evaluated once and carried to the next row in registers,
// each interior x-face once and handed to the right neighbour by shuffle, so the interface flux stays single valued to
// the last bit -- but everything lives in registers: rows come by plain coalesced loads issued two rows ahead, nothing
// goes through shared memory, there is no barrier, and what does not change along the march (x-dependent terms,
// pointers, boundary flags) is set up once.  4 warps per block, each with its own segment of rows.
// Not used for grids whose last 32-cell block holds a single cell (that lane would need both x-neighbours): the launch
// code falls back to dg::stage_kernel there.
#pragma once
#include "dg_kernels.cuh"

namespace dg {

constexpr int M1_WARPS = 4;

template <int EOS, int GRAV, int KIND, int FLUX = 0>
__global__ void __launch_bounds__(M1_WARPS * 32, 4)
stage_kernel_m1(const __grid_constant__ StageArgs A) {
  constexpr bool grav = GRAV != G_NONE;
  constexpr bool gen = KIND == K_GEN || KIND == K_GENL;
  constexpr bool add_u = KIND != K_RHS;
  constexpr bool use_un = KIND == K_MID || KIND == K_LAST || KIND == K_LASTD || gen;
  constexpr bool do_cfl = KIND == K_LAST || KIND == K_LASTD || KIND == K_GENL;
  constexpr bool do_damp = KIND == K_LASTD || KIND == K_GENL;    // K_GENL: only if the zone is enabled
  constexpr int BS = 4 * 32;                     // doubles per 32-cell tile

  const int lane = threadIdx.x & 31;
  const int seg = (int)blockIdx.y * M1_WARPS + (int)(threadIdx.x >> 5);   // this warp's segment of rows
  const Geom& g = A.g;
  const int nsegB = A.rowB1 > A.rowB0 ? (A.rowB1 - A.rowB0 + A.rows - 1) / A.rows : 0;
  if (seg >= A.nblkA + nsegB) return;
  const bool regA = seg < A.nblkA;
  const int j0 = regA ? A.rowA0 + seg * A.rows : A.rowB0 + (seg - A.nblkA) * A.rows;
  const int j1 = min(regA ? A.rowA1 : A.rowB1, j0 + A.rows);
  const int ib = blockIdx.x;
  const int i = ib * 32 + lane;
  const bool valid = i < g.nx;
  const int last_lane = min(31, g.nx - 1 - ib * 32);
  const size_t row_stride = (size_t)g.nbx * BS;
  const size_t col = (size_t)ib * BS + lane;

  // what does not change along the march
  const double xc = g.x0 + (i + 0.5) * g.dx;
  const double xW = g.x0 + i * g.dx, xE = g.x0 + (i + 1) * g.dx;
  const double lxm = A.T.lxm[0], lxp = A.T.lxp[0], lym = A.T.lym[0], lyp = A.T.lyp[0];

  // the x-neighbour outside this 32-cell block that this lane needs: lane 0 the cell on its left, the last lane the
  // cell on its right; -1: there is none (domain boundary)
  const int iLn = ib > 0 ? ib * 32 - 1 : (g.bc == 0 ? g.nx - 1 : -1);
  const int iRn = ib * 32 + 32 < g.nx ? ib * 32 + 32 : (g.bc == 0 ? 0 : -1);
  const bool edgeL = lane == 0, edgeR = lane == last_lane;
  const int inb = edgeL ? iLn : (edgeR ? iRn : -1);
  const double* nbp = inb >= 0 ? A.qprev + (size_t)(inb >> 5) * BS + (inb & 31) + (size_t)j0 * row_stride : nullptr;
  const double* btrX = (edgeL ? A.btrW : A.btrE) + (size_t)j0 * 4;        // bc 2: trace of the initial state beyond the x-edge

  // source of row jj of the array qprev: wrapped for periodic domains; the neighbour strip's row when the domain is one
  // strip of a decomposition along y; null outside a non-periodic domain
  auto row_ptr = [&](int jj) -> const double* {
    if (jj < 0) return A.haloS ? A.haloS + col : (g.bc == 0 ? A.qprev + (size_t)(g.ny - 1) * row_stride + col : nullptr);
    if (jj >= g.ny) return A.haloN ? A.haloN + col : (g.bc == 0 ? A.qprev + col : nullptr);
    return A.qprev + (size_t)jj * row_stride + col;
  };
  auto load4 = [&](const double* p, double (&u)[4]) {
#pragma unroll
    for (int v = 0; v < 4; ++v) u[v] = p ? ldg_here(p + v * 32) : 0.0;
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

  // rows in flight: cur = row j, nxt = row j+1 (the N face needs it), far = row j+2 (requested now); the out-of-block
  // x-neighbour of the current row and of the next
  double cur[4], nxt[4], far[4], nbc[4], nbn[4];
  double HS[4];                                  // numerical flux (x2) through the row's S face
  const double* pnext = row_ptr(j0 + 1);         // row j+1 ...
  const bool top_open = row_ptr(j1) == nullptr;  // ... which does not exist above the last row of a non-periodic domain
  load4(A.qprev + (size_t)j0 * row_stride + col, cur);
  load4(nbp, nbc);
  {
    double below[4];
    const double* pb = row_ptr(j0 - 1);
    load4(pb, below);
    load4(pnext, nxt);
    if (j0 + 1 < j1) load4(nbp ? nbp + row_stride : nullptr, nbn);
    // S face of the first row: the only y-face whose two sides are both fetched for it
    if (!pb) {                                   // bottom of a non-periodic domain
#pragma unroll
      for (int v = 0; v < 4; ++v) below[v] = g.bc == 2 ? __ldg(A.btrS + (size_t)(ib * 4 + v) * 32 + lane) : cur[v];
    }
    y_flux(below, cur, g.y0 + j0 * g.dy, HS);
  }
  double spmax = 0.0;
  size_t cell_off = (size_t)j0 * row_stride + col;

  for (int j = j0; j < j1; ++j, cell_off += row_stride) {
    // requests for later rows and for the other arrays of this cell, before the arithmetic
    if (j + 2 <= j1) load4(row_ptr(j + 2), far);       // (row j1 is only the last row's N neighbour)
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

    // ---- W/E faces: each interior face once, by the cell on its left, handed to the right neighbour ----
    double cs2W, cW, cs2E, cE;
    cs_at(xW, yc, cs2W, cW);
    cs_at(xE, yc, cs2E, cE);
    double FWo[4], FEo[4];
    Wave<FLUX> wWo, wEo;
    face_flux<EOS, 0, FLUX>(A.ph, u, cs2W, cW, FWo, wWo);
    face_flux<EOS, 0, FLUX>(A.ph, u, cs2E, cE, FEo, wEo);
    // the state beyond the block's edge, for the two lanes that have one: neighbour cell, or the boundary condition
    double ux[4];
#pragma unroll
    for (int v = 0; v < 4; ++v) ux[v] = inb >= 0 ? nbc[v] : (g.bc == 1 ? u[v] : ((edgeL || edgeR) ? __ldg(btrX + (size_t)(j - j0) * 4 + v) : 0.0));
    double UR[4], FR[4];
    Wave<FLUX> wR;
#pragma unroll
    for (int v = 0; v < 4; ++v) { UR[v] = shfl_dn1(u[v]); FR[v] = shfl_dn1(FWo[v]); }
    wR = shfl_dn1(wWo);
    if (edgeR) {                                 // right neighbour is outside this block
#pragma unroll
      for (int v = 0; v < 4; ++v) UR[v] = ux[v];
      face_flux<EOS, 0, FLUX>(A.ph, UR, cs2E, cE, FR, wR);
    }
    double HE[4], HW[4];
    riemann2<FLUX, EOS, 0>(u, FEo, wEo, UR, FR, wR, HE);
#pragma unroll
    for (int v = 0; v < 4; ++v) HW[v] = shfl_up1(HE[v]);
    if (edgeL) {                                 // left neighbour is outside this block
      double FL[4];
      Wave<FLUX> wL;
      face_flux<EOS, 0, FLUX>(A.ph, ux, cs2W, cW, FL, wL);
      riemann2<FLUX, EOS, 0>(ux, FL, wL, u, FWo, wWo, HW);
    }

    // ---- N face against the row above ----
    double HN[4];
    if (j + 1 == j1 && top_open) {               // top of a non-periodic domain
      double hi[4];
#pragma unroll
      for (int v = 0; v < 4; ++v) hi[v] = g.bc == 2 ? __ldg(A.btrN + (size_t)(ib * 4 + v) * 32 + lane) : u[v];
      y_flux(u, hi, g.y0 + (j + 1) * g.dy, HN);
    } else {
      y_flux(u, nxt, g.y0 + (j + 1) * g.dy, HN);
    }

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

    // ---- update (rows a8, a9): a u^n + b u + beta N, beta folded into the lifting constants and the gravity ----
    double res[4];
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      double out = fma(lxm, HW[v], fma(-lxp, HE[v], src[v]));
      out = fma(lym, HS[v], fma(-lyp, HN[v], out));
      if (add_u) out = KIND == K_FIRST ? out + u[v] : fma(A.b, u[v], out);
      if (use_un) out = fma(A.a, un[v], out);
      if (gen) {
        if (KIND == K_GEN && A.zout && valid) A.zout[cell_off + v * 32] = out;
#pragma unroll
        for (int k = 0; k < MAXK; ++k) out = fma(A.kc[k], gk[k][v], out);   // kc = 0 beyond nk
      }
      if (do_damp && damp) out = fma(f0, z0[v], ft * out);
      if (valid) A.qout[cell_off + v * 32] = out;
      res[v] = out;
    }
    if (do_cfl) {                                // fused CFL wave speed (row a10): the state is its own average
      double sp = 0.0;
      if (valid) {
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
#pragma unroll
    for (int v = 0; v < 4; ++v) { HS[v] = HN[v]; cur[v] = nxt[v]; nxt[v] = far[v]; nbc[v] = nbn[v]; }
    if (j + 2 < j1) load4(nbp ? nbp + (size_t)(j + 2 - j0) * row_stride : nullptr, nbn);
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
