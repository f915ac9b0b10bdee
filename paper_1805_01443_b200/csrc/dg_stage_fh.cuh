// Stage kernel with a helper warp: the same operator and the same arithmetic as
// dg::stage_kernel in dg_kernels.cuh, but one 32-cell tile row is worked on by M + 1 warps instead of M.
//
//   worker warp r (X phase) / q (Y phase), r, q < M
//       the volume work of its eta-line / xi-column, the W/E Riemann fluxes between the cells of the tile (neighbour
//       lanes, by shuffle), the N face of its column, lifting, RK combine, store.  Straight-line code: no out-of-tile
//       cells, no boundary conditions in x, no TMA bookkeeping, no polling of tile barriers.
//   helper warp (index M)
//       * the two faces where the tile meets its x-neighbours (lane = (side, eta-line)): the neighbour cell's line
//         from L2 (requested two rows ahead), the own edge cell's line from the tile, boundary conditions, Riemann
//         flux -> sHX, one row ahead.  dg::stage_kernel does this on lanes 0 and 31 of every worker behind divergent
//         branches (~130 of its ~1400 instructions per row) and carries the prefetched lines in 20 registers;
//       * TMA issue, mbarrier waits for the tiles, L2 prefetches, the fused CFL reduction, the cells' wave-killing
//         factors (last stage).
//
// Why a sixth warp is free: five warps of 168 registers make two blocks per SM = 10 warps; 12 x 168 x 32 registers still
// fit the register file (3 warps per scheduler), and the shared memory of a block does not grow (114.6 KB).
// Measured at 1024^2, order 5 (B200): first / middle / last stage 0.450 / 0.490 / 0.554 ms against 0.469 / 0.487 /
// 0.650 ms of dg::stage_kernel.  Variants that were built and measured slower: the helper
// also evaluating the N faces of all M columns (one warp's dependent chains became the critical path: 0.53 / 0.57 /
// 0.65), the helper computing c_s^2 and gravity of the volume nodes with a two-slot tile ring to make room for them
// (0.47 / 0.50 / 0.64).
//
// Synchronisation per row:
//   barrier 2 (workers only)   X phase done: sN and sRi of the row are complete
//   barrier 3 + w (worker w and the helper)   the tile of the row above has landed: worker w syncs on its own barrier
//                              before its N face, the helper arrives at all M early in the row -- one barrier per
//                              worker warp, so that this is no rendezvous of the workers
//   barrier 0 (everybody)      end of the row: sN, sRi, the ring slot of row j-1 may be overwritten; sHX of the next
//                              row (double buffered by row parity) is written
#pragma once
#include "dg_kernels.cuh"

namespace dg {

template <int M>
constexpr size_t stage_fh_smem_bytes() {
  // tiles[NST] + sN + sRi + sHS + sHX[2] + mbarriers
  return ((size_t)(NST + 1) * 4 * M * M * 32 + (size_t)M * M * 32 + (size_t)4 * M * 32 + (size_t)2 * M * 8) * sizeof(double) + 64;
}

__device__ __forceinline__ void bar_sync_named(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ void bar_arrive_named(int id, int nthreads) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// Numerical flux (x2) through the y-face between the row whose tile is `lo` (trace at eta = +1) and the row whose
// tile is `hi` (trace at eta = -1), column q, for the 32 cells of the tile (lane = cell; lo / hi already carry the
// lane offset).  A null tile is the outside of a non-periodic domain: transmissive (bc 1) copies the other side,
// frozen (bc 2) reads the initial state's trace from `btr`.
template <int M, int EOS, int FLUX>
__device__ __forceinline__ void y_face(const StageArgs& A, const double* lo, const double* hi, const double* btr,
                                       int q, double xq, double yF, double (&H)[4]) {
  double cs2 = 0.0, ciso = 0.0;
  if (EOS == 1) {
    cs2 = A.ph.h2gm * rsqrt_fast(fma(xq, xq, fma(yF, yF, A.ph.eps2s)));
    ciso = sqrt_fast(cs2);
  }
  double UL[4], GL[4], UH[4], GH[4];
  Wave<FLUX> wl, wh;
  if (lo) {
    column_trace<M>(lo, 32, q, A.T.Ip, UL);
    face_flux<EOS, 1, FLUX>(A.ph, UL, cs2, ciso, GL, wl);
  }
  if (hi) {
    column_trace<M>(hi, 32, q, A.T.Im, UH);
    face_flux<EOS, 1, FLUX>(A.ph, UH, cs2, ciso, GH, wh);
  }
  if (!lo) {
    if (A.g.bc == 2) {
#pragma unroll
      for (int v = 0; v < 4; ++v) UL[v] = __ldg(btr + (v * M + q) * 32);
      face_flux<EOS, 1, FLUX>(A.ph, UL, cs2, ciso, GL, wl);
    } else {
#pragma unroll
      for (int v = 0; v < 4; ++v) { UL[v] = UH[v]; GL[v] = GH[v]; }
      wl = wh;
    }
  }
  if (!hi) {
    if (A.g.bc == 2) {
#pragma unroll
      for (int v = 0; v < 4; ++v) UH[v] = __ldg(btr + (v * M + q) * 32);
      face_flux<EOS, 1, FLUX>(A.ph, UH, cs2, ciso, GH, wh);
    } else {
#pragma unroll
      for (int v = 0; v < 4; ++v) { UH[v] = UL[v]; GH[v] = GL[v]; }
      wh = wl;
    }
  }
  riemann2<FLUX, EOS, 1>(UL, GL, wl, UH, GH, wh, H);
}

template <int M, int EOS, int GRAV, int KIND, int MINB, int FLUX = 0>
__global__ void __launch_bounds__(((M + 1) * 32), MINB)
stage_kernel_fh(const __grid_constant__ StageArgs A) {
  constexpr bool grav = GRAV != G_NONE;
  constexpr bool need_ri = EOS == 1 || grav;
  constexpr bool gen = KIND == K_GEN || KIND == K_GENL;
  constexpr bool add_u = KIND != K_RHS;
  constexpr bool use_un = KIND == K_MID || KIND == K_LAST || KIND == K_LASTD || gen;
  constexpr bool do_cfl = KIND == K_LAST || KIND == K_LASTD || KIND == K_GENL;
  constexpr bool do_damp = KIND == K_LASTD || KIND == K_GENL;    // K_GENL: only if the zone is enabled
  constexpr int C = 4 * M * M;                   // doubles per cell
  constexpr int BS = C * 32;                     // doubles per 32-cell tile
  constexpr int NS = NST;
  constexpr int NWORK = M * 32;
  constexpr uint32_t TILE_BYTES = BS * sizeof(double);
  constexpr int NTHR = (M + 1) * 32;
  extern __shared__ __align__(128) double smem[];
  double* tiles = smem;
  double* sN = tiles + NS * BS;                  // u^n landing buffer -> a u^n + x-part of beta N -> (fused CFL) partial averages
  double* sRi = sN + BS;                         // [r][q][lane]: 1/sqrt(x^2+y^2+eps^2) at the row's volume nodes
  double* sHS = sRi + M * M * 32;                // [v][q][lane]: the N-face fluxes one worker evaluates for another (M = 5);
                                                 // the wave-killing factors of the row's cells (last stage)
  double* sHX = sHS + 4 * M * 32;                // [row parity][r][side][v]: W flux of cell 0, E flux of the last cell
  uint64_t* mbar = reinterpret_cast<uint64_t*>(sHX + 2 * M * 8);   // [NS] tiles, u^n

  const int tid = threadIdx.x;
  const int lane = tid & 31;
  const int w = tid >> 5;                        // worker: eta-line (X phase) / xi-column (Y phase); M: the helper
  const bool worker = w < M;
  const bool issuer = tid == M * 32;             // lane 0 of the helper
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
  const double xW = g.x0 + i * g.dx;

  // tile t holds row j0-1+t (ring slot t mod NST): wrapped for periodic domains; the neighbour strip's row (-2 south,
  // -3 north) when the domain is one strip of a decomposition along y; absent (-1) outside a non-periodic domain
  auto tile_row = [&](int t) -> int {
    const int jj = j0 - 1 + t;
    if (jj < 0) return A.haloS ? -2 : (g.bc == 0 ? g.ny - 1 : -1);
    if (jj >= g.ny) return A.haloN ? -3 : (g.bc == 0 ? 0 : -1);
    return jj;
  };
  auto tile_src = [&](int jr) -> const double* {
    return (jr >= 0 ? A.qprev + jr * row_stride : (jr == -2 ? A.haloS : A.haloN)) + (size_t)ib * BS;
  };
  auto tile_issue = [&](int t) {                 // issuer only
    const int jr = tile_row(t);
    if (jr != -1) {
      uint64_t* bar = mbar + t % NS;
      mbar_expect_tx(bar, TILE_BYTES);
      bulk_g2s(tiles + (t % NS) * BS, tile_src(jr), TILE_BYTES, bar);
    }
  };
  // k-th copy into a slot completes mbarrier phase k; tile 0 is the only one that can be absent and still be followed
  // by later copies into its slot (non-periodic bottom row)
  const int skip0 = tile_row(0) == -1 ? 1 : 0;
  auto tile_wait = [&](int t) {
    if (tile_row(t) != -1) mbar_wait(mbar + t % NS, (uint32_t)((t / NS - (t % NS == 0 ? skip0 : 0)) & 1));
  };
  auto un_issue = [&](int j) {                   // issuer only; u^n tile of row j -> sN
    mbar_expect_tx(mbar + NS, TILE_BYTES);
    bulk_g2s(sN, A.qn + (size_t)j * row_stride + (size_t)ib * BS, TILE_BYTES, mbar + NS);
  };
  auto prefetch_q0 = [&](int j) {                // issuer only
    const double xl = g.x0 + ib * 32 * g.dx, xr = g.x0 + (ib * 32 + 32) * g.dx;
    const double yl = g.y0 + j * g.dy, yr = g.y0 + (j + 1) * g.dy;
    const double xa = fmax(fabs(xl), fabs(xr)), ya = fmax(fabs(yl), fabs(yr));
    bool want = xa * xa + ya * ya > A.D.r0 * A.D.r0;
    if (A.D.in_r0 > 0.0 && !want) {
      const double xn = (xl <= 0.0 && xr >= 0.0) ? 0.0 : fmin(fabs(xl), fabs(xr));
      const double yn = (yl <= 0.0 && yr >= 0.0) ? 0.0 : fmin(fabs(yl), fabs(yr));
      want = xn * xn + yn * yn < A.D.in_r0 * A.D.in_r0;
    }
    if (want) bulk_prefetch_l2(A.q0 + (size_t)j * row_stride + (size_t)ib * BS, TILE_BYTES);
  };
  auto prefetch_gen = [&](int j) {               // issuer only
    const size_t off = (size_t)j * row_stride + (size_t)ib * BS;
    for (int k = 0; k < A.nk; ++k) bulk_prefetch_l2(A.kin[k] + off, TILE_BYTES);
  };

  // ---- helper: the two faces where the tile meets its x-neighbours (lane = side * M + eta-line) ----
  const int es = lane >= M ? 1 : 0, er = lane - es * M;       // meaningful for lane < 2 M
  const bool edge_lane = !worker && lane < 2 * M;
  const int iLn = ib > 0 ? ib * 32 - 1 : (g.bc == 0 ? g.nx - 1 : -1);
  const int iRn = ib * 32 + 32 < g.nx ? ib * 32 + 32 : (g.bc == 0 ? 0 : -1);
  const int inb = es == 0 ? iLn : iRn;
  const double* nb_src = nullptr;                // line er of the neighbour cell, row 0
  if (edge_lane && inb >= 0) nb_src = A.qprev + (size_t)(inb >> 5) * BS + (inb & 31) + (size_t)(er * M) * 32;
  double nb[4][M];                               // the neighbour's line of the row whose edge faces come next
  auto nb_load = [&](int row) {
#pragma unroll
    for (int v = 0; v < 4; ++v)
#pragma unroll
      for (int q = 0; q < M; ++q)
        nb[v][q] = nb_src ? ldg_here(nb_src + (size_t)row * row_stride + ((v * M) * M + q) * 32) : 0.0;
  };
  // W flux of cell 0 (side 0) / E flux of the last cell (side 1) of line er in row `row`, whose tile is `tile`
  auto edge_faces = [&](int row, const double* tile, double* out) {
    if (!edge_lane) return;
    const int cell = es == 0 ? 0 : last_lane;
    double ext[4], own[4];
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      double se = 0.0, so = 0.0;
#pragma unroll
      for (int q = 0; q < M; ++q) {
        se = fma(es == 0 ? T.Ip[q] : T.Im[q], nb[v][q], se);
        so = fma(es == 0 ? T.Im[q] : T.Ip[q], tile[((v * M + er) * M + q) * 32 + cell], so);
      }
      ext[v] = se;
      own[v] = so;
    }
    if (inb < 0) {                               // domain boundary
      if (g.bc == 1) {
#pragma unroll
        for (int v = 0; v < 4; ++v) ext[v] = own[v];
      } else {
        const double* btr = es == 0 ? A.btrW : A.btrE;
#pragma unroll
        for (int v = 0; v < 4; ++v) ext[v] = __ldg(btr + ((size_t)row * 4 + v) * M + er);
      }
    }
    double cs2 = 0.0, ciso = 0.0;
    if (EOS == 1) {
      const double yc = g.y0 + (row + 0.5) * g.dy;
      const double yr = yc + g.hdy * T.xi[er];
      const double y2e = fma(yr, yr, A.ph.eps2s);
      const int iface = ib * 32 + (es == 0 ? 0 : last_lane + 1);
      const double xf = g.x0 + iface * g.dx;
      cs2 = A.ph.h2gm * rsqrt_fast(fma(xf, xf, y2e));
      ciso = sqrt_fast(cs2);
    }
    double Fe[4], Fo[4];
    Wave<FLUX> we, wo;
    face_flux<EOS, 0, FLUX>(A.ph, ext, cs2, ciso, Fe, we);
    face_flux<EOS, 0, FLUX>(A.ph, own, cs2, ciso, Fo, wo);
    double UL[4], FL[4], UR[4], FR[4];
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      UL[v] = es == 0 ? ext[v] : own[v]; FL[v] = es == 0 ? Fe[v] : Fo[v];
      UR[v] = es == 0 ? own[v] : ext[v]; FR[v] = es == 0 ? Fo[v] : Fe[v];
    }
    const Wave<FLUX> wL = es == 0 ? we : wo, wR = es == 0 ? wo : we;
    double H[4];
    riemann2<FLUX, EOS, 0>(UL, FL, wL, UR, FR, wR, H);
#pragma unroll
    for (int v = 0; v < 4; ++v) out[(er * 2 + es) * 4 + v] = H[v];
  };

  if (issuer) {
#pragma unroll
    for (int s = 0; s <= NS; ++s) mbar_init(mbar + s, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  double spmax = 0.0;                            // running CFL wave-speed maximum of this lane (helper)
  if (!worker) {
    if (issuer) {
      tile_issue(0);
      tile_issue(1);
      tile_issue(2);
      if (use_un) un_issue(j0);
      if (use_un && j0 + 1 < j1) bulk_prefetch_l2(A.qn + (size_t)(j0 + 1) * row_stride + (size_t)ib * BS, TILE_BYTES);
      if (do_damp) prefetch_q0(j0);
      if (gen && A.gen_pf) prefetch_gen(j0);
    }
    nb_load(j0);
    tile_wait(0);
    tile_wait(1);
    edge_faces(j0, tiles + BS, sHX);
    if (j0 + 1 < j1) nb_load(j0 + 1);            // consumed in the first row's iteration
  }
  // S face of the segment's first row: every worker its own column, straight into its registers, while the helper
  // does the tile-edge faces.  (The helper used to evaluate all M columns one after the other with the workers waiting
  // at the barrier below: 6 % of all warp stall samples of the first stage sat on that barrier, about one row's time
  // per 16-row segment.)  The workers wait for the two tiles on the tiles' own mbarriers -- here and nowhere else.
  double HS[4] = {0, 0, 0, 0};                   // numerical flux (x2) through the row's S face, column q = w
  if (worker) {
    tile_wait(0);
    tile_wait(1);
    const double* lo = tile_row(0) != -1 ? tiles + lane : nullptr;
    const double* hi = tiles + BS + lane;
    const double* btr = A.btrS + (size_t)(ib * 4) * M * 32 + lane;
    y_face<M, EOS, FLUX>(A, lo, hi, btr, w, xc + g.hdx * T.xi[w], g.y0 + j0 * g.dy, HS);
  }
  __syncthreads();                               // sHX of the first row is written; tile 0's slot may be overwritten

  // N face of column qn of the row whose tile is tlo: the row's trace UNq at eta = +1 against the S trace of the row
  // above (tile tlo + 1) or the boundary condition
  auto n_face = [&](int tlo, int jrow, int qn, const double (&UNq)[4], double (&HNq)[4]) {
    const double xqn = xc + g.hdx * T.xi[qn];
    const double yN = g.y0 + (jrow + 1) * g.dy;
    double cs2N = 0.0, cN = 0.0;
    if (EOS == 1) {
      cs2N = A.ph.h2gm * rsqrt_fast(fma(xqn, xqn, fma(yN, yN, A.ph.eps2s)));
      cN = sqrt_fast(cs2N);
    }
    double GNo[4];
    Wave<FLUX> lamNo;
    face_flux<EOS, 1, FLUX>(A.ph, UNq, cs2N, cN, GNo, lamNo);
    double aU[4], aG[4];
    Wave<FLUX> aLam;
    if (tile_row(tlo + 1) != -1) {
      column_trace<M>(tiles + ((tlo + 1) % NS) * BS + lane, 32, qn, T.Im, aU);
      face_flux<EOS, 1, FLUX>(A.ph, aU, cs2N, cN, aG, aLam);
    } else if (g.bc == 1) {
#pragma unroll
      for (int v = 0; v < 4; ++v) { aU[v] = UNq[v]; aG[v] = GNo[v]; }
      aLam = lamNo;
    } else {
#pragma unroll
      for (int v = 0; v < 4; ++v) aU[v] = __ldg(A.btrN + ((size_t)(ib * 4 + v) * M + qn) * 32 + lane);
      face_flux<EOS, 1, FLUX>(A.ph, aU, cs2N, cN, aG, aLam);
    }
    riemann2<FLUX, EOS, 1>(UNq, GNo, lamNo, aU, aG, aLam, HNq);
  };
  // Balance between the warps (M = 5).  A block's warps 0..5 sit on schedulers (s, s+1, s+2, s+3, s, s+1) (%warpid mod 4
  // over the 2048 blocks of a launch; s uniform in 0..3, so how the two blocks of an SM overlap varies): workers 0 and
  // 4 always share a scheduler.  Workers 1 and 3 therefore also do the N face of columns 0 and M - 1 (first thing in
  // their Y phase, through sHS) and workers 0 and M - 1 skip theirs.  Found by measurement, with per-warp clock traces
  // of the row phases: before, workers 0 / 4 / 2 were last at the end-of-row barrier; other assignments (workers 2 and
  // 3 as takers; worker 1 taking column 2 as well) were slower.  Correct under any slot layout.
  // Measured at 1024^2: first / middle stage 0.450 / 0.490 ms instead of 0.464 / 0.494; in the stages whose helper also
  // carries the CFL reduction: last stage 0.582 instead of 0.566, so not there.
  constexpr bool REBAL = M == 5 && !do_cfl;
  const bool donor = REBAL && (w == 0 || w == M - 1);
  const bool taker = REBAL && (w == 1 || w == M - 2);
  const int pair = w <= 1 ? 0 : 1;               // donor 0 <-> taker 1 (barrier 8), donor M-1 <-> taker M-2 (barrier 9)

  // Two loops over the rows, one per role, meeting at the same named barriers: what each role carries from row to
  // row (the workers' S-face flux, the helper's neighbour lines) costs registers in its own loop only.
  if (worker) {
    for (int j = j0; j < j1; ++j) {
      const int t = j - j0 + 1;                  // tile index of row j
      const double* tu = tiles + (t % NS) * BS + lane;
      const double yc = g.y0 + (j + 0.5) * g.dy;
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
        // own W/E face states, fluxes, speeds; c_s at the E face is the right neighbour's W value (the last
        // lane's E face belongs to the helper, so what lane 31 gets here does not matter)
        double cs2W = 0.0, cW = 0.0, cs2E = 0.0, cE = 0.0;
        if (EOS == 1) {
          cs2W = A.ph.h2gm * rsqrt_fast(fma(xW, xW, y2e));
          cW = sqrt_fast(cs2W);
          cs2E = shfl_dn1(cs2W);
          cE = shfl_dn1(cW);
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
        double HE[4], HW[4];
        riemann2<FLUX, EOS, 0>(UE, FEo, lamEo, UR, FR, lamR, HE);
#pragma unroll
        for (int v = 0; v < 4; ++v) HW[v] = shfl_up1(HE[v]);
        // the tile's two outer faces come from the helper
        const double* hx = sHX + ((j - j0) & 1) * (M * 8) + r * 8;
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          const double hw = hx[v], he = hx[4 + v];
          HW[v] = lane == 0 ? hw : HW[v];
          HE[v] = lane == last_lane ? he : HE[v];
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
      bar_sync_named(2, NWORK);

      // =========================== Y phase: xi-column q = w ===========================
      if (taker) {                               // the N face of a three-to-a-scheduler worker's column, for it
        const int qx = pair == 0 ? 0 : M - 1;
        bar_sync_named(3 + w, 64);               // the tile of the row above has landed
        double UNx[4], HNx[4];
        column_trace<M>(tu, 32, qx, T.Ip, UNx);
        n_face(t, j, qx, UNx, HNx);
#pragma unroll
        for (int v = 0; v < 4; ++v) sHS[(v * M + qx) * 32 + lane] = HNx[v];
        __threadfence_block();
        bar_arrive_named(8 + pair, 64);
      }
      {
        const int q = w;
        const double xq = xc + g.hdx * T.xi[q];
        double acc[4][M];
#pragma unroll
        for (int v = 0; v < 4; ++v)
#pragma unroll
          for (int r = 0; r < M; ++r) acc[v][r] = 0.0;
        // wave-killing factors of this cell (row a12): out <- f0 u0 + ft out
        double f0 = 0.0, ft = 1.0;                 // (from the helper, once the N face is done)
        bool damp = false;
        constexpr bool early_q0 = false;
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
          if (!donor) {
#pragma unroll
            for (int v = 0; v < 4; ++v) UN[v] = fma(T.Ip[r], u[v], UN[v]);
          }
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
        // north face: own trace against the S trace of the row above (tile t+1: the helper arrives at barrier 3 + w
        // once it has seen that tile land), or -- workers 0 and M-1 at M = 5 -- what workers 1 and M-2 have put into sHS
        double HN[4];
        if (donor) {
          bar_sync_named(8 + pair, 64);
#pragma unroll
          for (int v = 0; v < 4; ++v) HN[v] = sHS[(v * M + q) * 32 + lane];
        } else {
          if (!taker) bar_sync_named(3 + w, 64);
          n_face(t, j, q, UN, HN);
        }
        if (do_damp) {                           // the cell's wave-killing factors: one evaluation per row, by the helper
          f0 = sHS[lane];
          ft = sHS[32 + lane];
          damp = f0 != 0.0;
        }

        // modal update in nodal form + RK combination (rows a8, a9) and store
        const size_t cell_off = j * row_stride + (size_t)ib * BS + lane;
        double* __restrict__ qo = A.qout + cell_off;
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          double avg = 0.0;
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
          // partial cell average of this column: into the column's own (v, 0, q) entry of sN, read above and dead
          // until the next row's u^n lands there
          if (do_cfl) sN[((v * M) * M + q) * 32 + lane] = 0.25 * T.w[q] * avg;
        }
#pragma unroll
        for (int v = 0; v < 4; ++v) HS[v] = HN[v];   // this row's N face is the next row's S face
      }
      bar_sync_named(0, NTHR);
    }
  } else {
    // =========================== helper warp ===========================
    for (int j = j0; j < j1; ++j) {
      const int t = j - j0 + 1;                  // tile index of row j
      const bool more = j + 1 < j1;
      // fused CFL wave speed of the row finished in the previous iteration (row a10): its partial
      // averages sit in sN and must be out before the next u^n tile is sent there
      double avg[4] = {1.0, 0.0, 0.0, 1.0};
      if (do_cfl && j > j0) {
#pragma unroll
        for (int v = 0; v < 4; ++v) {
          double s = 0.0;
#pragma unroll
          for (int qq = 0; qq < M; ++qq) s += sN[((v * M) * M + qq) * 32 + lane];
          avg[v] = s;
        }
      }
      __syncwarp();
      if (issuer) {
        fence_proxy_async();                     // the slots about to be refilled were read through the generic proxy
        if (more) tile_issue(t + 2);             // row j+2 -> the slot row j-1 has just left
        if (use_un && j > j0) un_issue(j);       // sN is free again
        if (use_un && more) bulk_prefetch_l2(A.qn + (size_t)(j + 1) * row_stride + (size_t)ib * BS, TILE_BYTES);   // so that the next row's copy comes from L2
        if (do_damp && more) prefetch_q0(j + 1);
        if (gen && A.gen_pf == 2 && more) prefetch_gen(j + 1);
        if (gen && A.gen_pf == 1 && j > j0) prefetch_gen(j);
      }
      if (do_cfl && j > j0) {
        double sp = 0.0;
        if (valid) {
          const double ycp = g.y0 + (j - 0.5) * g.dy;
          const double rinv = rcp_fast(avg[0]);
          const double vx = avg[1] * rinv, vy = avg[2] * rinv;
          double c;
          if (EOS == 0) c = sqrt_fast(A.ph.gamma * A.ph.gm1 * (avg[3] - 0.5 * (avg[1] * vx + avg[2] * vy)) * rinv);
          else          c = sqrt_fast(A.ph.h2gm * rsqrt_fast(fma(xc, xc, fma(ycp, ycp, A.ph.eps2s))));
          sp = (fabs(vx) + c) * g.inv_dx + (fabs(vy) + c) * g.inv_dy;
          if (!(sp >= 0.0)) sp = __longlong_as_double(0x7ff0000000000000LL);   // NaN -> +inf
        }
        spmax = fmax(spmax, sp);                 // per lane; reduced once after the last row
      }
      // wave-killing factors of the row's cells (row a12): out <- f0 u0 + ft out.  One evaluation per cell
      // here instead of one per column warp; the workers read them after they have synchronised on barrier 3 + w
      // (sHS is free in these stages: the N-face hand-over runs only in stages without the CFL reduction)
      if (do_damp) {
        double f0 = 0.0, ft = 1.0;
        const double ycj = g.y0 + (j + 0.5) * g.dy;
        if (KIND != K_GENL || A.D.on) {
          if (!damp_factors(A.D, sqrt_fast(fma(xc, xc, ycj * ycj) + 1e-300), f0, ft)) { f0 = 0.0; ft = 1.0; }   // + tiny: a centre at the origin
        }
        sHS[lane] = f0;
        sHS[32 + lane] = ft;
        __threadfence_block();
      }
      tile_wait(t + 1);                          // sent a whole row ago; the workers' N faces and the next row read it
#pragma unroll
      for (int k = 0; k < M; ++k)
        if (!(REBAL && (k == 0 || k == M - 1))) bar_arrive_named(3 + k, 64);   // (those two take their N face from a neighbour)
      if (gen && A.gen_pf == 3 && issuer) prefetch_gen(j);
      // next row's outer x-faces (the neighbours' lines were requested a row ago), then the request for the row after
      if (more) edge_faces(j + 1, tiles + ((t + 1) % NS) * BS, sHX + ((j + 1 - j0) & 1) * (M * 8));
      if (j + 2 < j1) nb_load(j + 2);
      __threadfence_block();
      bar_sync_named(0, NTHR);
    }
  }
  // CFL wave speed of the last row of the segment, then one reduction per thread block
  if (do_cfl && !worker) {
    double avg[4];
#pragma unroll
    for (int v = 0; v < 4; ++v) {
      double s = 0.0;
#pragma unroll
      for (int qq = 0; qq < M; ++qq) s += sN[((v * M) * M + qq) * 32 + lane];
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
    unsigned long long bits = (unsigned long long)__double_as_longlong(fmax(spmax, sp));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const unsigned long long other = __shfl_xor_sync(FULL, bits, o);
      bits = other > bits ? other : bits;
    }
    if (lane == 0) atomicMax(A.wmax, bits);
  }
}

}  // namespace dg
