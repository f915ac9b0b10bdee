/* CPU ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT.  See ref_dg.h.
 *
 * Follows SURVEY.md section 8(c) step by step (readings G1..G20 are listed in DESIGN.md):
 *   C1  tables          PAPER.md:65, 95-97, 155       Gauss-Legendre nodes/weights, phi_a = sqrt(2a+1) P_a
 *   C2  nodal values    PAPER.md:73-75                u_h = sum_ab U_ab phi_a(xi) phi_b(eta)
 *   C3  Euler fluxes    PAPER.md:36-43  Eq.(1)
 *   C4  EOS             PAPER.md:45-49  Eq.(2); locally isothermal closure from BASELINE.json
 *   C5  numerical flux  PAPER.md:97  (type unnamed; BASELINE cfg0: local Lax-Friedrichs)
 *   C5b HLLC / HLL flux option (PAPER.md:97 leaves the flux unnamed)
 *   C6  gravity source
 *   C7  RHS             PAPER.md:85-97  Eq.(3), divided by the (diagonal) mass
 *   C8  SSP-RK          PAPER.md:105-111 (Gottlieb & Shu 1998, Shu-Osher form)
 *   C9  boundaries
 *   C10 CFL
 *   C11 wave damping
 *   C8b Butcher-form RK PAPER.md:445-457 (Appendix A), Table 1, Table 2
 *   C12 positivity limiter  PAPER.md:129-131, 150 (Zhang & Shu 2010; readings L1..L5 in DESIGN.md)
 *   C13 torque on the planet  PAPER.md:321-328  Eq.(6); C13b its normalisation gamma Gamma/Gamma_0
 *
 * No blocking, fusion, sum-factorisation or reordering: every sum is written as the nested loop
 * the formula states, in fp64, compiled with -O2 -ffp-contract=off.
 *
 * Pins (tests/test_oracle_tables.py, test_oracle_pointwise.py, test_oracle_rhs.py,
 * test_oracle_time.py; none of them re-types these formulas):
 *   C1  sum w = 2; exactness on x^k, k <= 2m-1; closed forms m = 1,2,3; orthonormality; numpy leggauss
 *   C3-C5  consistency H(U,U) = f(U).n; bitwise antisymmetry; Rankine-Hugoniot-free upwind limit
 *   C6  centred finite difference of the potential; planet period 2 pi / Omega_p
 *   C2+C7 volume term: 24-point brute-force quadrature of int_K f(u_h).grad(phi) (exact integrands)
 *   C7  free-stream L(const) = 0; conservation on periodic domains; face term by 24-point quadrature
 *   C6+C7  Keplerian equilibrium residual -> 0 at rate h^(p+1)
 *   C8  y' = lambda y observed order 2 / 3; exact on polynomials of degree <= order
 *   C7+C8  isentropic-vortex L1 error slope ~ p+1
 *   C10 hand value on a constant state;  C11 R = 0 identity, fixed point, tau -> 0 limit; damp_mode 1: node-wise
 *       relation of the primitive fields through NumPy's basis evaluation, a hand-worked constant cell
 *   C9  frozen boundary: = transmissive before the state moves; NumPy traces of U / U0 afterwards
 *   C4  eos 1 on faces: m-point quadrature of the point-wise flux with c_s at the face nodes
 *   C8b the tableaus against the paper's printed digits (tests/golden/rk_tableaus.txt), row sums = c,
 *       order conditions, observed order 4 / 5 on y' = lambda y and on a non-autonomous ODE
 *   C12 Gauss-Lobatto closed forms and exactness; the cell average as a convex combination of the
 *       limiter's point values; averages kept bitwise; admissibility after limiting; identity on
 *       admissible cells; hand-worked theta on a linear cell; p = eps at the binding point
 *   C13 torque of a single massive cell by hand; zero for an axisymmetric ring; antisymmetry
 *   absolute per-step values: PARITY UNPINNED (paper prints none).
 */
#include "ref_dg.h"

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

const int MAXM = 5;
const int NV = 4;                         /* rho, rho vx, rho vy, E */

struct Tables {
  int m;
  double xi[MAXM], w[MAXM];
  double B[MAXM][MAXM];                   /* B[q][a] = phi_a(xi_q)   */
  double D[MAXM][MAXM];                   /* D[q][a] = phi_a'(xi_q)  */
  double Ep[MAXM], Em[MAXM];              /* phi_a(+1), phi_a(-1)    */
};

/* Legendre P_n(x) and P_n'(x) by the three-term recurrence. */
void legendre(int n, double x, double* P, double* dP) {
  double p0 = 1.0, p1 = x, d0 = 0.0, d1 = 1.0;
  if (n == 0) { *P = p0; *dP = d0; return; }
  for (int k = 2; k <= n; ++k) {
    double pk = ((2.0 * k - 1.0) * x * p1 - (k - 1.0) * p0) / k;
    double dk = d0 + (2.0 * k - 1.0) * p1;          /* P_k' = P_{k-2}' + (2k-1) P_{k-1} */
    p0 = p1; p1 = pk; d0 = d1; d1 = dk;
  }
  *P = p1; *dP = d1;
}

/* C1 */
void build_tables(int m, Tables* T) {
  T->m = m;
  const double pi = 3.14159265358979323846;
  for (int q = 0; q < m; ++q) {
    /* Newton iteration on P_m from the Chebyshev guess; nodes in ascending order */
    double x = -std::cos(pi * (q + 0.75) / (m + 0.5));
    for (int it = 0; it < 100; ++it) {
      double P, dP;
      legendre(m, x, &P, &dP);
      double dx = P / dP;
      x -= dx;
      if (std::fabs(dx) < 1e-16) break;
    }
    double P, dP;
    legendre(m, x, &P, &dP);
    T->xi[q] = x;
    T->w[q] = 2.0 / ((1.0 - x * x) * dP * dP);
  }
  if (m % 2 == 1) T->xi[m / 2] = 0.0;
  for (int q = 0; q < m; ++q)
    for (int a = 0; a < m; ++a) {
      double P, dP;
      legendre(a, T->xi[q], &P, &dP);
      double s = std::sqrt(2.0 * a + 1.0);
      T->B[q][a] = s * P;
      T->D[q][a] = s * dP;
    }
  for (int a = 0; a < m; ++a) {
    double s = std::sqrt(2.0 * a + 1.0);
    T->Ep[a] = s;
    T->Em[a] = (a % 2 == 0) ? s : -s;
  }
}

/* C4: sound speed squared of the locally isothermal closure at (x,y). */
inline double cs2_iso(const ref_params& p, double x, double y) {
  return p.h_aspect * p.h_aspect * p.gm_star / std::sqrt(x * x + y * y + p.eps_star * p.eps_star);
}

/* C3 + C4: flux in direction dir of the state U at the point (x,y); also v_n and c. */
void point_flux(const ref_params& p, const double* U, double x, double y, int dir,
                double* F, double* vn, double* c) {
  const double rho = U[0], mx = U[1], my = U[2], E = U[3];
  const double vx = mx / rho, vy = my / rho;
  double pr, cc;
  if (p.eos == 0) {
    pr = (p.gamma - 1.0) * (E - 0.5 * (mx * mx + my * my) / rho);
    cc = std::sqrt(p.gamma * pr / rho);
  } else {
    const double cs2 = cs2_iso(p, x, y);
    pr = cs2 * rho;
    cc = std::sqrt(cs2);
  }
  if (dir == 0) {
    F[0] = mx; F[1] = mx * vx + pr; F[2] = my * vx; F[3] = (E + pr) * vx; *vn = vx;
  } else {
    F[0] = my; F[1] = mx * vy; F[2] = my * vy + pr; F[3] = (E + pr) * vy; *vn = vy;
  }
  *c = cc;
}

/* C5 */
void llf(const ref_params& p, const double* UL, const double* UR, double x, double y, int dir,
         double* H) {
  double FL[NV], FR[NV], vL, vR, cL, cR;
  point_flux(p, UL, x, y, dir, FL, &vL, &cL);
  point_flux(p, UR, x, y, dir, FR, &vR, &cR);
  const double lam = std::fmax(std::fabs(vL) + cL, std::fabs(vR) + cR);
  for (int v = 0; v < NV; ++v) H[v] = 0.5 * (FL[v] + FR[v]) - 0.5 * lam * (UR[v] - UL[v]);
}

/* C5b: HLL-type fluxes with the wave-speed estimates of Davis (1988),
 *   S_L = min(v_L - c_L, v_R - c_R),  S_R = max(v_L + c_L, v_R + c_R).
 * eos 1 (isothermal, no contact wave):  HLL  H = (S_R F_L - S_L F_R + S_L S_R (U_R - U_L))/(S_R - S_L) for
 * S_L < 0 < S_R, else the upwind flux.  eos 0: HLLC (Toro, Spruce & Speares 1994) with the contact speed
 *   S* = (p_R - p_L + rho_L v_L (S_L - v_L) - rho_R v_R (S_R - v_R)) / (rho_L (S_L - v_L) - rho_R (S_R - v_R))
 * and the star states U*_K = rho_K (S_K - v_K)/(S_K - S*) (1, S* | v_t, E_K/rho_K + (S* - v_K)(S* + p_K/(rho_K (S_K - v_K)))),
 * H = F_L | F_L + S_L (U*_L - U_L) | F_R + S_R (U*_R - U_R) | F_R  for  0 <= S_L | S_L <= 0 <= S* | S* <= 0 <= S_R | S_R <= 0. */
void hllc(const ref_params& p, const double* UL, const double* UR, double x, double y, int dir, double* H) {
  double FL[NV], FR[NV], vL, vR, cL, cR;
  point_flux(p, UL, x, y, dir, FL, &vL, &cL);
  point_flux(p, UR, x, y, dir, FR, &vR, &cR);
  const double SL = std::fmin(vL - cL, vR - cR), SR = std::fmax(vL + cL, vR + cR);
  if (SL >= 0.0) { for (int v = 0; v < NV; ++v) H[v] = FL[v]; return; }
  if (SR <= 0.0) { for (int v = 0; v < NV; ++v) H[v] = FR[v]; return; }
  if (p.eos == 1) {
    for (int v = 0; v < NV; ++v) H[v] = (SR * FL[v] - SL * FR[v] + SL * SR * (UR[v] - UL[v])) / (SR - SL);
    return;
  }
  const int n = 1 + dir, tg = 2 - dir;               /* normal and tangential momentum components */
  const double pL = (p.gamma - 1.0) * (UL[3] - 0.5 * (UL[1] * UL[1] + UL[2] * UL[2]) / UL[0]);
  const double pR = (p.gamma - 1.0) * (UR[3] - 0.5 * (UR[1] * UR[1] + UR[2] * UR[2]) / UR[0]);
  const double mL = UL[0] * (SL - vL), mR = UR[0] * (SR - vR);
  const double Ss = (pR - pL + UL[n] * (SL - vL) - UR[n] * (SR - vR)) / (mL - mR);
  const double* U = Ss >= 0.0 ? UL : UR;
  const double* F = Ss >= 0.0 ? FL : FR;
  const double S = Ss >= 0.0 ? SL : SR, vK = Ss >= 0.0 ? vL : vR, pK = Ss >= 0.0 ? pL : pR;
  const double fac = U[0] * (S - vK) / (S - Ss);
  double Us[NV];
  Us[0] = fac;
  Us[n] = fac * Ss;
  Us[tg] = fac * (U[tg] / U[0]);
  Us[3] = fac * (U[3] / U[0] + (Ss - vK) * (Ss + pK / (U[0] * (S - vK))));
  for (int v = 0; v < NV; ++v) H[v] = F[v] + S * (Us[v] - U[v]);
}

/* the numerical flux selected by params.flux */
inline void num_flux(const ref_params& p, const double* UL, const double* UR, double x, double y, int dir, double* H) {
  if (p.flux == 1) hllc(p, UL, UR, x, y, dir, H);
  else llf(p, UL, UR, x, y, dir, H);
}

/* C6 */
void gravity(const ref_params& p, double t, double x, double y, double* g) {
  g[0] = 0.0; g[1] = 0.0;
  if (p.gm_star == 0.0) return;
  {
    const double r2 = x * x + y * y + p.eps_star * p.eps_star;
    const double r3 = r2 * std::sqrt(r2);
    g[0] -= p.gm_star * x / r3;
    g[1] -= p.gm_star * y / r3;
  }
  if (p.q_planet != 0.0) {
    const double ang = p.omega_planet * t + p.phase0;
    const double xp = p.r_planet * std::cos(ang), yp = p.r_planet * std::sin(ang);
    const double dx = x - xp, dy = y - yp;
    const double r2 = dx * dx + dy * dy + p.eps_planet * p.eps_planet;
    const double r3 = r2 * std::sqrt(r2);
    g[0] -= p.q_planet * p.gm_star * dx / r3;
    g[1] -= p.q_planet * p.gm_star * dy / r3;
  }
}

/* C12 tables (see build_lobatto) */
struct LimTables {
  int nh;
  double xh[4], wh[4];                    /* Lobatto nodes on [-1,1]; weights normalised to sum 1 */
  double Bh[4][MAXM];                     /* phi_a(xh_k) */
};

}  // namespace

struct ref_ctx {
  ref_params p;
  Tables T;
  LimTables LT;
  int m;
  long ncoef;                 /* ny*nx*4*m*m */
  double dx, dy, t;
  bool has_state;
  std::vector<double> U, U0;
};

namespace {

inline long cell_off(const ref_ctx* c, int i, int j) { return ((long)j * c->p.nx + i) * NV * c->m * c->m; }

/* trace of the polynomial of cell (i,j) in array A at xi = side (x-faces, function of eta_r)
 * or eta = side (y-faces, function of xi_q):  U(+-1, eta_r) = sum_b sum_a A_ab E[a] B[r][b]. */
void trace_x(const ref_ctx* c, const double* A, int i, int j, int side, int r, double* out) {
  const int m = c->m;
  const double* E = side > 0 ? c->T.Ep : c->T.Em;
  const double* a0 = A + cell_off(c, i, j);
  for (int v = 0; v < NV; ++v) {
    double s = 0.0;
    for (int b = 0; b < m; ++b)
      for (int a = 0; a < m; ++a) s += a0[(v * m + b) * m + a] * E[a] * c->T.B[r][b];
    out[v] = s;
  }
}
void trace_y(const ref_ctx* c, const double* A, int i, int j, int side, int q, double* out) {
  const int m = c->m;
  const double* E = side > 0 ? c->T.Ep : c->T.Em;
  const double* a0 = A + cell_off(c, i, j);
  for (int v = 0; v < NV; ++v) {
    double s = 0.0;
    for (int b = 0; b < m; ++b)
      for (int a = 0; a < m; ++a) s += a0[(v * m + b) * m + a] * c->T.B[q][a] * E[b];
    out[v] = s;
  }
}

/* C7 (with C2, C3, C5, C6, C9).  parts: 1 volume flux, 2 faces, 4 source. */
void compute_rhs(const ref_ctx* c, const double* U, double t, int parts, double* L) {
  const ref_params& p = c->p;
  const Tables& T = c->T;
  const int m = c->m, nx = p.nx, ny = p.ny;
  const double dx = c->dx, dy = c->dy;

  /* numerical fluxes on all x-faces [j][f][r][v], f = 0..nx, and y-faces [f][i][q][v], f = 0..ny */
  std::vector<double> HX((size_t)ny * (nx + 1) * m * NV, 0.0), HY((size_t)(ny + 1) * nx * m * NV, 0.0);
  if (parts & 2) {
#pragma omp parallel for schedule(static)
    for (int j = 0; j < ny; ++j)
      for (int f = 0; f <= nx; ++f)
        for (int r = 0; r < m; ++r) {
          double UL[NV], UR[NV];
          const double xf = p.x0 + f * dx;
          const double yr = p.y0 + (j + 0.5) * dy + 0.5 * dy * T.xi[r];
          if (f > 0 && f < nx) {
            trace_x(c, U, f - 1, j, +1, r, UL);
            trace_x(c, U, f, j, -1, r, UR);
          } else if (p.bc == 0) {                       /* C9 periodic: wrap */
            trace_x(c, U, nx - 1, j, +1, r, UL);
            trace_x(c, U, 0, j, -1, r, UR);
          } else if (f == 0) {
            trace_x(c, U, 0, j, -1, r, UR);
            if (p.bc == 1) std::memcpy(UL, UR, sizeof UL);           /* transmissive */
            else trace_x(c, c->U0.data(), 0, j, -1, r, UL);            /* frozen to initial */
          } else {
            trace_x(c, U, nx - 1, j, +1, r, UL);
            if (p.bc == 1) std::memcpy(UR, UL, sizeof UR);
            else trace_x(c, c->U0.data(), nx - 1, j, +1, r, UR);
          }
          num_flux(p, UL, UR, xf, yr, 0, &HX[(((size_t)j * (nx + 1) + f) * m + r) * NV]);
        }
#pragma omp parallel for schedule(static)
    for (int f = 0; f <= ny; ++f)
      for (int i = 0; i < nx; ++i)
        for (int q = 0; q < m; ++q) {
          double UL[NV], UR[NV];
          const double yf = p.y0 + f * dy;
          const double xq = p.x0 + (i + 0.5) * dx + 0.5 * dx * T.xi[q];
          if (f > 0 && f < ny) {
            trace_y(c, U, i, f - 1, +1, q, UL);
            trace_y(c, U, i, f, -1, q, UR);
          } else if (p.bc == 0) {
            trace_y(c, U, i, ny - 1, +1, q, UL);
            trace_y(c, U, i, 0, -1, q, UR);
          } else if (f == 0) {
            trace_y(c, U, i, 0, -1, q, UR);
            if (p.bc == 1) std::memcpy(UL, UR, sizeof UL);
            else trace_y(c, c->U0.data(), i, 0, -1, q, UL);
          } else {
            trace_y(c, U, i, ny - 1, +1, q, UL);
            if (p.bc == 1) std::memcpy(UR, UL, sizeof UR);
            else trace_y(c, c->U0.data(), i, ny - 1, +1, q, UR);
          }
          num_flux(p, UL, UR, xq, yf, 1, &HY[(((size_t)f * nx + i) * m + q) * NV]);
        }
  }

#pragma omp parallel for schedule(static)
  for (int j = 0; j < ny; ++j)
    for (int i = 0; i < nx; ++i) {
      const double* u = U + cell_off(c, i, j);
      double* Lc = L + cell_off(c, i, j);
      const double xc = p.x0 + (i + 0.5) * dx, yc = p.y0 + (j + 0.5) * dy;
      /* C2: nodal values at the m x m Gauss-Legendre points; C3: F, G; C6: S */
      double Fq[MAXM][MAXM][NV], Gq[MAXM][MAXM][NV], Sq[MAXM][MAXM][NV];
      for (int r = 0; r < m; ++r)
        for (int q = 0; q < m; ++q) {
          double Un[NV];
          for (int v = 0; v < NV; ++v) {
            double s = 0.0;
            for (int b = 0; b < m; ++b)
              for (int a = 0; a < m; ++a) s += u[(v * m + b) * m + a] * T.B[q][a] * T.B[r][b];
            Un[v] = s;
          }
          const double x = xc + 0.5 * dx * T.xi[q], y = yc + 0.5 * dy * T.xi[r];
          double vn, cc;
          point_flux(p, Un, x, y, 0, Fq[q][r], &vn, &cc);
          point_flux(p, Un, x, y, 1, Gq[q][r], &vn, &cc);
          double g[2];
          gravity(p, t, x, y, g);
          Sq[q][r][0] = 0.0;
          Sq[q][r][1] = Un[0] * g[0];
          Sq[q][r][2] = Un[0] * g[1];
          Sq[q][r][3] = Un[1] * g[0] + Un[2] * g[1];
        }
      for (int v = 0; v < NV; ++v)
        for (int b = 0; b < m; ++b)
          for (int a = 0; a < m; ++a) {
            double vol = 0.0, src = 0.0, fx = 0.0, fy = 0.0;
            for (int q = 0; q < m; ++q)
              for (int r = 0; r < m; ++r) {
                const double ww = T.w[q] * T.w[r];
                vol += ww * ((2.0 / dx) * Fq[q][r][v] * T.D[q][a] * T.B[r][b] +
                             (2.0 / dy) * Gq[q][r][v] * T.B[q][a] * T.D[r][b]);
                src += ww * Sq[q][r][v] * T.B[q][a] * T.B[r][b];
              }
            if (parts & 2) {
              for (int r = 0; r < m; ++r) {
                const double hE = HX[(((size_t)j * (nx + 1) + i + 1) * m + r) * NV + v];
                const double hW = HX[(((size_t)j * (nx + 1) + i) * m + r) * NV + v];
                fx += T.w[r] * (hE * T.Ep[a] - hW * T.Em[a]) * T.B[r][b];
              }
              for (int q = 0; q < m; ++q) {
                const double hN = HY[(((size_t)(j + 1) * nx + i) * m + q) * NV + v];
                const double hS = HY[(((size_t)j * nx + i) * m + q) * NV + v];
                fy += T.w[q] * (hN * T.Ep[b] - hS * T.Em[b]) * T.B[q][a];
              }
            }
            double acc = 0.0;
            if (parts & 1) acc += 0.25 * vol;
            if (parts & 4) acc += 0.25 * src;
            if (parts & 2) acc += -fx / (2.0 * dx) - fy / (2.0 * dy);
            Lc[(v * m + b) * m + a] = acc;
          }
    }
}

struct RhsClosure { const ref_ctx* c; };
void dg_ode(void* user, double t, const double* y, double* dydt) {
  compute_rhs(static_cast<RhsClosure*>(user)->c, y, t, 7, dydt);
}

/* C11: Q <- (dt Q0 + tau Q)/(tau + dt), tau = 2 pi sqrt(r_d^3/GM)/R(r), R(r) = ((r - r_d)/(r_b - r_d))^2
 * clamped to 1 beyond the boundary radius r_b.  Outer zone: r_d = damp_r0 < r,
 * r_b = damp_r1; inner zone (the paper's own disc): r_d = damp_in_r0 > r, r_b = damp_in_r1.  r = the cell centre.
 * damp_mode 0 (reading G13): Q runs over the conservative modal coefficients.
 * damp_mode 1 ("The dampened fields are the density, velocities and temperature"; reading D2):
 * at each of the cell's m x m Gauss points (C2) Q runs over rho, v_x = m_x/rho, v_y = m_y/rho and T = p/rho
 * (p from Eq.(2), of the carried energy for either closure), Q0 over the same fields of the initial
 * state; the conservative state (rho, rho v, rho T/(gamma-1) + rho v^2/2) rebuilt from the relaxed fields is
 * projected back onto the modes with the m-point rule, which is exact here. */
void damp_cell_primitive(const ref_ctx* c, double f0, double ft, double* u, const double* u0) {
  const int mo = c->m;                               /* order (m[] below are a node's conservative values) */
  const Tables& T = c->T;
  const double gm1 = c->p.gamma - 1.0;
  double nod[MAXM][MAXM][NV];
  for (int r = 0; r < mo; ++r)
    for (int q = 0; q < mo; ++q) {
      double m[NV], m0[NV];                          /* C2: nodal values of U and of the initial state U0 */
      for (int v = 0; v < NV; ++v) {
        double s = 0.0, s0 = 0.0;
        for (int b = 0; b < mo; ++b)
          for (int a = 0; a < mo; ++a) {
            s += u[(v * mo + b) * mo + a] * T.B[q][a] * T.B[r][b];
            s0 += u0[(v * mo + b) * mo + a] * T.B[q][a] * T.B[r][b];
          }
        m[v] = s; m0[v] = s0;
      }
      const double r0 = m0[0], v0x = m0[1] / m0[0], v0y = m0[2] / m0[0];
      const double pr0 = gm1 * (m0[3] - 0.5 * (m0[1] * m0[1] + m0[2] * m0[2]) / m0[0]);
      const double T0 = pr0 / r0;
      const double pr = gm1 * (m[3] - 0.5 * (m[1] * m[1] + m[2] * m[2]) / m[0]);
      const double rho = f0 * r0 + ft * m[0];
      const double vx = f0 * v0x + ft * (m[1] / m[0]);
      const double vy = f0 * v0y + ft * (m[2] / m[0]);
      const double T = f0 * T0 + ft * (pr / m[0]);
      nod[q][r][0] = rho;
      nod[q][r][1] = rho * vx;
      nod[q][r][2] = rho * vy;
      nod[q][r][3] = rho * T / gm1 + 0.5 * rho * (vx * vx + vy * vy);
    }
  for (int v = 0; v < NV; ++v)
    for (int b = 0; b < mo; ++b)
      for (int a = 0; a < mo; ++a) {
        double s = 0.0;
        for (int q = 0; q < mo; ++q)
          for (int r = 0; r < mo; ++r) s += T.w[q] * T.w[r] * nod[q][r][v] * T.B[q][a] * T.B[r][b];
        u[(v * mo + b) * mo + a] = 0.25 * s;
      }
}

void damp(ref_ctx* c, double dt) {
  const ref_params& p = c->p;
  if (!(p.damp_r0 > 0.0) && !(p.damp_in_r0 > 0.0)) return;
  const int m = c->m;
  const double pi = 3.14159265358979323846;
  for (int j = 0; j < p.ny; ++j)
    for (int i = 0; i < p.nx; ++i) {
      const double xc = p.x0 + (i + 0.5) * c->dx, yc = p.y0 + (j + 0.5) * c->dy;
      const double r = std::sqrt(xc * xc + yc * yc);
      double rd, s;
      if (p.damp_r0 > 0.0 && r > p.damp_r0) {
        rd = p.damp_r0;
        s = (r - p.damp_r0) / (p.damp_r1 - p.damp_r0);
      } else if (p.damp_in_r0 > 0.0 && r < p.damp_in_r0) {
        rd = p.damp_in_r0;
        s = (p.damp_in_r0 - r) / (p.damp_in_r0 - p.damp_in_r1);
      } else {
        continue;
      }
      double R = s * s;
      if (R > 1.0) R = 1.0;
      if (!(R > 0.0)) continue;
      const double tau = 2.0 * pi * std::sqrt(rd * rd * rd / p.gm_star) / R;
      double* u = c->U.data() + cell_off(c, i, j);
      const double* u0 = c->U0.data() + cell_off(c, i, j);
      if (p.damp_mode == 1) damp_cell_primitive(c, dt / (tau + dt), tau / (tau + dt), u, u0);
      else for (int k = 0; k < NV * m * m; ++k) u[k] = (dt * u0[k] + tau * u[k]) / (tau + dt);
    }
}

/* ---- C12: positivity-preserving limiter (Zhang & Shu 2010, step (iii)(d) PAPER.md:150) ----
 * Point set S_K of a rectangle (Zhang & Shu 2010, their S_ij): (Gauss_m in x) x (Lobatto_nh in y) united
 * with (Lobatto_nh in x) x (Gauss_m in y), nh the smallest Gauss-Lobatto rule exact for degree
 * N_p: 2 nh - 3 >= N_p; plus the m x m tensor Gauss points at which the volume integral of Eq.(3)
 * samples the flux (Zhang & Shu's remark that the points used by the scheme's quadratures belong to
 * the set; reading L2), so that every state the scheme evaluates a flux at is admissible. */

void build_lobatto(int m, LimTables* LT) {
  const int Np = m - 1;
  int nh = 2;
  while (2 * nh - 3 < Np) ++nh;
  LT->nh = nh;
  const int n = nh - 1;                   /* interior nodes are the roots of P_n' */
  const double pi = 3.14159265358979323846;
  LT->xh[0] = -1.0; LT->xh[n] = 1.0;
  for (int k = 1; k < n; ++k) {
    double x = -std::cos(pi * k / n);     /* Chebyshev-Lobatto guess, ascending */
    for (int it = 0; it < 100; ++it) {
      double P, dP;
      legendre(n, x, &P, &dP);
      const double d2P = (2.0 * x * dP - n * (n + 1.0) * P) / (1.0 - x * x);   /* Legendre's equation */
      const double dx = dP / d2P;
      x -= dx;
      if (std::fabs(dx) < 1e-16) break;
    }
    LT->xh[k] = x;
  }
  if (n % 2 == 0) LT->xh[n / 2] = 0.0;
  for (int k = 0; k <= n; ++k) {
    double P, dP;
    legendre(n, LT->xh[k], &P, &dP);
    LT->wh[k] = 0.5 * 2.0 / (n * (n + 1.0) * P * P);                          /* sum = 1 */
    for (int a = 0; a < m; ++a) {
      double Pa, dPa;
      legendre(a, LT->xh[k], &Pa, &dPa);
      LT->Bh[k][a] = std::sqrt(2.0 * a + 1.0) * Pa;
    }
  }
}

/* value of the cell polynomial with basis values px[a] = phi_a(x), py[b] = phi_b(y) */
void eval_cell(int m, const double* u, const double* px, const double* py, double* out) {
  for (int v = 0; v < NV; ++v) {
    double s = 0.0;
    for (int b = 0; b < m; ++b)
      for (int a = 0; a < m; ++a) s += u[(v * m + b) * m + a] * px[a] * py[b];
    out[v] = s;
  }
}

inline double pressure_ideal(const ref_params& p, const double* U) {
  return (p.gamma - 1.0) * (U[3] - 0.5 * (U[1] * U[1] + U[2] * U[2]) / U[0]);
}

/* the points of S_K, one after the other: k-th point's basis values */
struct LimPoint { const double* px; const double* py; };
int limiter_points(const Tables& T, const LimTables& LT, LimPoint* pts) {
  int n = 0;
  for (int q = 0; q < T.m; ++q)
    for (int k = 0; k < LT.nh; ++k) {
      pts[n].px = T.B[q];  pts[n].py = LT.Bh[k]; ++n;      /* Gauss in x, Lobatto in y */
      pts[n].px = LT.Bh[k]; pts[n].py = T.B[q];  ++n;      /* Lobatto in x, Gauss in y */
    }
  for (int q = 0; q < T.m; ++q)
    for (int r = 0; r < T.m; ++r) { pts[n].px = T.B[q]; pts[n].py = T.B[r]; ++n; }   /* volume Gauss points */
  return n;
}

void limit_cell(const ref_params& p, const Tables& T, const LimTables& LT, double* u, double* theta) {
  const int m = T.m;
  double th1 = 1.0, th2 = 1.0;
  if (m > 1) {
    LimPoint pts[2 * MAXM * 4 + MAXM * MAXM];
    const int npts = limiter_points(T, LT, pts);
    double ubar[NV];
    for (int v = 0; v < NV; ++v) ubar[v] = u[v * m * m];          /* mode (0,0) = cell average */
    /* step 1: density.  theta1 = min(1, (rhobar - eps)/(rhobar - rho_min)) */
    double rho_min = ubar[0];
    for (int k = 0; k < npts; ++k) {
      double s[NV];
      eval_cell(m, u, pts[k].px, pts[k].py, s);
      if (s[0] < rho_min) rho_min = s[0];
    }
    const double eps_rho = std::fmin(p.lim_eps, ubar[0]);
    if (rho_min < eps_rho) {
      th1 = (ubar[0] - eps_rho) / (ubar[0] - rho_min);
      for (int k = 1; k < m * m; ++k) u[k] *= th1;                /* rho <- rhobar + theta1 (rho - rhobar) */
    }
    /* step 2: pressure (ideal gas only; the isothermal closure has p = c_s^2 rho > 0 with rho).
     * For every point with p < eps, the intersection s(t) = ubar + t (u(x) - ubar) of the segment
     * with the surface p = eps; theta2 = min t. */
    if (p.eos == 0) {
      const double pbar = pressure_ideal(p, ubar);
      const double eps_p = std::fmin(p.lim_eps, pbar);
      const double e1 = eps_p / (p.gamma - 1.0);
      for (int k = 0; k < npts; ++k) {
        double s[NV];
        eval_cell(m, u, pts[k].px, pts[k].py, s);
        if (pressure_ideal(p, s) < eps_p) {
          /* g(t) = E(t) rho(t) - |m(t)|^2/2 - e1 rho(t) = A t^2 + B t + C, g(0) >= 0 > g(1) */
          const double dr = s[0] - ubar[0], dmx = s[1] - ubar[1], dmy = s[2] - ubar[2], dE = s[3] - ubar[3];
          const double A = dE * dr - 0.5 * (dmx * dmx + dmy * dmy);
          const double B = ubar[3] * dr + ubar[0] * dE - (ubar[1] * dmx + ubar[2] * dmy) - e1 * dr;
          const double C = ubar[3] * ubar[0] - 0.5 * (ubar[1] * ubar[1] + ubar[2] * ubar[2]) - e1 * ubar[0];
          const double disc = B * B - 4.0 * A * C;
          const double den = std::sqrt(disc > 0.0 ? disc : 0.0) - B;
          double t = den > 0.0 ? 2.0 * C / den : 0.0;             /* the root the segment meets first */
          if (!(t >= 0.0)) t = 0.0;
          if (t > 1.0) t = 1.0;
          if (t < th2) th2 = t;
        }
      }
      if (th2 < 1.0)
        for (int v = 0; v < NV; ++v)
          for (int k = 1; k < m * m; ++k) u[v * m * m + k] *= th2;
    }
  }
  if (theta) { theta[0] = th1; theta[1] = th2; }
}

void limit_all(const ref_ctx* c, const LimTables& LT, double* U) {
#pragma omp parallel for schedule(static)
  for (int j = 0; j < c->p.ny; ++j)
    for (int i = 0; i < c->p.nx; ++i) limit_cell(c->p, c->T, LT, U + cell_off(c, i, j), nullptr);
}

/* ---- C8b: explicit Runge-Kutta in Butcher form (Appendix A) ----
 * Coefficients typed from the paper: Table 1 and Table 2.
 * Table 1's printed b row sums to 1 - 8.8e-11 (14 printed digits): b is divided by its sum
 * (reading G20) so that the scheme stays exactly consistent. */
struct Butcher { int s; double a[6][6], b[6], c[6]; };

void butcher_tableau(int rk, Butcher* T) {
  std::memset(T, 0, sizeof *T);
  if (rk == 4) {
    T->s = 5;
    T->c[1] = 0.39175222700392; T->a[1][0] = 0.39175222700392;
    T->c[2] = 0.58607968896779; T->a[2][0] = 0.21766909633821; T->a[2][1] = 0.36841059262959;
    T->c[3] = 0.47454236302687; T->a[3][0] = 0.08269208670950; T->a[3][1] = 0.13995850206999;
    T->a[3][2] = 0.25189177424738;
    T->c[4] = 0.93501063100924; T->a[4][0] = 0.06796628370320; T->a[4][1] = 0.11503469844438;
    T->a[4][2] = 0.20703489864929; T->a[4][3] = 0.54497475021237;
    T->b[0] = 0.14681187618661; T->b[1] = 0.24848290924556; T->b[2] = 0.10425883036650;
    T->b[3] = 0.27443890091960; T->b[4] = 0.22600748319395;
    double sum = 0.0;
    for (int i = 0; i < 5; ++i) sum += T->b[i];
    for (int i = 0; i < 5; ++i) T->b[i] /= sum;
  } else {                                /* rk == 5: Cash & Karp 1990 */
    T->s = 6;
    T->c[1] = 1.0 / 5.0;  T->a[1][0] = 1.0 / 5.0;
    T->c[2] = 3.0 / 10.0; T->a[2][0] = 3.0 / 40.0; T->a[2][1] = 9.0 / 40.0;
    T->c[3] = 3.0 / 5.0;  T->a[3][0] = 3.0 / 10.0; T->a[3][1] = -9.0 / 10.0; T->a[3][2] = 6.0 / 5.0;
    T->c[4] = 1.0;        T->a[4][0] = -11.0 / 54.0; T->a[4][1] = 5.0 / 2.0; T->a[4][2] = -70.0 / 27.0;
    T->a[4][3] = 35.0 / 27.0;
    T->c[5] = 7.0 / 8.0;  T->a[5][0] = 1631.0 / 55296.0; T->a[5][1] = 175.0 / 512.0;
    T->a[5][2] = 575.0 / 13824.0; T->a[5][3] = 44275.0 / 110592.0; T->a[5][4] = 253.0 / 4096.0;
    T->b[0] = 37.0 / 378.0; T->b[2] = 250.0 / 621.0; T->b[3] = 125.0 / 594.0; T->b[5] = 512.0 / 1771.0;
  }
}

typedef void (*post_fn)(void* user, double* y);   /* applied to every sub-step's result (the limiter) */

/* y_i = y^n + h sum_{j<i} a_ij k_j,  k_i = f(t^n + c_i h, y_i),  y^{n+1} = y^n + h sum_i b_i k_i.
 * stages receives y_2 .. y_s and y^{n+1}: the results of the s sub-steps. */
int butcher_step(int rk, long n, double* y, double t, double dt, ref_ode_fn f, void* user,
                 double* stages, post_fn post, void* post_user) {
  Butcher T;
  butcher_tableau(rk, &T);
  std::vector<std::vector<double>> k(T.s, std::vector<double>(n));
  std::vector<double> yi(y, y + n);
  for (int i = 0; i < T.s; ++i) {
    f(user, t + T.c[i] * dt, yi.data(), k[i].data());
    const double* coef = (i + 1 < T.s) ? T.a[i + 1] : T.b;
    for (long e = 0; e < n; ++e) {
      double s = 0.0;
      for (int j = 0; j <= i; ++j) s += coef[j] * k[j][e];
      yi[e] = y[e] + dt * s;
    }
    if (post) post(post_user, yi.data());
    if (stages) std::memcpy(stages + (size_t)i * n, yi.data(), sizeof(double) * n);
  }
  std::memcpy(y, yi.data(), sizeof(double) * n);
  return 0;
}

int check_params(const ref_params* p) {
  if (!p) return -1;
  if (p->nx < 1 || p->ny < 1 || p->order < 1 || p->order > MAXM) return -1;
  if (!(p->x1 > p->x0) || !(p->y1 > p->y0)) return -1;
  if (p->rk < 2 || p->rk > 5) return -1;
  if (p->bc < 0 || p->bc > 2 || p->eos < 0 || p->eos > 1) return -1;
  if (p->eos == 0 && !(p->gamma > 1.0)) return -1;
  if (p->eos == 1 && !(p->h_aspect > 0.0 && p->gm_star > 0.0)) return -1;
  if (p->damp_r0 > 0.0 && !(p->damp_r1 > p->damp_r0 && p->gm_star > 0.0)) return -1;
  if (p->limiter != 0 && p->limiter != 1) return -1;
  if (p->flux != 0 && p->flux != 1) return -1;
  if (p->limiter == 1 && !(p->lim_eps > 0.0)) return -1;
  if (p->damp_in_r0 > 0.0 && !(p->damp_in_r1 >= 0.0 && p->damp_in_r1 < p->damp_in_r0 && p->gm_star > 0.0)) return -1;
  if (p->damp_mode != 0 && p->damp_mode != 1) return -1;
  return 0;
}

}  // namespace

extern "C" {

int ref_init(const ref_params* p, ref_ctx** out) {
  if (!out || check_params(p) != 0) return -1;
  ref_ctx* c = new ref_ctx;
  c->p = *p;
  c->m = p->order;
  build_tables(c->m, &c->T);
  build_lobatto(c->m, &c->LT);
  c->ncoef = (long)p->ny * p->nx * NV * c->m * c->m;
  c->dx = (p->x1 - p->x0) / p->nx;
  c->dy = (p->y1 - p->y0) / p->ny;
  c->t = p->t0;
  c->has_state = false;
  *out = c;
  return 0;
}

int ref_set_state(ref_ctx* c, const double* U) {
  if (!c || !U) return -1;
  c->U.assign(U, U + c->ncoef);
  c->U0 = c->U;
  c->has_state = true;
  return 0;
}

int ref_load_working_state(ref_ctx* c, const double* U) {
  if (!c || !U || !c->has_state) return -1;
  c->U.assign(U, U + c->ncoef);
  return 0;
}

int ref_get_state(ref_ctx* c, double* U) {
  if (!c || !U || !c->has_state) return -1;
  std::memcpy(U, c->U.data(), sizeof(double) * c->ncoef);
  return 0;
}

int ref_rhs(ref_ctx* c, double t, double* L) { return ref_rhs_parts(c, t, 7, L); }

int ref_rhs_parts(ref_ctx* c, double t, int parts, double* L) {
  if (!c || !L || !c->has_state) return -1;
  compute_rhs(c, c->U.data(), t, parts, L);
  return 0;
}

/* C10 */
int ref_cfl_dt(ref_ctx* c, double cfl, double* dt) {
  if (!c || !dt || !c->has_state) return -1;
  const ref_params& p = c->p;
  const int m = c->m;
  double worst = 0.0;
  for (int j = 0; j < p.ny; ++j)
    for (int i = 0; i < p.nx; ++i) {
      const double* u = c->U.data() + cell_off(c, i, j);
      const double rho = u[0 * m * m], mx = u[1 * m * m], my = u[2 * m * m], E = u[3 * m * m];
      const double vx = mx / rho, vy = my / rho;
      double cs;
      if (p.eos == 0) {
        const double pr = (p.gamma - 1.0) * (E - 0.5 * (mx * mx + my * my) / rho);
        cs = std::sqrt(p.gamma * pr / rho);
      } else {
        const double xc = p.x0 + (i + 0.5) * c->dx, yc = p.y0 + (j + 0.5) * c->dy;
        cs = std::sqrt(cs2_iso(p, xc, yc));
      }
      const double s = (std::fabs(vx) + cs) / c->dx + (std::fabs(vy) + cs) / c->dy;
      if (s > worst) worst = s;
    }
  double factor = 1.0 / (2.0 * (m - 1) + 1.0);
  if (p.limiter) factor = std::fmin(factor, 0.5 * c->LT.wh[0]);     /* min(1/(2N_p+1), w_1/2) */
  *dt = cfl * factor / worst;
  return 0;
}

int ref_rk_stages(int rk) { return rk == 2 ? 2 : rk == 3 ? 3 : rk == 4 ? 5 : rk == 5 ? 6 : -1; }

/* C8: Shu-Osher form of SSP(2,2) and SSP(3,3) (Gottlieb & Shu 1998), stage times
 * c = (0,1) and (0,1,1/2); rk 4, 5: Butcher form (C8b).  post: applied to every sub-step's result. */
static int rk_step_impl(int rk, long n, double* y, double t, double dt, ref_ode_fn f, void* user,
                        double* stages, post_fn post, void* pu) {
  if (rk == 4 || rk == 5) return butcher_step(rk, n, y, t, dt, f, user, stages, post, pu);
  if (rk != 2 && rk != 3) return -1;
  std::vector<double> L(n), u1(n), u2(n);
  f(user, t, y, L.data());
  for (long k = 0; k < n; ++k) u1[k] = y[k] + dt * L[k];
  if (post) post(pu, u1.data());
  if (stages) std::memcpy(stages, u1.data(), sizeof(double) * n);
  f(user, t + dt, u1.data(), L.data());
  if (rk == 2) {
    for (long k = 0; k < n; ++k) y[k] = 0.5 * y[k] + 0.5 * (u1[k] + dt * L[k]);
    if (post) post(pu, y);
    if (stages) std::memcpy(stages + n, y, sizeof(double) * n);
    return 0;
  }
  for (long k = 0; k < n; ++k) u2[k] = 0.75 * y[k] + 0.25 * (u1[k] + dt * L[k]);
  if (post) post(pu, u2.data());
  if (stages) std::memcpy(stages + n, u2.data(), sizeof(double) * n);
  f(user, t + 0.5 * dt, u2.data(), L.data());
  for (long k = 0; k < n; ++k) y[k] = (1.0 / 3.0) * y[k] + (2.0 / 3.0) * (u2[k] + dt * L[k]);
  if (post) post(pu, y);
  if (stages) std::memcpy(stages + 2 * n, y, sizeof(double) * n);
  return 0;
}

int ref_rk_step(int rk, long n, double* y, double t, double dt, ref_ode_fn f, void* user,
                double* stages) {
  return rk_step_impl(rk, n, y, t, dt, f, user, stages, nullptr, nullptr);
}

static void limiter_hook(void* user, double* y) {
  const ref_ctx* c = static_cast<const ref_ctx*>(user);
  limit_all(c, c->LT, y);
}

/* one time step: the RK sub-steps (C8 / C8b), each followed by the limiter when it is on
 * (step (iii)(d)), then the wave damping (C11) */
int ref_step_debug(ref_ctx* c, double dt, double* stages) {
  if (!c || !c->has_state) return -1;
  RhsClosure cl{c};
  int e = rk_step_impl(c->p.rk, c->ncoef, c->U.data(), c->t, dt, dg_ode, &cl, stages,
                       c->p.limiter ? limiter_hook : nullptr, c);
  if (e) return e;
  damp(c, dt);
  c->t += dt;
  return 0;
}

int ref_limit(ref_ctx* c) {
  if (!c || !c->has_state) return -1;
  limit_all(c, c->LT, c->U.data());
  return 0;
}

int ref_lobatto(int m, double* xh, double* wh) {
  if (m < 1 || m > MAXM || !xh || !wh) return -1;
  LimTables LT;
  build_lobatto(m, &LT);
  for (int k = 0; k < LT.nh; ++k) { xh[k] = LT.xh[k]; wh[k] = LT.wh[k]; }
  return LT.nh;
}

int ref_limit_cell(const ref_params* p, double* u, double* theta) {
  if (check_params(p) != 0 || !u) return -1;
  Tables T;
  LimTables LT;
  build_tables(p->order, &T);
  build_lobatto(p->order, &LT);
  limit_cell(*p, T, LT, u, theta);
  return 0;
}

/* C13: specific torque on the planet, Eq.(6) PAPER.md:321-328:
 *   Gamma = r_p x sum_n G M_n (r_n - r_p) / (|r_n - r_p|^2 + eps_p^2)^(3/2)   (z component),
 * M_n = (cell average of the density) x (cell area), r_n = the cell centre, planet position at time t. */
int ref_torque(ref_ctx* c, double t, double* gamma_z) {
  if (!c || !gamma_z || !c->has_state) return -1;
  const ref_params& p = c->p;
  const int m = c->m;
  const double ang = p.omega_planet * t + p.phase0;
  const double xp = p.r_planet * std::cos(ang), yp = p.r_planet * std::sin(ang);
  double ax = 0.0, ay = 0.0;
  for (int j = 0; j < p.ny; ++j)
    for (int i = 0; i < p.nx; ++i) {
      const double Mn = c->U[cell_off(c, i, j)] * c->dx * c->dy;
      const double ddx = p.x0 + (i + 0.5) * c->dx - xp, ddy = p.y0 + (j + 0.5) * c->dy - yp;
      const double r2 = ddx * ddx + ddy * ddy + p.eps_planet * p.eps_planet;
      const double r3 = r2 * std::sqrt(r2);
      ax += p.gm_star * Mn * ddx / r3;
      ay += p.gm_star * Mn * ddy / r3;
    }
  (void)m;
  *gamma_z = xp * ay - yp * ax;
  return 0;
}

/* C13b: the quantity the paper plots, gamma Gamma / Gamma_0 with Gamma_0 = Sigma Omega^2 r_p^4 q / h^2 */
int ref_torque_normalised(ref_ctx* c, double t, double sigma_p, double* out) {
  if (!c || !out || !(c->p.q_planet > 0.0) || !(c->p.h_aspect > 0.0)) return -1;
  double g;
  if (ref_torque(c, t, &g) != 0) return -1;
  const ref_params& p = c->p;
  const double rp2 = p.r_planet * p.r_planet;
  const double gamma0 = sigma_p * p.omega_planet * p.omega_planet * rp2 * rp2 * p.q_planet / (p.h_aspect * p.h_aspect);
  *out = p.gamma * g / gamma0;
  return 0;
}

int ref_step(ref_ctx* c, double dt) { return ref_step_debug(c, dt, nullptr); }

int ref_damp(ref_ctx* c, double dt) {
  if (!c || !c->has_state) return -1;
  damp(c, dt);
  return 0;
}

double ref_time(const ref_ctx* c) { return c ? c->t : 0.0; }
int ref_set_time(ref_ctx* c, double t) { if (!c) return -1; c->t = t; return 0; }
void ref_destroy(ref_ctx* c) { delete c; }

int ref_tables(int m, double* xi, double* w, double* B, double* D, double* Ep, double* Em) {
  if (m < 1 || m > MAXM) return -1;
  Tables T;
  build_tables(m, &T);
  for (int q = 0; q < m; ++q) {
    xi[q] = T.xi[q]; w[q] = T.w[q]; Ep[q] = T.Ep[q]; Em[q] = T.Em[q];
    for (int a = 0; a < m; ++a) { B[q * m + a] = T.B[q][a]; D[q * m + a] = T.D[q][a]; }
  }
  return 0;
}

int ref_point_flux(const ref_params* p, const double* U4, double x, double y, int dir,
                   double* F4, double* vn, double* c) {
  if (!p || (dir != 0 && dir != 1)) return -1;
  point_flux(*p, U4, x, y, dir, F4, vn, c);
  return 0;
}

int ref_llf(const ref_params* p, const double* UL, const double* UR, double x, double y, int dir,
            double* H4) {
  if (!p || (dir != 0 && dir != 1)) return -1;
  llf(*p, UL, UR, x, y, dir, H4);
  return 0;
}

int ref_hllc(const ref_params* p, const double* UL, const double* UR, double x, double y, int dir,
             double* H4) {
  if (!p || (dir != 0 && dir != 1)) return -1;
  hllc(*p, UL, UR, x, y, dir, H4);
  return 0;
}

int ref_gravity(const ref_params* p, double t, double x, double y, double* g2) {
  if (!p) return -1;
  gravity(*p, t, x, y, g2);
  return 0;
}

int ref_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void ref_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

}  // extern "C"
