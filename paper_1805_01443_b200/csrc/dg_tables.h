// Host-side quadrature / basis tables for the CUDA path ("quadrature values and
// their respective weights as well as the Legendre polynomials evaluated at these quadrature
// points").  Built from closed forms (m <= 5), independently of the oracle's Newton/recurrence code.
//
// The state lives on the device as NODAL values at the m x m tensor Gauss-Legendre points
// (DESIGN.md "Data layout").  With m points for m modes the map modes <-> nodal values is a
// bijection and the m-point rule makes the mass matrix diagonal in both bases,
// so Eq.(3) becomes, at node (q', r'):
//   N(q',r') = (1/dx) [ sum_q Dh[q'][q] F(q,r') - lp[q'] Fhat_E(r') + lm[q'] Fhat_W(r') ]
//            + (1/dy) [ sum_r Dh[r'][r] G(q',r) - lp[r'] Ghat_N(q') + lm[r'] Ghat_S(q') ] + S(q',r')
// with   Dh[q'][q] = w_q sum_a phi_a(xi_q') phi_a'(xi_q),   l+-[q'] = sum_a phi_a(xi_q') phi_a(+-1),
// and the face traces  u(+-1, eta_r) = sum_q I+-[q] u(q,r),  I+-[q] = (w_q/2) l+-[q].
#pragma once
#include <cmath>

namespace dg {

constexpr int MAXM = 5;

struct HostTables {
  int m;
  double xi[MAXM], w[MAXM];
  double B[MAXM][MAXM];     // B[q][a] = phi_a(xi_q)
  double P[MAXM][MAXM];     // P[q][a] = (w_q/2) phi_a(xi_q)        (nodal -> modal)
  double Dh[MAXM][MAXM];    // Dh[q'][q]
  double lp[MAXM], lm[MAXM];
  double Ip[MAXM], Im[MAXM];
};

inline long double legendre_closed(int n, long double x) {
  switch (n) {
    case 0: return 1.0L;
    case 1: return x;
    case 2: return 0.5L * (3.0L * x * x - 1.0L);
    case 3: return 0.5L * (5.0L * x * x * x - 3.0L * x);
    default: return 0.125L * (35.0L * x * x * x * x - 30.0L * x * x + 3.0L);
  }
}
inline long double dlegendre_closed(int n, long double x) {
  switch (n) {
    case 0: return 0.0L;
    case 1: return 1.0L;
    case 2: return 3.0L * x;
    case 3: return 0.5L * (15.0L * x * x - 3.0L);
    default: return 0.125L * (140.0L * x * x * x - 60.0L * x);
  }
}

// Gauss-Legendre rules in closed form (Abramowitz & Stegun 25.4.29), nodes ascending.
inline void gauss_legendre_closed(int m, long double* x, long double* w) {
  const long double s30 = sqrtl(30.0L), s70 = sqrtl(70.0L);
  switch (m) {
    case 1: x[0] = 0; w[0] = 2; break;
    case 2: x[1] = 1.0L / sqrtl(3.0L); x[0] = -x[1]; w[0] = w[1] = 1; break;
    case 3: x[2] = sqrtl(0.6L); x[1] = 0; x[0] = -x[2];
            w[0] = w[2] = 5.0L / 9.0L; w[1] = 8.0L / 9.0L; break;
    case 4: {
      long double a = sqrtl(3.0L / 7.0L - 2.0L / 7.0L * sqrtl(1.2L));
      long double b = sqrtl(3.0L / 7.0L + 2.0L / 7.0L * sqrtl(1.2L));
      x[0] = -b; x[1] = -a; x[2] = a; x[3] = b;
      w[1] = w[2] = (18.0L + s30) / 36.0L; w[0] = w[3] = (18.0L - s30) / 36.0L; break;
    }
    default: {
      long double a = sqrtl(5.0L - 2.0L * sqrtl(10.0L / 7.0L)) / 3.0L;
      long double b = sqrtl(5.0L + 2.0L * sqrtl(10.0L / 7.0L)) / 3.0L;
      x[0] = -b; x[1] = -a; x[2] = 0; x[3] = a; x[4] = b;
      w[2] = 128.0L / 225.0L;
      w[1] = w[3] = (322.0L + 13.0L * s70) / 900.0L; w[0] = w[4] = (322.0L - 13.0L * s70) / 900.0L; break;
    }
  }
}

inline void build_host_tables(int m, HostTables* T) {
  long double x[MAXM], w[MAXM], B[MAXM][MAXM], D[MAXM][MAXM];
  gauss_legendre_closed(m, x, w);
  T->m = m;
  for (int q = 0; q < m; ++q)
    for (int a = 0; a < m; ++a) {
      const long double s = sqrtl(2.0L * a + 1.0L);
      B[q][a] = s * legendre_closed(a, x[q]);
      D[q][a] = s * dlegendre_closed(a, x[q]);
    }
  for (int q = 0; q < m; ++q) {
    T->xi[q] = (double)x[q];
    T->w[q] = (double)w[q];
    long double lp = 0, lm = 0;
    for (int a = 0; a < m; ++a) {
      const long double s = sqrtl(2.0L * a + 1.0L);
      T->B[q][a] = (double)B[q][a];
      T->P[q][a] = (double)(0.5L * w[q] * B[q][a]);
      lp += B[q][a] * s;
      lm += B[q][a] * ((a & 1) ? -s : s);
    }
    T->lp[q] = (double)lp;
    T->lm[q] = (double)lm;
    T->Ip[q] = (double)(0.5L * w[q] * lp);
    T->Im[q] = (double)(0.5L * w[q] * lm);
    for (int qq = 0; qq < m; ++qq) {       // Dh[q][qq] = w_qq sum_a B[q][a] D[qq][a]
      long double s = 0;
      for (int a = 0; a < m; ++a) s += B[q][a] * D[qq][a];
      T->Dh[q][qq] = (double)(w[qq] * s);
    }
  }
}

// Tables of the positivity limiter (Zhang & Shu 2010): the Gauss-Lobatto rule with
// the fewest points that is exact for degree N_p = m-1 (2 nh - 3 >= N_p), nodes in closed form
// (nh = 2: +-1; 3: 0, +-1; 4: +-1, +-1/sqrt 5), its first weight normalised to sum 1,
// w_1 = 1/(nh (nh-1)) (the factor of PAPER.md:131), and the interpolation Lh[k][r] = l_r(xh_k) from
// the Gauss nodes to the Lobatto nodes, l_r(x) = sum_a P[r][a] phi_a(x).
struct HostLimTables {
  int nh;
  double xh[4];
  double w1;
  double Lh[4][MAXM];
};

inline void build_limiter_tables(int m, HostLimTables* L) {
  const int nh = m <= 2 ? 2 : (m <= 4 ? 3 : 4);
  long double xh[4];
  if (nh == 2) { xh[0] = -1; xh[1] = 1; }
  else if (nh == 3) { xh[0] = -1; xh[1] = 0; xh[2] = 1; }
  else { const long double a = 1.0L / sqrtl(5.0L); xh[0] = -1; xh[1] = -a; xh[2] = a; xh[3] = 1; }
  long double x[MAXM], w[MAXM];
  gauss_legendre_closed(m, x, w);
  L->nh = nh;
  L->w1 = 1.0 / (double)(nh * (nh - 1));
  for (int k = 0; k < nh; ++k) {
    L->xh[k] = (double)xh[k];
    for (int r = 0; r < m; ++r) {
      long double s = 0;
      for (int a = 0; a < m; ++a)
        s += 0.5L * w[r] * (2.0L * a + 1.0L) * legendre_closed(a, x[r]) * legendre_closed(a, xh[k]);
      L->Lh[k][r] = (double)s;
    }
  }
}

// Explicit Runge-Kutta schemes in Butcher form (Appendix A), coefficients typed from
// the paper: rk 4 = Table 1 (five-stage fourth-order SSP scheme), rk 5 = Table 2
// (Cash & Karp).  Table 1's printed b row sums to 1 - 8.8e-11 (14 digits): b is
// divided by its sum so that the scheme is exactly consistent (reading G20).
struct ButcherTableau { int s; double a[6][6], b[6], c[6]; };

inline bool butcher_tableau(int rk, ButcherTableau* B) {
  *B = ButcherTableau{};
  if (rk == 4) {
    static const double A54[5][5] = {
        {0, 0, 0, 0, 0},
        {0.39175222700392, 0, 0, 0, 0},
        {0.21766909633821, 0.36841059262959, 0, 0, 0},
        {0.08269208670950, 0.13995850206999, 0.25189177424738, 0, 0},
        {0.06796628370320, 0.11503469844438, 0.20703489864929, 0.54497475021237, 0}};
    static const double b54[5] = {0.14681187618661, 0.24848290924556, 0.10425883036650, 0.27443890091960,
                                  0.22600748319395};
    static const double c54[5] = {0, 0.39175222700392, 0.58607968896779, 0.47454236302687, 0.93501063100924};
    B->s = 5;
    double sum = 0.0;
    for (int i = 0; i < 5; ++i) sum += b54[i];
    for (int i = 0; i < 5; ++i) {
      B->b[i] = b54[i] / sum;
      B->c[i] = c54[i];
      for (int j = 0; j < 5; ++j) B->a[i][j] = A54[i][j];
    }
    return true;
  }
  if (rk == 5) {
    B->s = 6;
    B->c[1] = 1.0 / 5; B->c[2] = 3.0 / 10; B->c[3] = 3.0 / 5; B->c[4] = 1.0; B->c[5] = 7.0 / 8;
    B->a[1][0] = 1.0 / 5;
    B->a[2][0] = 3.0 / 40; B->a[2][1] = 9.0 / 40;
    B->a[3][0] = 3.0 / 10; B->a[3][1] = -9.0 / 10; B->a[3][2] = 6.0 / 5;
    B->a[4][0] = -11.0 / 54; B->a[4][1] = 5.0 / 2; B->a[4][2] = -70.0 / 27; B->a[4][3] = 35.0 / 27;
    B->a[5][0] = 1631.0 / 55296; B->a[5][1] = 175.0 / 512; B->a[5][2] = 575.0 / 13824;
    B->a[5][3] = 44275.0 / 110592; B->a[5][4] = 253.0 / 4096;
    B->b[0] = 37.0 / 378; B->b[2] = 250.0 / 621; B->b[3] = 125.0 / 594; B->b[5] = 512.0 / 1771;
    return true;
  }
  return false;
}

// Any explicit scheme with non-zero sub-diagonal, rewritten on the stage STATES instead of the slopes: with
// y_1 = u^n and K_j = dt L(y_j), the Butcher rows y_l = u^n + sum_{j<l} a_lj K_j (l = 2..s+1, row s+1 = b) give
// K_j = (y_{j+1} - u^n - sum_{k<j} a_{j+1,k} K_k)/a_{j+1,j} recursively, hence
//   y_{i+2} = sum_{m=0..i} g[i][m] y_{m+1} + beta[i] dt L(y_{i+1}),     i = 0..s-1,   beta[i] = a_{i+2,i+1}.
// A sub-step then reads its input y_{i+1} (whose tile it holds anyway), u^n and the earlier states with
// g != 0, and writes ONE array -- no slope is ever stored.  Same arithmetic up to rounding (the
// reconstruction divides state differences of size dt |L| by a_{j+1,j}: errors of 1e-16 |y|).
struct StateForm { int s; bool ok; double g[6][7], beta[6]; };

inline StateForm state_form_from_butcher(const ButcherTableau& B) {
  StateForm F{};
  F.s = B.s;
  F.ok = true;
  double kap[6][7] = {};                       // K_j = sum_m kap[j][m] y_{m+1}
  for (int i = 0; i < B.s; ++i) {
    const double* row = (i + 1 < B.s) ? B.a[i + 1] : B.b;   // row of y_{i+2}
    F.beta[i] = row[i];
    if (row[i] == 0.0) F.ok = false;
    for (int m = 0; m < 7; ++m) F.g[i][m] = 0.0;
    F.g[i][0] = 1.0;
    for (int j = 0; j < i; ++j)
      for (int m = 0; m <= j + 1; ++m) F.g[i][m] += row[j] * kap[j][m];
    // K_i from y_{i+2} = sum_m g[i][m] y_{m+1} + row[i] K_i
    if (row[i] != 0.0) {
      for (int m = 0; m <= i; ++m) kap[i][m] = -F.g[i][m] / row[i];
      kap[i][i + 1] = 1.0 / row[i];
    }
  }
  return F;
}

// The same scheme when a limiter modifies every y_l after it is formed: the slopes cannot be
// recovered from the (limited) states, so each sub-step also keeps Z_i = abar_i u^n + beta_i K_i -- its result
// before the earlier slopes' terms are added, which the limiter never touches.  With K_j = (Z_j - abar_j u^n)/beta_j,
//   y_{i+2} = abar_i u^n + sum_{j<i} z[i][j] Z_j + beta_i K_i,  z[i][j] = row_i[j]/beta_j,  abar_i = 1 - sum_{j<i} z[i][j] abar_j.
struct ZForm { int s; bool ok; double abar[6], z[6][6], beta[6]; };

inline ZForm z_form_from_butcher(const ButcherTableau& B) {
  ZForm F{};
  F.s = B.s;
  F.ok = true;
  for (int i = 0; i < B.s; ++i) {
    const double* row = (i + 1 < B.s) ? B.a[i + 1] : B.b;
    F.beta[i] = row[i];
    if (row[i] == 0.0 && i + 1 < B.s) F.ok = false;
    double abar = 1.0;
    for (int j = 0; j < i; ++j) {
      F.z[i][j] = row[j] / F.beta[j];
      abar -= F.z[i][j] * F.abar[j];
    }
    F.abar[i] = abar;
  }
  return F;
}

// Table 1's scheme in the low-storage (Shu-Osher) form it has by construction: rows 2..5 of the printed
// tableau are multiples of the row above plus one new entry, a_{i+1,j} = alpha_i a_{ij} (j < i), so that
//   y_{i+1} = (1 - alpha_i) u^n + alpha_i y_i + beta_i dt L(y_i),  i = 1..4  (alpha_1 = 1),
//   u^{n+1} = c2 y_3 + c3 y_4 + c4 y_5 + d3 dt L(y_4) + d4 dt L(y_5)   (dt L(y_4) = (y_5 - (1-alpha_4) u^n - alpha_4 y_4)/beta_4),
// all coefficients solved from the printed a, b (b renormalised).  Algebraically the Butcher form; in
// floating point it differs from it at the printed tableau's own precision (1e-14).  `ok` is false if the
// tableau does not have that structure to 1e-12 (then the Butcher form is used).
struct Ssp54 { bool ok; double alpha[4], beta[4], c2, c3, c4, d3, d4; };

inline Ssp54 ssp54_from_butcher(const ButcherTableau& B) {
  Ssp54 S{};
  S.ok = B.s == 5;
  if (!S.ok) return S;
  S.alpha[0] = 1.0;
  S.beta[0] = B.a[1][0];
  for (int i = 1; i < 4; ++i) {
    S.alpha[i] = B.a[i + 1][0] / B.a[i][0];
    S.beta[i] = B.a[i + 1][i];
    for (int j = 0; j < i; ++j)
      if (std::fabs(B.a[i + 1][j] - S.alpha[i] * B.a[i][j]) > 1e-12) S.ok = false;
  }
  const double r = B.b[2] / B.a[3][2];                       // c3 + alpha_4 c4
  S.c2 = B.b[0] / B.a[2][0] - S.alpha[2] * r;
  const double sum = 1.0 - S.c2;                              // c3 + c4
  S.c4 = (sum - r) / (1.0 - S.alpha[3]);
  S.c3 = sum - S.c4;
  S.d3 = B.b[3] - S.c4 * B.a[4][3];
  S.d4 = B.b[4];
  const double b1 = S.c2 * B.a[2][1] + S.c3 * B.a[3][1] + S.c4 * B.a[4][1];
  if (std::fabs(b1 - B.b[1]) > 1e-12 || !(S.c2 > 0 && S.c3 > 0 && S.c4 > 0 && S.d3 > 0)) S.ok = false;
  return S;
}

}  // namespace dg
