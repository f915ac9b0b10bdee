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

}  // namespace dg
