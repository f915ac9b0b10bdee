/* CPU ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, single-threaded (optionally one `omp parallel for` over cell rows) fp64 restatement
 * of the explicit modal DG right-hand side + SSP-RK stage update of arXiv:1805.01443 for the 2D
 * Euler equations, written step by step in the paper's order and notation (SURVEY.md section 8(c),
 * items C1..C11; C8b, C12, C13 for the rows of SURVEY.md 8(f)).  Host pointers only.  Shares no code, header, table or constant generator with
 * the CUDA path (paper_1805_01443_b200/csrc, include/dg.h); neither includes the other.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * load this library.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): see the header of ref_dg.cpp.
 * Absolute per-step numbers: PARITY UNPINNED (the paper prints none for this path, Fig. 2
 * is an image) -- every other function below is pinned.
 */
#ifndef REF_DG_H
#define REF_DG_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct ref_ctx ref_ctx;

typedef struct {
  int32_t nx, ny;            /* uniform Cartesian grid of rectangles K_ij */
  double  x0, x1, y0, y1;
  int32_t order;             /* m = N_p + 1 = 1..5 */
  int32_t rk;                /* 2: SSP(2,2), 3: SSP(3,3); 4: SSP-RK(5,4), Table 1 PAPER.md:463-471;
                                5: Cash-Karp, Table 2 PAPER.md:473-482 (Butcher form, Appendix A) */
  int32_t bc;                /* 0 periodic, 1 transmissive, 2 frozen to the initial state */
  int32_t eos;               /* 0 ideal gas p=(gamma-1)e; 1 locally isothermal */
  double  gamma;
  double  h_aspect;          /* eos 1: c_s^2 = h^2 GM / sqrt(r^2 + eps_star^2) */
  double  gm_star, eps_star; /* softened star potential; gm_star = 0: no gravity at all */
  double  q_planet, r_planet, eps_planet, omega_planet, phase0; /* planet on a fixed circular orbit */
  double  damp_r0, damp_r1;  /* wave-killing zone r0 < r; r0 <= 0: off */
  double  t0;
  int32_t limiter;           /* 1: positivity-preserving limiter (Zhang & Shu 2010) after every
                                RK sub-step and the w_1/2 factor in the time step */
  double  lim_eps;           /* the limiter's floor for density and pressure (Zhang & Shu use 1e-13) */
  int32_t flux;              /* numerical flux h_{e,K} (type unnamed): 0 local Lax-Friedrichs (C5);
                                1 HLLC (eos 0; Toro, Spruce & Speares 1994) / HLL (eos 1), Davis wave speeds (C5b) */
  double  damp_in_r0, damp_in_r1; /* inner wave-killing zone r < damp_in_r0 (r_d = r_in 1.15^(3/2),
                                     boundary radius r_in = damp_in_r1); damp_in_r0 <= 0: off */
  int32_t damp_mode;         /* which fields the wave-killing zones relax (C11): 0 the conservative coefficients
                                (reading G13); 1 "the density, velocities and temperature" at the
                                m x m Gauss points, the conservative state rebuilt from them (reading D2) */
} ref_params;

/* --- the same surface as include/dg.h, prefixed ref_, host memory --- */
int    ref_init(const ref_params* p, ref_ctx** out);
int    ref_set_state(ref_ctx*, const double* U);   /* [ny][nx][4][m][m], snapshots U0 */
int    ref_get_state(ref_ctx*, double* U);
int    ref_rhs(ref_ctx*, double t, double* L);     /* L(u) of Eq.(3) divided by the mass, at time t */
int    ref_cfl_dt(ref_ctx*, double cfl, double* dt);
int    ref_step(ref_ctx*, double dt);              /* RK step (C8) + damping (C11); t += dt */
int    ref_step_debug(ref_ctx*, double dt, double* stages); /* also u^(1..k), before damping; k = ref_rk_stages */
int    ref_rk_stages(int rk);                      /* sub-steps of the scheme: 2, 3, 5 (rk 4), 6 (rk 5) */
int    ref_limit(ref_ctx*);                        /* C12 alone: limit the current state in place */
int    ref_torque(ref_ctx*, double t, double* gamma_z); /* C13: Eq.(6) */
/* C13b: gamma Gamma / Gamma_0, Gamma_0 = Sigma Omega^2 r_p^4 q / h^2; Sigma = sigma_p, the unperturbed
 * surface density at the planet (a property of the initial data, passed in), Omega = omega_planet, h = h_aspect */
int    ref_torque_normalised(ref_ctx*, double t, double sigma_p, double* out);
double ref_time(const ref_ctx*);
int    ref_set_time(ref_ctx*, double t);
void   ref_destroy(ref_ctx*);

/* --- pieces exposed so that tests can pin them one by one --- */
/* C1: Gauss-Legendre nodes/weights and the basis tables; arrays sized m, m, m*m, m*m, m, m. */
int  ref_tables(int m, double* xi, double* w, double* B, double* D, double* Eplus, double* Eminus);
/* C3/C4: physical flux in direction dir (0:x, 1:y) at point (x,y); returns normal velocity and c. */
int  ref_point_flux(const ref_params*, const double* U4, double x, double y, int dir,
                    double* F4, double* vn, double* c);
/* C5: local Lax-Friedrichs flux across a face with normal +dir, left state UL, right state UR. */
int  ref_llf(const ref_params*, const double* UL, const double* UR, double x, double y, int dir,
             double* H4);
/* C5b: HLLC (eos 0) / HLL (eos 1) flux, same arguments as ref_llf. */
int  ref_hllc(const ref_params*, const double* UL, const double* UR, double x, double y, int dir,
              double* H4);
/* C6: gravitational acceleration g = -grad Phi at (x,y), time t. */
int  ref_gravity(const ref_params*, double t, double x, double y, double* g2);
/* C7 split: parts bitmask 1 = volume flux term, 2 = face term, 4 = source term. */
int  ref_rhs_parts(ref_ctx*, double t, int parts, double* L);
/* C11 alone. */
int  ref_damp(ref_ctx*, double dt);
/* replaces the working state and leaves the snapshot U0 of the last ref_set_state alone (pins of C9, C11) */
int  ref_load_working_state(ref_ctx*, const double* U);
/* C12 pieces: Gauss-Lobatto nodes on [-1,1] and weights normalised to sum 1 (Zhang & Shu's hat-w)
 * for the limiter of order m (nh = ceil((m+2)/2) points); returns nh.  xh, wh sized 4. */
int  ref_lobatto(int m, double* xh, double* wh);
/* C12 on one cell: u[4][m][m] modal, in place; theta (nullable) receives theta1, theta2. */
int  ref_limit_cell(const ref_params*, double* u, double* theta);
/* C8 alone: one RK step of y' = f(t,y) for n unknowns; stages (nullable) receives y^(1..k). */
typedef void (*ref_ode_fn)(void* user, double t, const double* y, double* dydt);
int  ref_rk_step(int rk, long n, double* y, double t, double dt, ref_ode_fn f, void* user,
                 double* stages);
/* number of OpenMP threads the library will use (1 if built without -fopenmp) */
int  ref_threads(void);
void ref_set_threads(int n);

#ifdef __cplusplus
}
#endif
#endif
