/* libdg -- C-ABI boundary of the B200 (sm_100a) discontinuous-Galerkin Euler hot path.
 *
 * Method: arXiv:1805.01443 ("Planet-disc interactions with Discontinuous Galerkin Methods using
 * GPUs"), cited below as PAPER.md:<line> (the text under /root/reference at build time).
 * One GPU, fp64, DG orders m = 1..5 (polynomial degree N_p = m-1), uniform Cartesian mesh.
 *
 * Conventions
 * -----------
 *  - Plain C: pointers and sizes only.  Every pointer argument is tagged DEVICE or HOST below.
 *  - The library never allocates device memory: the caller passes a DEVICE workspace of at least
 *    dg_workspace_bytes() bytes (256-byte aligned) to dg_init and keeps it alive until dg_destroy.
 *    The library owns only the host-side context.
 *  - All work is enqueued on the CUDA stream given to dg_init (a cudaStream_t passed as void*,
 *    0 = legacy default stream).  Calls are asynchronous unless stated otherwise.
 *  - External state layout (both directions), fp64, C order:
 *        U[ny][nx][4][m][m]  =  U[j][i][v][b][a]
 *    j,i cell indices (i along x, fastest of the two), v in {rho, rho*vx, rho*vy, E},
 *    a = Legendre degree in x (fastest), b = degree in y, of the orthonormal tensor basis
 *    phi_a(xi) phi_b(eta), phi_n = sqrt(2n+1) P_n on the reference square [-1,1]^2
 *    (mode (0,0) is the cell average).
 *    Inside the workspace the state lives in a different, kernel-friendly layout.
 *  - Return value: 0 (DG_OK) or a negative DG_E* code; dg_last_error() gives a message.
 *    No exceptions, no aborts, nothing is printed.
 *  - There is no CPU fallback: without a CUDA device every compute call returns DG_ECUDA.
 */
#ifndef DG_H
#define DG_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define DG_OK       0
#define DG_EINVAL  (-1)   /* bad parameter, null or misaligned pointer */
#define DG_ENOSPC  (-2)   /* workspace too small */
#define DG_ESTATE  (-3)   /* state not set yet, or the call is not allowed between dg_step_begin and dg_step_end */
#define DG_ECUDA   (-4)   /* CUDA runtime / launch error (message in dg_last_error) */

typedef struct dg_ctx dg_ctx;     /* opaque, host-side, owned by the library */

typedef struct {
  int32_t nx, ny;                 /* cells K_ij = [x_{i-1/2},x_{i+1/2}] x [y_{j-1/2},y_{j+1/2}] */
  double  x0, x1, y0, y1;         /* domain; dx = (x1-x0)/nx, dy = (y1-y0)/ny */
  int32_t order;                  /* m = 1..5: m x m modes per cell and variable */
  int32_t rk;                     /* 2: SSP-RK(2,2), 3: SSP-RK(3,3) (Gottlieb & Shu 1998);
                                     4: the five-stage fourth-order SSP scheme of Table 1,
                                     5: the six-stage Cash-Karp scheme of Table 2, both printed in
                                     Butcher form (Appendix A) and evaluated on the stage states
                                     (coefficients solved from the printed tableau; with the limiter on, in a form that
                                     keeps the slopes of the limited states); see dg_rk_stages */
  int32_t bc;                     /* 0 periodic; 1 transmissive (exterior trace = interior);
                                     2 frozen: exterior trace = trace of the state given to the last
                                     dg_set_state*, same boundary cell, same face point */
  int32_t eos;                    /* 0 ideal gas p = (gamma-1) e, Eq.(2) PAPER.md:45-49;
                                     1 locally isothermal p = c_s^2(x,y) rho (BASELINE.json configs 1-4) */
  double  gamma;                  /* adiabatic index (eos 0) */
  double  h_aspect;               /* eos 1: c_s^2 = h^2 GM / sqrt(x^2 + y^2 + eps_star^2) */
  double  gm_star, eps_star;      /* star potential -GM/sqrt(r^2+eps^2); gm_star = 0: no gravity */
  double  q_planet, r_planet, eps_planet, omega_planet, phase0;
                                  /* planet of mass ratio q on the fixed circular orbit
                                     r_p (cos, sin)(omega_p t + phase0), softening eps_p;
                                     no indirect term; q = 0: no planet */
  double  damp_r0, damp_r1;       /* wave-killing zone r0 < r (<= r1 and beyond); r0 <= 0: off */
  double  t0;                     /* initial time */
  int32_t limiter;                /* 1: positivity-preserving limiter (Zhang & Shu 2010) after
                                     every RK sub-step (step (iii)(d)), and dg_cfl_dt uses the factor
                                     min(1/(2N_p+1), w_1/2) of PAPER.md:131; 0: off */
  double  lim_eps;                /* limiter floor for density and pressure (> 0 when limiter = 1; 1e-13) */
  int32_t flux;                   /* numerical flux h_{e,K} of Eq.(3) (PAPER.md:97 leaves its type open): 0 local
                                     Lax-Friedrichs (BASELINE cfg0); 1 HLLC (eos 0) / HLL (eos 1), Davis wave speeds */
  double  damp_in_r0, damp_in_r1; /* inner wave-killing zone of the paper's own disc: active for
                                     r < damp_in_r0 (= r_d), full strength for r <= damp_in_r1 (= r_in < r_d);
                                     damp_in_r0 <= 0: off */
  int32_t halo_south, halo_north; /* 1: this context is one strip of a domain decomposed along y (the paper's
                                     one-sub-domain-per-GPU design): the rows below y0 / above y1
                                     belong to a neighbour strip and are read from a halo row the caller fills before
                                     every sub-step (dg_halo_layout), instead of applying `bc` at that edge */
  int32_t damp_mode;              /* fields the wave-killing zones relax: 0 the conservative state
                                     (reading G13); 1 "the density, velocities and temperature"
                                     at the m x m Gauss points, conservative state rebuilt from them (reading D2) */
} dg_params;

/* Bytes of DEVICE workspace dg_init needs for these parameters (0 if they are invalid). */
size_t dg_workspace_bytes(const dg_params* params /*HOST*/);

/* Create a context.  workspace: DEVICE, 256-byte aligned, >= dg_workspace_bytes(params) bytes,
 * owned by the caller.  cuda_stream: cudaStream_t.  Builds the quadrature/basis tables
 * on the host.  Errors: DG_EINVAL, DG_ENOSPC. */
int dg_init(const dg_params* params /*HOST*/, void* workspace /*DEVICE*/, size_t workspace_bytes,
            void* cuda_stream, dg_ctx** out /*HOST*/);

/* Copy a modal state into the context (steps (i)(b)-(c) of PAPER.md:141-144 are the caller's).
 * U: [ny][nx][4][m][m] doubles.  Also snapshots it as the "initial" state used by bc 2 and by the
 * damping zones, and resets the time to t0.  _host variant: U is HOST memory (pinned memory makes
 * the copy asynchronous); the host->device copy is enqueued on the stream. */
int dg_set_state(dg_ctx*, const double* U /*DEVICE*/);
int dg_set_state_host(dg_ctx*, const double* U /*HOST*/);

/* Copy the current modal state out.  dg_get_state_host synchronises the stream before returning. */
int dg_get_state(dg_ctx*, double* U /*DEVICE*/);
int dg_get_state_host(dg_ctx*, double* U /*HOST*/);

/* L(u) at time t: right-hand side of the semi-discrete form Eq.(3) divided by the
 * diagonal mass: volume flux term + face term with the local Lax-Friedrichs
 * numerical flux + gravity source.  L: [ny][nx][4][m][m] DEVICE.  The state is not changed. */
int dg_rhs(dg_ctx*, double t, double* L /*DEVICE*/);

/* Global time step:
 *   dt = cfl/(2 N_p + 1) / max_K [ (|vx|+c)/dx + (|vy|+c)/dy ]   from the cell averages.
 * Synchronises the stream (the only blocking call of the time loop) and writes one HOST double. */
int dg_cfl_dt(dg_ctx*, double cfl, double* dt /*HOST*/);

/* One full time step of size dt (Algorithm 1, in Shu-Osher form): rk stages of
 * u^(s) = alpha_s u^n + beta_s (u^(s-1) + dt L(u^(s-1), t^n + c_s dt)), then the wave-killing
 * relaxation Q <- (dt Q0 + tau Q)/(tau + dt) if enabled; t += dt. */
int dg_step(dg_ctx*, double dt);

/* The same step, one sub-step at a time, for strips of a decomposed domain ("one layer of ghost
 * cells per side", exchanged after every sub-step): dg_step_begin(dt); then k = dg_rk_stages(rk) times
 * { fill the halo rows; dg_substep(); }; then dg_step_end().  dg_step is exactly this sequence. */
int dg_step_begin(dg_ctx*, double dt);
int dg_substep(dg_ctx*);
int dg_step_end(dg_ctx*);
/* A sub-step in two launches, so that the halo exchange overlaps the bulk of the strip: part 0 = the row segments
 * that touch no halo row (launch it while the exchange is in flight), part 1 = the first and last row segment
 * (after the halo rows have arrived), followed by the limiter pass when it is on.  dg_substep = part 0 + part 1.
 * Same arithmetic, same result bitwise.  DG_ESTATE if called out of order. */
int dg_substep_part(dg_ctx*, int part);
/* Between dg_step_begin and dg_step_end the workspace's spare state buffers hold live sub-step data: dg_rhs,
 * dg_get_state*, dg_limit, dg_cfl_dt, dg_torque*, dg_step and dg_step_debug return DG_ESTATE there (they use those
 * buffers as scratch, or would act on a state that is not a time level).  dg_set_state* abandons the split step. */

/* Where the halo exchange reads and writes, as byte offsets into the workspace given to dg_init (internal
 * layout, one row of cells = *row_bytes contiguous bytes): offsets[0], [1] = first and last row of the array
 * the next stage kernel reads (the next sub-step's input inside a split step, else the current state; the same
 * for dg_rhs): what the south / north neighbour needs; offsets[2], [3] = this context's south / north halo row
 * ((size_t)-1 if that edge is a domain boundary).  The caller copies neighbour rows into the halo rows on the
 * context's stream (cudaMemcpyAsync, NCCL send/recv, or a peer-to-peer copy over NVLink). */
int dg_halo_layout(dg_ctx*, size_t offsets[4] /*HOST*/, size_t* row_bytes /*HOST*/);

/* Same, and also writes the results of the k = dg_rk_stages(rk) sub-steps (after the limiter, before
 * damping; the last one is u^{n+1}), modal layout, stages: [k][ny][nx][4][m][m] DEVICE.  For per-stage
 * parity tests. */
int dg_step_debug(dg_ctx*, double dt, double* stages /*DEVICE*/);

/* Sub-steps (right-hand-side evaluations) per time step of scheme rk: 2, 3, 5 (rk 4), 6 (rk 5); -1 if unknown. */
int dg_rk_stages(int rk);

/* Apply the positivity-preserving limiter (Zhang & Shu 2010) to the current state, in
 * place, with floor lim_eps -- whether or not params.limiter is set (e.g. on a freshly projected initial
 * state).  Cell averages are unchanged.  Per cell K, with S_K = (Gauss_m x Lobatto_nh) U (Lobatto_nh x Gauss_m)
 * U (Gauss_m x Gauss_m, the volume quadrature points), nh the smallest Gauss-Lobatto rule exact for degree N_p:
 *   theta1 = min(1, (rho_bar - eps)/(rho_bar - min_S rho)) scales the density's non-constant part; then
 *   (eos 0) theta2 = min over the points of S_K with p < eps of the parameter t at which the segment
 *   u_bar + t (u(x) - u_bar) meets p = eps, and scales all four variables' non-constant parts. */
int dg_limit(dg_ctx*);

/* Specific torque on the planet at time t, Eq.(6) PAPER.md:321-328 (z component):
 *   Gamma = r_p x sum_n G M_n (r_n - r_p) / (|r_n - r_p|^2 + eps_p^2)^(3/2),
 * M_n = cell-average density x cell area, r_n = cell centre, G = gm_star (unit stellar mass).
 * Synchronises the stream and writes one HOST double. */
int dg_torque(dg_ctx*, double t, double* gamma_z /*HOST*/);

/* The torque as the paper quotes it: gamma Gamma / Gamma_0 with Gamma_0 = Sigma Omega^2 r_p^4 q / h^2,
 * Sigma = sigma_p (the unperturbed surface density at the planet's orbit: a property of the caller's initial data),
 * Omega = omega_planet, q = q_planet, h = h_aspect, gamma = the adiabatic index.  DG_EINVAL without a planet or
 * with h_aspect <= 0.  Synchronises the stream and writes one HOST double. */
int dg_torque_normalised(dg_ctx*, double t, double sigma_p, double* out /*HOST*/);

/* Convenience for end-to-end runs from HOST buffers: set_state_host(U_in), then nsteps times
 * { dg_cfl_dt(cfl); dg_step(dt) }, then get_state_host(U_out).  Blocking. */
int dg_run_host(dg_ctx*, const double* U_in /*HOST*/, int nsteps, double cfl, double* U_out /*HOST*/);

double dg_time(const dg_ctx*);
int    dg_set_time(dg_ctx*, double t);

/* Number of kernels this context has launched so far (for launch accounting in bench.py). */
long long dg_launch_count(const dg_ctx*);

/* Tuning knobs (all have defaults; DG_EINVAL on unknown key or bad value).
 *   DG_TUNE_ROWS_PER_CTA : rows of cells one thread block marches over in the stage kernel (default: 4..16,
 *                          chosen at dg_init: long segments re-read fewer neighbour rows, and the number of blocks
 *                          should come close to a multiple of what the GPU holds at once)
 *   DG_TUNE_FUSED_CFL    : 1 = the last RK stage also reduces the CFL wave speed (default), 0 = separate kernel */
#define DG_TUNE_ROWS_PER_CTA 1
#define DG_TUNE_FUSED_CFL    2
#define DG_TUNE_GEN_PREFETCH 3   /* general sub-steps: L2 prefetch of the earlier stage states: 0 none, 1 at the start of the row, 2 a row ahead, 3 between the x and y phases of the row (default) */
#define DG_TUNE_RK4_FORM     4   /* rk 4, limiter off: 1 = Table 1's scheme in its low-storage (Shu-Osher) form, from the
                                   printed tableau's row ratios (default); 0 = the generic state form */
#define DG_TUNE_STAGE_IMPL   5   /* which fused stage kernel runs: 0 = the default (orders 3 to 5: the kernel with the helper
                                   warp, dg_stage_fh.cuh, except for the sub-steps of the general schemes that gather earlier
                                   stage states; order 1: the register-only kernel, dg_stage_m1fv.cuh; order 2: M
                                   worker warps), 1 = M worker warps (dg::stage_kernel) at every order, 2 = like 0 but
                                   the helper-warp kernel for every sub-step of orders 3 to 5.  Same results to a few ulp. */
int dg_set_tuning(dg_ctx*, int key, int value);

/* Average-duration probe: enqueue CUDA events around the stage kernels of the next dg_step calls.
 * dg_stage_time_ms returns the mean stage-kernel time (ms) accumulated since the last reset and
 * the number of launches measured (synchronises). */
int dg_stage_timing(dg_ctx*, int enable);
int dg_stage_time_ms(dg_ctx*, double* mean_ms /*HOST*/, long long* launches /*HOST*/);
/* The individual durations (ms) of up to `capacity` measured stage launches, in launch order (synchronises). */
int dg_stage_times_ms(dg_ctx*, double* ms /*HOST, capacity doubles*/, long long capacity, long long* launches /*HOST*/);

/* Diagnostic: sustained fp64 FMA throughput of this GPU (register-resident DFMA loop),
 * TFLOP/s counting an FMA as 2 flops.  Uses the context's stream; blocking. */
int dg_probe_fp64_peak(dg_ctx*, double* tflops /*HOST*/);

const char* dg_last_error(const dg_ctx*);
void dg_destroy(dg_ctx*);

/* --- An entry point that allocates nothing, for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it): no context, no workspace, no host allocation either. ---
 *
 * dg_torque_static: the torque of Eq.(6), exactly as dg_torque defines it (M_n = cell-average
 * density x cell area, r_n = cell centre, planet at r_p (cos, sin)(omega_p t + phase0), softening eps_p), computed
 * straight from a modal state in the external layout (mode (0,0) = the cell average).
 *   params : HOST.  Read: nx, ny, x0, x1, y0, y1, order, gm_star, r_planet, eps_planet, omega_planet, phase0.
 *   U      : DEVICE, [ny][nx][4][m][m] doubles (m = order), the caller's; not changed.
 *   out    : DEVICE, 3 doubles, the caller's: out[0] = Gamma_z, out[1] = a_x, out[2] = a_y (Gamma_z = x_p a_y - y_p a_x).
 *   cuda_stream : cudaStream_t; two kernels are enqueued on it, nothing is synchronised, nothing is copied to the host.
 * The scratch of the reduction (per-block partial sums) is a file-scope __device__ array inside the library:
 * 2 x DG_STATIC_MAX_BLOCKS doubles = 1 MiB, held by every GPU that loads the library until the process exits.  A
 * thread block covers 32 x 32 cells, so grids with ceil(nx/32) x ceil(ny/32) <= DG_STATIC_MAX_BLOCKS are accepted (up to
 * 8192 x 8192 cells); larger ones return DG_ENOSPC (use dg_torque: its scratch is in the workspace).  Every call on a
 * device shares that array; it is never cleared and need not be (a call overwrites every slot it later reads), but
 * calls that overlap on the GPU -- different streams with no ordering between them -- race on it: order them.
 * The array's device address is looked up (cudaGetSymbolAddress) once per device, with that device current: on the first
 * dg_torque_static call there, or by dg_static_setup() -- call that before a stream capture begins.
 * Errors: DG_EINVAL (null / misaligned pointer, bad sizes), DG_ENOSPC, DG_ECUDA; message in dg_static_last_error()
 * (per host thread). */
#define DG_STATIC_MAX_BLOCKS 65536
int dg_static_setup(void);
int dg_torque_static(const dg_params* params /*HOST*/, const double* U /*DEVICE*/, double t,
                     double* out /*DEVICE, 3 doubles*/, void* cuda_stream);
const char* dg_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* DG_H */
