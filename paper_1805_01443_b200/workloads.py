"""Seeded synthetic workloads (inputs only) for the DG Euler hot path.

This module produces *data*: a parameter dict (the fields of ``dg_params`` in
``include/dg.h``) and the initial modal state ``U[ny][nx][4][m][m]`` (fp64,
index order ``[j][i][v][b][a]``, a = x-degree fastest).  Identical bytes are fed to
the CUDA path and to the CPU oracle.  It holds none of the solver's arithmetic: no
fluxes, no RHS, no time stepping.  The only numerical ingredient is the L2
projection of the initial data onto the Legendre modes (PAPER.md:141-144 steps
(i)(a)-(c)), done here with NumPy's library routines
(``numpy.polynomial.legendre.leggauss`` / ``legval``) so that neither solver's
table code is involved.

Workloads (they stand in for the paper's planet-disc runs,
PAPER.md:266-313, with the shapes BASELINE.json fixes):

* ``vortex``  -- isentropic vortex, beta = 5 (BASELINE cfg0).
* ``disc``    -- locally isothermal Keplerian disc, optional planet and seeded
                 multiplicative noise (BASELINE cfg1..cfg4).
* ``random_smooth`` -- seeded smooth positive random state for parity tests.
* ``gresho``  -- Gresho vortex.
* ``paper_disc`` -- the paper's own adiabatic planet-disc setup, PAPER.md:266-313 (NEXT-3).
"""
from __future__ import annotations

import math

import numpy as np
from numpy.polynomial import legendre as _npleg

NOISE_SEED = 180501443  # numpy.random.default_rng(180501443)

_PARAM_DEFAULTS = dict(
    nx=0, ny=0, x0=0.0, x1=1.0, y0=0.0, y1=1.0,
    order=1, rk=2, bc=0, eos=0, gamma=1.4, h_aspect=0.0,
    gm_star=0.0, eps_star=0.0,
    q_planet=0.0, r_planet=1.0, eps_planet=0.0, omega_planet=1.0, phase0=0.0,
    damp_r0=0.0, damp_r1=0.0, t0=0.0,
    limiter=0, lim_eps=1e-13, flux=0,
    damp_in_r0=0.0, damp_in_r1=0.0,
    halo_south=0, halo_north=0,
    damp_mode=0,
)


def make_params(**kw) -> dict:
    """Parameter dict with every ``dg_params`` field present."""
    p = dict(_PARAM_DEFAULTS)
    for k, v in kw.items():
        if k not in p:
            raise KeyError(k)
        p[k] = v
    return p


def _nodes_weights(m: int):
    x, w = _npleg.leggauss(m)
    return np.asarray(x, dtype=np.float64), np.asarray(w, dtype=np.float64)


def _phi(xi: np.ndarray, m: int) -> np.ndarray:
    """phi[q][a] = sqrt(2a+1) P_a(xi_q)  (SURVEY.md 8 notation)."""
    out = np.empty((xi.size, m))
    for a in range(m):
        c = np.zeros(a + 1)
        c[a] = 1.0
        out[:, a] = math.sqrt(2 * a + 1) * _npleg.legval(xi, c)
    return out


def node_coordinates(p: dict):
    """x[i][q], y[j][r]: physical coordinates of the m Gauss-Legendre nodes per cell."""
    m = p["order"]
    xi, _ = _nodes_weights(m)
    dx = (p["x1"] - p["x0"]) / p["nx"]
    dy = (p["y1"] - p["y0"]) / p["ny"]
    xc = p["x0"] + (np.arange(p["nx"]) + 0.5) * dx
    yc = p["y0"] + (np.arange(p["ny"]) + 0.5) * dy
    return xc[:, None] + 0.5 * dx * xi[None, :], yc[:, None] + 0.5 * dy * xi[None, :]


def project_nodal(p: dict, nodal: np.ndarray) -> np.ndarray:
    """L2-project nodal conservative values ``nodal[j][i][v][r][q]`` onto the modes.

    U[j][i][v][b][a] = 1/4 sum_{q,r} w_q w_r nodal[j][i][v][r][q] phi_a(xi_q) phi_b(xi_r)
    """
    m = p["order"]
    xi, w = _nodes_weights(m)
    P = _phi(xi, m) * (0.5 * w)[:, None]       # P[q][a]
    return np.einsum("jivrq,qa,rb->jivba", nodal, P, P, optimize=True).copy()


def evaluate_nodal(p: dict, U: np.ndarray) -> np.ndarray:
    """Inverse of :func:`project_nodal` on the polynomial space: nodal[j][i][v][r][q]."""
    m = p["order"]
    xi, _ = _nodes_weights(m)
    B = _phi(xi, m)
    return np.einsum("jivba,qa,rb->jivrq", U, B, B, optimize=True).copy()


def _conservative(rho, vx, vy, pr, gamma):
    E = pr / (gamma - 1.0) + 0.5 * rho * (vx * vx + vy * vy)
    return np.stack([rho, rho * vx, rho * vy, E], axis=2)  # [j][i][v][r][q]


def _mesh(p):
    xq, yr = node_coordinates(p)                 # [nx][m], [ny][m]
    X = xq[None, :, None, :]                     # [1][nx][1][m]
    Y = yr[:, None, :, None]                     # [ny][1][m][1]
    X, Y = np.broadcast_arrays(X, Y)
    return X, Y                                  # [ny][nx][r][q]


# ----------------------------------------------------------------------------------------------
def vortex(n: int = 32, order: int = 2, rk: int = 2, beta: float = 5.0, gamma: float = 1.4):
    """Isentropic vortex; BASELINE cfg0 (32^2, order 2, SSP-RK2, CFL 0.2)."""
    p = make_params(nx=n, ny=n, x0=0.0, x1=10.0, y0=0.0, y1=10.0, order=order, rk=rk,
                    bc=0, eos=0, gamma=gamma)
    X, Y = _mesh(p)
    prim = vortex_exact(X, Y, 0.0, beta, gamma)
    return p, project_nodal(p, _conservative(*prim, gamma))


def vortex_exact(X, Y, t, beta=5.0, gamma=1.4):
    """Exact primitive solution at time t: the initial vortex advected by (1,1), periodic on
    [0,10]^2."""
    xc = 5.0 + t
    yc = 5.0 + t
    dx = (X - xc + 5.0) % 10.0 - 5.0
    dy = (Y - yc + 5.0) % 10.0 - 5.0
    r2 = dx * dx + dy * dy
    rho = (1.0 - (gamma - 1.0) * beta ** 2 / (8.0 * gamma * math.pi ** 2) * np.exp(1.0 - r2)) \
        ** (1.0 / (gamma - 1.0))
    vx = 1.0 - beta / (2.0 * math.pi) * np.exp(0.5 * (1.0 - r2)) * dy
    vy = 1.0 + beta / (2.0 * math.pi) * np.exp(0.5 * (1.0 - r2)) * dx
    return rho, vx, vy, rho ** gamma


def entropy_wave(n: int = 16, order: int = 3, rk: int = 3, amp: float = 0.2):
    """Smooth exact solution of the Euler equations used to pin the convergence order without the
    vortex's periodic-image kink: a density wave rho = 1 + amp sin(2 pi (x + y - 2t)/10) carried by
    the uniform flow v = (1,1), p = 1, periodic on [0,10]^2 (a contact wave: v and p stay uniform)."""
    p = make_params(nx=n, ny=n, x0=0.0, x1=10.0, y0=0.0, y1=10.0, order=order, rk=rk,
                    bc=0, eos=0, gamma=1.4)
    X, Y = _mesh(p)
    rho = entropy_wave_exact(X, Y, 0.0, amp)
    one = np.ones_like(rho)
    return p, project_nodal(p, _conservative(rho, one, one, one, 1.4))


def entropy_wave_exact(X, Y, t, amp: float = 0.2):
    return 1.0 + amp * np.sin(2.0 * math.pi * (X + Y - 2.0 * t) / 10.0)


def gresho(n: int = 40, order: int = 3, rk: int = 3, gamma: float = 1.4):
    """Gresho vortex: steady rotating flow on [0,1]^2 centred at (0.5, 0.5), rho = 1,
    v_phi = 5r | 2-5r | 0 and the pressure that balances it, gradient-free boundaries (the
    transmissive bc 1).  Table 1 is quoted at 40 x 40 cells, T = 3.  gamma is not
    stated in the paper; 1.4 as in Liska & Wendroff (2003), whom the paper follows."""
    p = make_params(nx=n, ny=n, x0=0.0, x1=1.0, y0=0.0, y1=1.0, order=order, rk=rk, bc=1, eos=0, gamma=gamma)
    X, Y = _mesh(p)
    rho, vx, vy, pr = gresho_exact(X, Y)
    return p, project_nodal(p, _conservative(rho, vx, vy, pr, gamma))


def gresho_exact(X, Y):
    """Primitive fields of the (time-independent) Gresho vortex."""
    dx, dy = X - 0.5, Y - 0.5
    r = np.sqrt(dx * dx + dy * dy)
    rs = np.maximum(r, 1e-300)
    vphi = np.where(r < 0.2, 5.0 * r, np.where(r < 0.4, 2.0 - 5.0 * r, 0.0))
    pr = np.where(r < 0.2, 5.0 + 12.5 * r * r,
                  np.where(r < 0.4, 9.0 - 4.0 * math.log(0.2) + 12.5 * r * r - 20.0 * r + 4.0 * np.log(rs),
                           3.0 + 4.0 * math.log(2.0)))
    return np.ones_like(r), -vphi * dy / rs, vphi * dx / rs, pr


def l1_error_percent(p: dict, U: np.ndarray, exact_nodal: np.ndarray, v: int = 0) -> float:
    """Relative L1 error (%) of variable v by the quadrature of Eq.(5):
    100 * sum_K sum_ij |u_h - u| w_i w_j / sum_K sum_ij |u| w_i w_j  (the 1/4 dx dy cancels)."""
    m = p["order"]
    _, w = _nodes_weights(m)
    ww = w[:, None] * w[None, :]
    uh = evaluate_nodal(p, U)[:, :, v]
    return float(100.0 * (np.abs(uh - exact_nodal) * ww).sum() / (np.abs(exact_nodal) * ww).sum())


# ----------------------------------------------------------------------------------------------
def disc(n: int = 256, order: int = 3, planet: bool = False, noise: float = 0.0,
         eos: int = 1, rk: int = 3, damping: bool = True, half_width: float = 2.5,
         nx: int | None = None, ny: int | None = None,
         floor: float = 1e-2, taper: float = 0.1, eps_star: float = 0.2):
    """Keplerian disc of BASELINE cfg1..cfg4 (recipe: SURVEY.md 8(d)).

    With r_s = sqrt(r^2 + eps_*^2), T(r) = (1 + tanh((r - 0.4)/taper))/2:
      Sigma   = floor + (r_s^-1/2 - floor) T(r)           (Sigma ~ r^-1/2, hole of depth `floor` inside 0.4)
      c_s^2   = h^2 GM / r_s,   p = c_s^2 Sigma,  E = p/(gamma-1) + Sigma v^2 / 2
      Omega^2 = GM/r_s^3 + (1/(r Sigma)) d(c_s^2 Sigma)/dr    (exact rotational equilibrium of the
                softened potential with this pressure; equals GM(1-1.5h^2)/r_s^3
                where T = 1),   v = Omega (-y, x).
    ``eos=0`` gives the adiabatic variant (same initial data, ideal-gas closure).
    ``noise`` multiplies Sigma at each volume node by 1 + noise*(2u-1), u seeded (cfg2..cfg4: 1e-4).
    Defaults (floor 1e-2, taper 0.1, star softening 0.2) are the values with which the disc stays
    positive and finite, without a limiter, for every BASELINE config's step count (checked with the
    oracle: 256^2 x 200, 512^2 x 500 steps at order 3, 64^2 x 120 at order 5).  BASELINE.json's literal
    numbers (floor 1e-6, softening 0.02: ``LITERAL_BASELINE_DISC``) go negative at the unresolved
    potential well / hole within ~20-170 steps on every grid tried, because the positivity limiter
    is not on the hot path; see DESIGN.md "Input recipe".  Kernel work is
    independent of the values, so throughput is unaffected by this choice.
    """
    nx = n if nx is None else nx
    ny = n if ny is None else ny
    h, gm, gamma = 0.05, 1.0, 1.4
    p = make_params(nx=nx, ny=ny, x0=-half_width, x1=half_width, y0=-half_width, y1=half_width,
                    order=order, rk=rk, bc=2, eos=eos, gamma=gamma, h_aspect=h,
                    gm_star=gm, eps_star=eps_star,
                    q_planet=1e-5 if planet else 0.0, r_planet=1.0, eps_planet=0.6 * h,
                    omega_planet=1.0, phase0=0.0,
                    damp_r0=2.2 if damping else 0.0, damp_r1=2.5 if damping else 0.0)
    X, Y = _mesh(p)
    r2 = X * X + Y * Y
    r = np.sqrt(r2)
    rs2 = r2 + eps_star * eps_star
    rs = np.sqrt(rs2)
    a = (r - 0.4) / taper
    T = 0.5 * (1.0 + np.tanh(a))
    base = rs ** -0.5
    sigma = floor + (base - floor) * T
    # (dSigma/dr)/r, an even function of r (finite at the origin)
    dT_r = 0.5 / np.cosh(a) ** 2 / taper / np.maximum(r, 1e-300)
    dsigma_r = -0.5 * rs ** -2.5 * T + (base - floor) * dT_r
    cs2 = h * h * gm / rs
    om2 = gm / rs ** 3 - cs2 / rs2 + cs2 * dsigma_r / sigma
    if om2.min() <= 0.0:
        raise ValueError("disc recipe: pressure gradient exceeds gravity; no rotational equilibrium")
    om = np.sqrt(om2)
    if noise != 0.0:
        u = np.random.default_rng(NOISE_SEED).random((ny, nx, order, order))
        sigma = sigma * (1.0 + noise * (2.0 * u - 1.0))
    return p, project_nodal(p, _conservative(sigma, -om * Y, om * X, cs2 * sigma, gamma))


def paper_disc(n: int = 256, order: int = 3, rk: int = 2, planet: bool = True, limiter: bool = True,
               eps_star: float = 0.2, half_width: float = 2.25):
    """The paper's own planet-disc setup: adiabatic disc
    (gamma = 1.4), box [-2.25, 2.25]^2, Sigma = Sigma0/(1+f), p = p0/(1+f), f = exp((r - r_ex)/(r_p h)),
    Sigma0 = 1, p0 = 2.5e-3, r_in = 0.4, r_ex = 1.75, h = 0.05; planet q = 6e-5 at r_p = 1, eps_p = 0.03;
    v_phi^2 = r^2 Omega^2 - r c_iso^2 f / (r_p h (1+f)) with c_iso^2 = p0/Sigma0 (reading G12) and
    Omega^2 = GM/r_in^3 inside r_in, GM/r^3 outside (reading G11: solid rotation inside);
    wave-killing zones r_d = r_in 1.15^(3/2) -> r_in and r_d = r_ex 1.15^(-3/2) -> r_ex relaxing "the density,
    velocities and temperature" (damp_mode 1); frozen box edge
    (G14).  The density falls to ~4e-13 in the box corners: the positivity limiter is on by default.
    The paper does not soften the star's potential; with eps_star = 0 the four cells around the origin blow up within
    one step on a Cartesian grid, so the default is the BASELINE disc's 0.2 (inside the damped hole r < r_in)."""
    h, gm, gamma = 0.05, 1.0, 1.4
    r_in, r_ex, sigma0, p0 = 0.4, 1.75, 1.0, 2.5e-3
    p = make_params(nx=n, ny=n, x0=-half_width, x1=half_width, y0=-half_width, y1=half_width,
                    order=order, rk=rk, bc=2, eos=0, gamma=gamma, h_aspect=h, gm_star=gm, eps_star=eps_star,
                    q_planet=6.0e-5 if planet else 0.0, r_planet=1.0, eps_planet=0.03, omega_planet=1.0,
                    phase0=0.0, damp_r0=r_ex * 1.15 ** -1.5, damp_r1=r_ex,
                    damp_in_r0=r_in * 1.15 ** 1.5, damp_in_r1=r_in, damp_mode=1,
                    limiter=1 if limiter else 0, lim_eps=1e-13)
    X, Y = _mesh(p)
    r = np.sqrt(X * X + Y * Y)
    f = np.exp((r - r_ex) / h)
    sigma = sigma0 / (1.0 + f)
    pr = p0 / (1.0 + f)
    om2 = np.where(r <= r_in, gm / r_in ** 3, gm / np.maximum(r, 1e-300) ** 3)
    vphi2 = r * r * om2 - r * (p0 / sigma0) * f / (h * (1.0 + f))
    om = np.sqrt(np.maximum(vphi2, 0.0)) / np.maximum(r, 1e-300)
    return p, project_nodal(p, _conservative(sigma, -om * Y, om * X, pr, gamma))


LITERAL_BASELINE_DISC = dict(floor=1e-6, taper=0.05, eps_star=0.02)   # BASELINE.json's numbers (need a limiter)


# ----------------------------------------------------------------------------------------------
def random_smooth(nx: int, ny: int, order: int, seed: int = 0, eos: int = 0, bc: int = 0,
                  rk: int = 3, gravity: bool = False, amp: float = 0.2, **extra):
    """Seeded, smooth, strictly positive random state on [0,1]x[0,1] (or a box around the origin
    when ``gravity``): a few random Fourier modes in each primitive variable, plus independent
    per-cell high-mode jitter so that every modal coefficient and every interface jump is exercised.
    """
    rng = np.random.default_rng(seed)
    if gravity:
        kw = dict(x0=-1.3, x1=1.1, y0=-0.9, y1=1.4, gm_star=1.0, eps_star=0.05, h_aspect=0.07,
                  q_planet=2e-3, r_planet=0.8, eps_planet=0.04, omega_planet=1.3, phase0=0.4)
    else:
        kw = dict(x0=0.0, x1=1.0, y0=0.0, y1=1.5)
    kw.update(extra)
    p = make_params(nx=nx, ny=ny, order=order, rk=rk, bc=bc, eos=eos, gamma=1.4, **kw)
    X, Y = _mesh(p)
    Lx, Ly = p["x1"] - p["x0"], p["y1"] - p["y0"]

    def field(mean):
        f = np.full(X.shape, mean)
        for _ in range(3):
            kx, ky = rng.integers(1, 4, size=2)
            ph = rng.uniform(0, 2 * math.pi, size=2)
            f = f + amp * mean * rng.uniform(0.3, 1.0) / 3.0 * \
                np.sin(2 * math.pi * kx * (X - p["x0"]) / Lx + ph[0]) * \
                np.cos(2 * math.pi * ky * (Y - p["y0"]) / Ly + ph[1])
        return f

    rho = field(1.0)
    pr = field(0.8)
    vx = field(1.0) - 0.7
    vy = field(1.0) - 1.2
    U = project_nodal(p, _conservative(rho, vx, vy, pr, p["gamma"]))
    # per-cell jitter on all non-mean modes (keeps cell means, creates interface jumps)
    jit = rng.standard_normal(U.shape) * 0.01 * amp
    jit[..., 0, 0] = 0.0
    scale = np.array([1.0, 0.5, 0.5, 2.0])[None, None, :, None, None]
    return p, (U + jit * scale).copy()


def dof_count(p: dict) -> int:
    """Degrees of freedom as the paper counts them: nx*ny*m^2, variables not counted."""
    return p["nx"] * p["ny"] * p["order"] ** 2
