"""Pins added in round 2 for the oracle parts a line-by-line mutation of oracle/ref_dg.cpp showed unpinned
("What's weak" 1-6).  Each test names the mutation it turns red; tests/golden/README.md lists them.
None re-types the oracle: traces and quadratures come from numpy.polynomial.legendre, point-wise fluxes from the
(separately pinned) oracle.llf / oracle.point_flux, expected limiter factors from node values evaluated by NumPy,
the HLLC star state from the Rankine-Hugoniot conditions."""
import math

import numpy as np
import pytest
from numpy.polynomial import legendre as npleg

import oracle
from paper_1805_01443_b200 import workloads as W

GAMMA = 1.4


def _phi(x, a):
    c = np.zeros(a + 1)
    c[a] = math.sqrt(2 * a + 1)
    return npleg.legval(np.asarray(x, dtype=float), c)


def _trace(Uc, side, axis, pts):
    """Values [v][len(pts)] of the cell polynomial Uc[v][b][a] on the face xi = side (axis 0) or eta = side
    (axis 1) at the reference points pts along the face -- NumPy's Legendre evaluation."""
    m = Uc.shape[-1]
    Pe = np.array([_phi(np.array([float(side)]), a)[0] for a in range(m)])
    Pt = np.array([_phi(pts, a) for a in range(m)])                       # [a][pt]
    if axis == 0:
        return np.einsum("vba,a,bp->vp", Uc, Pe, Pt)
    return np.einsum("vba,ap,b->vp", Uc, Pt, Pe)


def _face_term_of_cell(p, U, U0, i, j, flux):
    """-(1/2dx) sum_r w_r [H_E phi_a(1) - H_W phi_a(-1)] phi_b(eta_r) - (1/2dy) sum_q w_q [H_N phi_b(1) - H_S phi_b(-1)] phi_a(xi_q)
    of cell (i,j) (Eq.(3)'s face sum over the m Gauss points of each face, divided by the mass), bc 2: the exterior
    state at a box edge is the trace of the INITIAL state U0 of the same cell on the same face."""
    m, nx, ny = p["order"], p["nx"], p["ny"]
    dx, dy = (p["x1"] - p["x0"]) / nx, (p["y1"] - p["y0"]) / ny
    xg, wg = npleg.leggauss(m)
    xc, yc = p["x0"] + (i + 0.5) * dx, p["y0"] + (j + 0.5) * dy
    out = np.zeros((4, m, m))
    own = U[j, i]
    for side in (-1, +1):
        # x-faces
        xf = xc + side * 0.5 * dx
        inner = _trace(own, side, 0, xg)
        ii = i + side
        if 0 <= ii < nx:
            outer = _trace(U[j, ii], -side, 0, xg)
        else:
            outer = _trace(U0[j, i], side, 0, xg)
        for r in range(m):
            UL, UR = (inner[:, r], outer[:, r]) if side > 0 else (outer[:, r], inner[:, r])
            H = flux(p, UL, UR, xf, yc + 0.5 * dy * xg[r], 0)
            for a in range(m):
                for b in range(m):
                    out[:, b, a] -= side * wg[r] * H * _phi([side], a)[0] * _phi([xg[r]], b)[0] / (2 * dx)
        # y-faces
        yf = yc + side * 0.5 * dy
        inner = _trace(own, side, 1, xg)
        jj = j + side
        if 0 <= jj < ny:
            outer = _trace(U[jj, i], -side, 1, xg)
        else:
            outer = _trace(U0[j, i], side, 1, xg)
        for q in range(m):
            UL, UR = (inner[:, q], outer[:, q]) if side > 0 else (outer[:, q], inner[:, q])
            H = flux(p, UL, UR, xc + 0.5 * dx * xg[q], yf, 1)
            for a in range(m):
                for b in range(m):
                    out[:, b, a] -= side * wg[q] * H * _phi([side], b)[0] * _phi([xg[q]], a)[0] / (2 * dy)
    return out


# ------------------------------------------------------------------------------------------------
# C9: frozen boundary, m > 1.  Mutation caught: the side of the U0 trace at any of the four box edges
# (ref_dg.cpp, compute_rhs: trace_x(c, U0, 0, j, -1) / (nx-1, +1), trace_y(c, U0, i, 0, -1) / (ny-1, +1)).
@pytest.mark.parametrize("eos", [0, 1])
@pytest.mark.parametrize("m", [2, 3, 4, 5])
def test_frozen_boundary_equals_transmissive_before_the_state_moves(m, eos):
    """Straight after set_state the frozen exterior trace IS the interior trace at every boundary face point
    (same cell, same face, U0 = U), so L with bc 2 equals L with bc 1 (bc 1 is pinned by the 24-point brute
    force).  A U0 trace taken on the wrong side of the cell differs from the interior trace as soon as m > 1."""
    p, U = W.random_smooth(5, 4, m, seed=40 + m, eos=eos, bc=2, gravity=bool(eos), amp=0.3)
    r2 = oracle.RefDG(p)
    r2.set_state(U)
    r1 = oracle.RefDG(dict(p, bc=1))
    r1.set_state(U)
    L2, L1 = r2.rhs(0.1), r1.rhs(0.1)
    assert np.abs(L1).max() > 1.0
    np.testing.assert_allclose(L2, L1, rtol=0, atol=1e-14 * np.abs(L1).max())


@pytest.mark.parametrize("eos", [0, 1])
@pytest.mark.parametrize("m", [2, 4])
def test_frozen_boundary_trace_after_the_state_has_moved(m, eos):
    """After a step U != U0: the face term of the boundary cells (one per box edge and the corners) against
    point-wise oracle.llf(trace of U, trace of U0 on the same face of the same cell) with NumPy traces."""
    nx, ny = 4, 3
    p, U0 = W.random_smooth(nx, ny, m, seed=50 + m, eos=eos, bc=2, gravity=bool(eos), amp=0.3, rk=2)
    r = oracle.RefDG(p)
    r.set_state(U0)
    for _ in range(3):
        r.step(2.0 * r.cfl_dt(0.2))
    U = r.get_state()
    assert np.abs(U - U0).max() > 1e-3
    L = r.rhs(0.0, parts=2)
    for (i, j) in [(0, 1), (nx - 1, 1), (1, 0), (2, ny - 1), (0, 0), (nx - 1, ny - 1)]:
        ref = _face_term_of_cell(p, U, U0, i, j, oracle.llf)
        np.testing.assert_allclose(L[j, i], ref, rtol=0, atol=5e-13 * max(1.0, np.abs(ref).max()))
    # the test has teeth: taking U0's trace on the opposite face changes the expected value visibly
    wrong = _face_term_of_cell(p, U, U0[:, ::-1].copy(), 0, 1, oracle.llf)
    assert np.abs(wrong - L[1, 0]).max() > 1e-4


# ------------------------------------------------------------------------------------------------
# C4 at face nodes, eos 1.  Mutation caught: the face node's y (x) replaced by the cell centre's in the
# x-face (y-face) loop of compute_rhs -- it only feeds c_s^2 inside the numerical flux.
@pytest.mark.parametrize("m", [2, 3, 5])
def test_isothermal_sound_speed_is_taken_at_the_face_nodes(m):
    """Cell-wise constant states on a box close to the star, where c_s^2 = h^2 GM / sqrt(r^2 + eps^2) changes by
    tens of per cent along one face: the numerical flux then varies along a face only through c_s at the face
    node, and the face term is the m-point Gauss quadrature of oracle.llf(UL, UR, x_f, y_r) against phi_b."""
    nx, ny = 3, 3
    p = W.make_params(nx=nx, ny=ny, order=m, x0=0.05, x1=0.65, y0=-0.3, y1=0.45, eos=1, gamma=GAMMA, bc=0,
                      h_aspect=0.4, gm_star=1.0, eps_star=0.02)
    rng = np.random.default_rng(60 + m)
    U = np.zeros((ny, nx, 4, m, m))
    U[..., 0, 0, 0] = rng.uniform(0.8, 1.5, (ny, nx))
    U[..., 1, 0, 0] = rng.normal(size=(ny, nx)) * 0.3
    U[..., 2, 0, 0] = rng.normal(size=(ny, nx)) * 0.3
    U[..., 3, 0, 0] = rng.uniform(2.5, 3.5, (ny, nx))
    r = oracle.RefDG(p)
    r.set_state(U)
    L = r.rhs(0.0, parts=2)
    Uper = np.pad(U, ((1, 1), (1, 1), (0, 0), (0, 0), (0, 0)), mode="wrap")
    # periodic neighbours through a padded copy: reuse the bc-2 helper on the padded array's interior cell
    pp = dict(p, nx=nx + 2, ny=ny + 2, x0=p["x0"] - 0.2, x1=p["x1"] + 0.2, y0=p["y0"] - 0.25, y1=p["y1"] + 0.25)
    for (i, j) in [(0, 0), (1, 1), (2, 0), (0, 2)]:
        ref = _face_term_of_cell(pp, Uper, Uper, i + 1, j + 1, oracle.llf)
        np.testing.assert_allclose(L[j, i], ref, rtol=0, atol=2e-13 * max(1.0, np.abs(ref).max()))
        if m > 1:
            assert np.abs(ref[:, 1:, 0]).max() > 1e-3 and np.abs(ref[:, 0, 1:]).max() > 1e-3   # c_s varies along faces


# ------------------------------------------------------------------------------------------------
# C12, reading L2: the m x m volume Gauss points belong to the limiter's point set.
# Mutation caught: removing the volume-point loop of limiter_points().
def _gauss_lagrange_cell(m, node_values):
    """Modal coefficients [b][a] of the polynomial with the given values [r][q] at the tensor Gauss points."""
    xg, wg = npleg.leggauss(m)
    P = np.array([_phi(xg, a) for a in range(m)]) * (0.5 * wg)[None, :]   # [a][q]
    return np.einsum("rq,aq,br->ba", node_values, P, P)


def _values(cu, xs, ys):
    m = cu.shape[-1]
    Px = np.array([_phi(xs, a) for a in range(m)])
    Py = np.array([_phi(ys, b) for b in range(m)])
    return np.einsum("ba,ax,by->yx", cu, Px, Py)


def test_limiter_acts_on_a_cell_whose_only_bad_point_is_a_volume_gauss_node():
    """m = 3: rho = 1 - c g(x) g(y), g(s) = 1 - 0.3 (s - x_G)^2 peaked at the last Gauss node x_G = sqrt(0.6).
    Every point of Zhang & Shu's set (Gauss x Lobatto and Lobatto x Gauss) keeps rho >= 0.004, the corner Gauss
    node (x_G, x_G) has rho = -0.0101: theta_1 = (rhobar - eps)/(rhobar - rho(x_G, x_G)) with the node value
    from NumPy, and the limited density at that node equals eps."""
    m, eps = 3, 1e-9
    xg, _ = npleg.leggauss(m)
    xh, _ = oracle.lobatto(m)
    g = lambda s: 1.0 - 0.3 * (s - xg[-1]) ** 2
    c = 1.0 / 0.99
    nodal = 1.0 - c * g(xg)[:, None] * g(xg)[None, :]                      # [r][q]
    u = np.zeros((4, m, m))
    u[0] = _gauss_lagrange_cell(m, nodal)
    u[3, 0, 0] = 10.0                                                      # pressure comfortably positive
    zs = np.concatenate([_values(u[0], xg, xh).ravel(), _values(u[0], xh, xg).ravel()])
    vol = _values(u[0], xg, xg)
    assert zs.min() > 3e-3                                                 # admissible on Zhang & Shu's own set
    assert vol[-1, -1] < -0.01 and np.sort(vol.ravel())[1] > 0             # exactly one bad volume node
    p = W.make_params(nx=1, ny=1, order=m, eos=0, gamma=GAMMA, limiter=1, lim_eps=eps)
    lim, th1, th2 = oracle.limit_cell(p, u)
    rbar = u[0, 0, 0]
    assert abs(th1 - (rbar - eps) / (rbar - vol[-1, -1])) < 1e-14 and th2 == 1.0
    assert abs(_values(lim[0], xg, xg)[-1, -1] - eps) < 1e-15


# ------------------------------------------------------------------------------------------------
# C12: eps = min(lim_eps, rhobar) (Zhang & Shu 2010: eps = min(1e-13, rhobar, pbar)).
# Mutation caught: eps_rho = lim_eps.
def test_limiter_floor_is_capped_by_the_cell_average():
    """rhobar = 1e-3 < lim_eps = 1e-2 with a negative point: eps_rho = rhobar, theta_1 = 0 exactly -- the cell
    becomes the constant rhobar.  With eps_rho = lim_eps the factor would be (1e-3 - 1e-2)/(...) < 0."""
    m = 2
    p = W.make_params(nx=1, ny=1, order=m, eos=1, h_aspect=0.05, gm_star=1.0, eps_star=0.1, limiter=1, lim_eps=1e-2)
    u = np.zeros((4, m, m))
    u[0, 0, 0] = 1e-3
    u[0, 0, 1] = 2e-3                                                      # rho(-1) = 1e-3 - 2e-3 sqrt 3 < 0
    u[0, 1, 1] = 1e-4
    lim, th1, th2 = oracle.limit_cell(p, u)
    assert th1 == 0.0 and th2 == 1.0
    assert lim[0, 0, 0] == 1e-3 and np.abs(lim[0].ravel()[1:]).max() == 0.0
    # and with an average above the floor the floor itself is used: theta = (rhobar - eps)/(rhobar - rho_min)
    u[0, 0, 0] = 1.0
    u[0, 0, 1] = 0.9
    u[0, 1, 1] = 0.0
    lim, th1, _ = oracle.limit_cell(p, u)
    assert abs(th1 - (1.0 - 1e-2) / (0.9 * math.sqrt(3.0))) < 1e-15


def test_limiter_pressure_floor_is_capped_by_the_cell_average():
    """Ideal gas, eps_p = min(lim_eps, pbar) (Zhang & Shu 2010: eps = min(1e-13, rhobar, pbar)).  A cell at rest with
    the uniform pressure p0 = 1e-3 < lim_eps = 1e-2 and a linear, positive density: every point has p = p0 = pbar, so
    no point is below the floor min(lim_eps, pbar) = pbar and the cell is left alone (theta_2 = 1, coefficients
    bitwise).  With eps_p = lim_eps every point counts as inadmissible and the segment to the average never reaches
    p = lim_eps: theta_2 = 0, the density slope would be wiped out.  Mutation caught: eps_p = lim_eps."""
    m = 2
    gamma = 1.4
    p = W.make_params(nx=1, ny=1, order=m, eos=0, gamma=gamma, limiter=1, lim_eps=1e-2)
    u = np.zeros((4, m, m))
    u[0, 0, 0] = 1.0
    u[0, 0, 1] = 0.3                                                       # rho = 1 + 0.3 sqrt(3) xi > 0.48
    u[0, 1, 0] = -0.2
    u[3, 0, 0] = 1e-3 / (gamma - 1.0)                                      # E = p0/(gamma-1), no momentum
    lim, th1, th2 = oracle.limit_cell(p, u)
    assert th1 == 1.0 and th2 == 1.0
    assert np.array_equal(lim, u)
    # with the average pressure above the floor a point below it is pulled to p = lim_eps exactly (linear E, rho = 1:
    # p is linear along the segment, t = (pbar - eps)/(pbar - p_point))
    u = np.zeros((4, m, m))
    u[0, 0, 0] = 1.0
    u[3, 0, 0] = 1.0 / (gamma - 1.0)                                       # pbar = 1
    u[3, 0, 1] = 0.7 / (gamma - 1.0)                                       # p(xi) = 1 + 0.7 sqrt(3) xi: p(-1) = -0.212
    lim, th1, th2 = oracle.limit_cell(p, u)
    assert th1 == 1.0
    assert abs(th2 - (1.0 - 1e-2) / (0.7 * math.sqrt(3.0))) < 1e-14


# ------------------------------------------------------------------------------------------------
# C8b + C12: the limiter inside the Butcher-form sub-steps.  Mutation caught: deleting post() in butcher_step.
def _limiter_points_min_rho(m, cell):
    xg = npleg.leggauss(m)[0]
    xh, _ = oracle.lobatto(m)
    return min(_values(cell[0], xg, xh).min(), _values(cell[0], xh, xg).min(), _values(cell[0], xg, xg).min())


@pytest.mark.parametrize("rk", [4, 5])
def test_limiter_is_applied_after_every_butcher_substep(rk):
    """rk 4 (Table 1) and rk 5 (Cash-Karp): from a state the limiter has just made admissible, a step four times the
    CFL step drives INTERMEDIATE sub-step results of the unlimited scheme negative at the limiter's points; with the
    limiter on, every sub-step result y_2..y_s, u^{n+1} is admissible there (step (iii)(d)), and mass
    is conserved to round-off (periodic, no gravity)."""
    m, eps = 3, 1e-10
    p, U = W.random_smooth(6, 5, m, seed=3, bc=0, rk=rk)
    U[2, 3, 0, 0, 1] = 0.9                                 # rho dips below zero at the cell's west edge
    r = oracle.RefDG(dict(p, limiter=1, lim_eps=eps))
    r.set_state(U)
    r.limit()
    U1 = r.get_state()
    r0 = oracle.RefDG(p)
    r0.set_state(U1)
    dt = 4.0 * r0.cfl_dt(0.2)
    worst = lambda S: [min(_limiter_points_min_rho(m, S[s, j, i]) for j in range(5) for i in range(6))
                       for s in range(S.shape[0])]
    w0 = worst(r0.step_debug(dt))
    assert min(w0[:-1]) < -0.1, w0                          # the unlimited scheme needs it inside the step
    r.set_state(U1)
    st = r.step_debug(dt)
    w1 = worst(st)
    assert min(w1) >= eps * (1 - 1e-6), w1
    np.testing.assert_allclose(st[-1][..., 0, 0].sum(axis=(0, 1)), U[..., 0, 0].sum(axis=(0, 1)), rtol=1e-14)


# ------------------------------------------------------------------------------------------------
# C5b: HLL's jump term and HLLC's star energy.
def _davis(p, UL, UR, d, x=1.0, y=0.0):
    _, vL, cL = oracle.point_flux(p, UL, x, y, d)
    _, vR, cR = oracle.point_flux(p, UR, x, y, d)
    return min(vL - cL, vR - cR), max(vL + cL, vR + cR)


def test_hll_hand_worked_pair_and_sign_of_the_jump_term():
    """Isothermal closure with c_s = 1 at (1, 0) (h = 1, GM = 1, eps = 0): UL = (1, 0, 0, 1), UR = (2, 0, 0, 1) at
    rest: S_L = -1, S_R = 1, F_L = (0, 1, 0, 0), F_R = (0, 2, 0, 0), H = (F_L + F_R - (U_R - U_L))/2 = (-1/2, 3/2, 0, 0):
    mass flows from the dense side.  Mutation caught: the sign of S_L S_R (U_R - U_L)."""
    p = W.make_params(nx=1, ny=1, order=1, eos=1, h_aspect=1.0, gm_star=1.0, eps_star=0.0, flux=1)
    H = oracle.hllc(p, [1.0, 0, 0, 1.0], [2.0, 0, 0, 1.0], 1.0, 0.0, 0)
    np.testing.assert_allclose(H, [-0.5, 1.5, 0.0, 0.0], rtol=0, atol=1e-15)
    rng = np.random.default_rng(7)
    for d in (0, 1):
        for _ in range(30):
            UL = np.array([1.0, 0.1, -0.1, 2.0]) + 0.3 * rng.uniform(-1, 1, 4)
            UR = np.array([1.4, -0.1, 0.2, 2.0]) + 0.3 * rng.uniform(-1, 1, 4)
            SL, SR = _davis(p, UL, UR, d)
            assert SL < 0 < SR
            FL, FR = oracle.point_flux(p, UL, 1.0, 0.0, d)[0], oracle.point_flux(p, UR, 1.0, 0.0, d)[0]
            D = oracle.hllc(p, UL, UR, 1.0, 0.0, d) - (SR * FL - SL * FR) / (SR - SL)
            # the dissipative part opposes the jump, component by component
            np.testing.assert_allclose(D, SL * SR / (SR - SL) * (UR - UL), rtol=1e-12, atol=1e-14)
            assert (D * (UR - UL) <= 1e-15).all()


@pytest.mark.parametrize("d", [0, 1])
def test_hllc_star_flux_satisfies_rankine_hugoniot(d):
    """Subsonic pairs with S* != v_K.  Across the outer wave S_K: F* - F_K = S_K (U* - U_K) gives rho* and E*
    from the mass and energy components of H; S* = H_mass/rho*, p* = H_n - rho* S*^2; the star flux must be the
    flux of a state moving at S* under the pressure p*: H_E = S* (E* + p*), H_t = rho* S* v_t.
    Mutations caught: the signs inside the star energy (S* - v_K)(S* + p_K/(rho_K (S_K - v_K)))."""
    p = W.make_params(nx=1, ny=1, order=1, eos=0, gamma=GAMMA, flux=1)
    rng = np.random.default_rng(11 + d)
    n, tg = 1 + d, 2 - d
    seen = {True: 0, False: 0}
    for _ in range(60):
        UL = np.array([1.0, 0.0, 0.0, 2.5]) + rng.uniform(-1, 1, 4) * [0.3, 0.5, 0.5, 0.5]
        UR = np.array([1.3, 0.0, 0.0, 2.0]) + rng.uniform(-1, 1, 4) * [0.3, 0.5, 0.5, 0.5]
        SL, SR = _davis(p, UL, UR, d)
        if not SL < 0 < SR:
            continue
        H = oracle.hllc(p, UL, UR, 0.0, 0.0, d)
        # which side's star state the flux is: try the left one, fall back to the right one
        for (UK, SK) in ((UL, SL), (UR, SR)):
            FK, vK, _ = oracle.point_flux(p, UK, 0.0, 0.0, d)
            rho_s = UK[0] + (H[0] - FK[0]) / SK
            S_s = H[0] / rho_s
            left = UK is UL
            if (left and S_s >= 0) or (not left and S_s <= 0):
                break
        assert abs(S_s - vK) > 1e-3
        seen[left] += 1
        E_s = UK[3] + (H[3] - FK[3]) / SK
        p_s = H[n] - rho_s * S_s ** 2
        assert p_s > 0 and rho_s > 0
        assert abs(H[3] - S_s * (E_s + p_s)) < 1e-12 * max(1.0, abs(H[3]))
        assert abs(H[tg] - rho_s * S_s * UK[tg] / UK[0]) < 1e-13
        # the same star pressure seen from the other side's jump conditions (the contact carries no pressure jump)
        UO, SO = (UR, SR) if left else (UL, SL)
        FO, vO, _ = oracle.point_flux(p, UO, 0.0, 0.0, d)
        pO = (GAMMA - 1) * (UO[3] - 0.5 * (UO[1] ** 2 + UO[2] ** 2) / UO[0])
        assert abs(p_s - (pO + UO[0] * (SO - vO) * (S_s - vO))) < 1e-12
    assert seen[True] > 5 and seen[False] > 5


# ------------------------------------------------------------------------------------------------
# C11, damp_mode 1 ("The dampened fields are the density, velocities and temperature"; reading D2).
# Mutations caught: relaxing the momentum instead of the velocity, the energy (p) instead of the temperature.
def _prim_nodal(p, U):
    n = W.evaluate_nodal(p, U)                              # NumPy's Legendre evaluation at the Gauss points
    rho, mx, my, E = n[:, :, 0], n[:, :, 1], n[:, :, 2], n[:, :, 3]
    T = (p["gamma"] - 1) * (E - 0.5 * (mx * mx + my * my) / rho) / rho
    return rho, mx / rho, my / rho, T


def _zone_factors(p, dt):
    n = p["nx"]
    xc = p["x0"] + (np.arange(n) + 0.5) * (p["x1"] - p["x0"]) / n
    yc = p["y0"] + (np.arange(p["ny"]) + 0.5) * (p["y1"] - p["y0"]) / p["ny"]
    rr = np.hypot(xc[None, :], yc[:, None])
    ft = np.ones_like(rr)
    out, inn = rr > p["damp_r0"], rr < p["damp_in_r0"]
    R = np.minimum(1.0, ((rr - p["damp_r0"]) / (p["damp_r1"] - p["damp_r0"])) ** 2)
    tau = 2 * math.pi * math.sqrt(p["damp_r0"] ** 3 / p["gm_star"]) / np.where(out, R, 1.0)
    ft = np.where(out, tau / (tau + dt), ft)
    if p["damp_in_r0"] > 0:
        R = np.minimum(1.0, ((p["damp_in_r0"] - rr) / (p["damp_in_r0"] - p["damp_in_r1"])) ** 2)
        tau = 2 * math.pi * math.sqrt(p["damp_in_r0"] ** 3 / p["gm_star"]) / np.where(inn, R, 1.0)
        ft = np.where(inn, tau / (tau + dt), ft)
    return ft


@pytest.mark.parametrize("m", [1, 2, 4])
def test_primitive_wave_killing_relaxes_density_velocity_and_temperature_node_by_node(m):
    """With Q0 = the fields of the snapshot and Q those of a different state, after ref_damp the nodal rho, v_x, v_y
    and T = p/rho (NumPy's Legendre evaluation of the modal states) satisfy Q' = (dt Q0 + tau Q)/(tau + dt) with the
    cell's tau, in both zones; cells between the zones are untouched bitwise; U = U0 is a fixed point; tau -> 0
    returns the initial state."""
    n = 24
    p, U0 = W.random_smooth(n, n, m, seed=70 + m, eos=0, bc=2, rk=2, gravity=True, amp=0.3)
    _, U = W.random_smooth(n, n, m, seed=170 + m, eos=0, bc=2, rk=2, gravity=True, amp=0.3)
    p.update(damp_r0=0.9, damp_r1=1.2, damp_in_r0=0.4, damp_in_r1=0.3, damp_mode=1)
    r = oracle.RefDG(p)
    r.set_state(U0)
    r.damp(0.3)
    np.testing.assert_allclose(r.get_state(), U0, rtol=0, atol=2e-15 * np.abs(U0).max())     # fixed point
    dtd = 0.37
    r.load_working_state(U)
    r.damp(dtd)
    V = r.get_state()
    ft = _zone_factors(p, dtd)[:, :, None, None]
    a, b, c = _prim_nodal(p, U0), _prim_nodal(p, U), _prim_nodal(p, V)
    for k in range(4):
        np.testing.assert_allclose(c[k], (1 - ft) * a[k] + ft * b[k], rtol=0, atol=1e-13)
    mid = (ft[:, :, 0, 0] == 1.0)
    np.testing.assert_array_equal(V[mid], U[mid])
    assert (~mid).sum() > 100 and np.abs(V - U)[~mid].max() > 1e-3
    # a different operation from relaxing the conservative coefficients (mode 0)
    r0 = oracle.RefDG(dict(p, damp_mode=0))
    r0.set_state(U0)
    r0.load_working_state(U)
    r0.damp(dtd)
    assert np.abs(r0.get_state() - V)[~mid].max() > 1e-4
    # tau -> 0 (GM -> infinity in tau = 2 pi sqrt(r_d^3/GM)/R): the initial state comes back where R > 0
    q = oracle.RefDG(dict(p, gm_star=1e40))
    q.set_state(U0)
    q.load_working_state(U)
    q.damp(1.0)
    np.testing.assert_allclose(q.get_state()[~mid], U0[~mid], rtol=0, atol=1e-10)


def test_primitive_wave_killing_hand_worked_cell():
    """m = 1, one cell in the fully damped region (R = 1), dt = tau so that f0 = ft = 1/2.  Initial state rho0 = 1,
    v0 = 0, T0 = 1 (E0 = 2.5); current state rho = 2, v = (1, 0), T = 1/4 (p = 1/2, E = 1.25 + 1 = 2.25):
    rho' = 3/2, v' = 1/2, T' = 5/8 -> m_x' = 3/4, E' = (3/2)(5/8)/0.4 + (3/2)(1/4)/2 = 2.53125.
    Relaxing the conservative fields instead (mode 0) gives m_x' = 1, E' = 2.375."""
    p = W.make_params(nx=1, ny=1, order=1, x0=2.0, x1=3.0, y0=-0.5, y1=0.5, eos=0, gamma=1.4, bc=2,
                      gm_star=1.0, damp_r0=1.0, damp_r1=1.5, damp_mode=1)
    U0 = np.zeros((1, 1, 4, 1, 1))
    U0[0, 0, :, 0, 0] = [1.0, 0.0, 0.0, 2.5]
    tau = 2 * math.pi * math.sqrt(1.0 ** 3 / 1.0)
    for mode, expect in ((1, [1.5, 0.75, 0.0, 2.53125]), (0, [1.5, 1.0, 0.0, 2.375])):
        c = oracle.RefDG(dict(p, damp_mode=mode))
        c.set_state(U0)
        c.load_working_state(np.array([2.0, 2.0, 0.0, 2.25]).reshape(1, 1, 4, 1, 1))
        c.damp(tau)
        np.testing.assert_allclose(c.get_state()[0, 0, :, 0, 0], expect, rtol=0, atol=1e-14)


def test_normalised_torque_hand_value():
    """gamma Gamma / Gamma_0, Gamma_0 = Sigma Omega^2 r_p^4 q / h^2: one massive cell, by hand."""
    p = W.make_params(nx=12, ny=12, order=2, x0=-2.0, x1=2.0, y0=-2.0, y1=2.0, eos=0, gamma=1.4, gm_star=1.0,
                      q_planet=1e-3, r_planet=1.0, eps_planet=0.1, omega_planet=1.0, phase0=0.0, h_aspect=0.05)
    U = np.zeros((12, 12, 4, 2, 2))
    U[9, 7, 0, 0, 0] = 3.0
    r = oracle.RefDG(p)
    r.set_state(U)
    dx = 4.0 / 12
    xcell, ycell = -2 + 7.5 * dx, -2 + 9.5 * dx
    gam = 3.0 * dx * dx * ycell / ((xcell - 1) ** 2 + ycell ** 2 + 0.01) ** 1.5
    sigma_p = 0.7
    gamma0 = sigma_p * 1.0 * 1.0 * 1e-3 / 0.05 ** 2
    assert abs(r.torque_normalised(0.0, sigma_p) - 1.4 * gam / gamma0) < 1e-12 * abs(gam / gamma0)
    # every factor of Gamma_0 with a value other than 1: r_p = 1.5 (fourth power), Omega = 0.6 (squared), planet at
    # phase 0.3
    rp, om, ph = 1.5, 0.6, 0.3
    p2 = dict(p, r_planet=rp, omega_planet=om, phase0=ph)
    r2 = oracle.RefDG(p2)
    r2.set_state(U)
    xp, yp = rp * math.cos(ph), rp * math.sin(ph)
    ddx, ddy = xcell - xp, ycell - yp
    d3 = (ddx ** 2 + ddy ** 2 + 0.01) ** 1.5
    gam2 = 3.0 * dx * dx * (xp * ddy - yp * ddx) / d3
    gamma02 = sigma_p * om ** 2 * rp ** 4 * 1e-3 / 0.05 ** 2
    assert abs(r2.torque_normalised(0.0, sigma_p) - 1.4 * gam2 / gamma02) < 1e-12 * abs(gam2 / gamma02)


# ------------------------------------------------------------------------------------------------
# Step (v) of the paper's loop: the time advances by the step just taken, and the planet of the
# next step's source term sits where that time puts it.  Mutation caught: `c->t += dt` dropped from the step.
def test_time_advances_and_the_planet_moves_with_it():
    p, U = W.disc(12, 2, planet=True, noise=0.0)
    p = dict(p, q_planet=1e-2, t0=0.25)
    a = oracle.RefDG(p)
    a.set_state(U)
    assert a.time == 0.25
    dt = a.cfl_dt(0.2)
    a.step(dt)
    assert a.time == 0.25 + dt
    a.step(dt)
    assert a.time == 0.25 + dt + dt
    # the same two steps with the clock put back by hand after the first one: the second step then evaluates the
    # planet's gravity dt too early, and the result differs
    b = oracle.RefDG(p)
    b.set_state(U)
    b.step(dt)
    b.time = 0.25
    b.step(dt)
    assert np.abs(b.get_state() - a.get_state()).max() > 1e-12
