"""Pins for oracle C3-C6: Euler flux and EOS, LLF numerical flux (PAPER.md:97,
reading G5), gravity source."""
import math
import os

import numpy as np
import pytest

import oracle
from paper_1805_01443_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _golden_flux():
    d = {}
    for line in open(os.path.join(GOLD, "euler_flux_hand.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        d[k] = np.array([float(x) for x in v])
    return d


def test_euler_flux_hand_values():
    g = _golden_flux()
    p = W.make_params(nx=1, ny=1, order=1, eos=0, gamma=float(g["gamma"][0]))
    F, vn, c = oracle.point_flux(p, g["U"], 0.3, 0.4, 0)
    np.testing.assert_allclose(F, g["F"], rtol=1e-15)
    assert vn == 3.0 and abs(c * c - g["c2"][0]) < 1e-15
    G, vn, c = oracle.point_flux(p, g["U"], 0.3, 0.4, 1)
    np.testing.assert_allclose(G, g["G"], rtol=1e-15)
    assert vn == -1.0


def test_isothermal_closure_hand_values():
    """eos 1: p = c_s^2 rho, c_s^2 = h^2 GM / sqrt(r^2 + eps^2) (BASELINE cfg1)."""
    p = W.make_params(nx=1, ny=1, order=1, eos=1, h_aspect=0.05, gm_star=4.0, eps_star=0.0)
    U = np.array([2.0, 6.0, -2.0, 123.0])   # E is passive: must not enter p or c
    F, vn, c = oracle.point_flux(p, U, 1.2, 1.6, 0)      # r = 2 -> cs2 = 0.0025*4/2 = 0.005
    pr = 0.005 * 2.0
    np.testing.assert_allclose(F, [6.0, 18.0 + pr, -6.0, (123.0 + pr) * 3.0], rtol=1e-15)
    assert abs(c - math.sqrt(0.005)) < 1e-16
    p["eps_star"] = 1.5                                   # r_s = 2.5
    _, _, c = oracle.point_flux(p, U, 1.2, 1.6, 1)
    assert abs(c * c - 0.0025 * 4.0 / 2.5) < 1e-16


@pytest.mark.parametrize("eos", [0, 1])
@pytest.mark.parametrize("direction", [0, 1])
def test_llf_consistency_and_dissipation(eos, direction):
    rng = np.random.default_rng(5)
    p = W.make_params(nx=1, ny=1, order=1, eos=eos, gamma=1.4, h_aspect=0.1, gm_star=1.0, eps_star=0.01)
    for _ in range(20):
        rho, vx, vy, pr = rng.uniform(0.5, 2), rng.normal(), rng.normal(), rng.uniform(0.5, 2)
        U = np.array([rho, rho * vx, rho * vy, pr / 0.4 + 0.5 * rho * (vx * vx + vy * vy)])
        x, y = rng.uniform(-1, 1, 2)
        F, vn, c = oracle.point_flux(p, U, x, y, direction)
        # consistency: H(U,U) = f(U).n
        np.testing.assert_array_equal(oracle.llf(p, U, U, x, y, direction), F)
        # H - mean flux = -lambda/2 (UR-UL), lambda = max(|v_n|+c) over both sides (pointwise, G5)
        d = rng.normal(size=4) * 1e-3
        UR = U + d
        FR, vnR, cR = oracle.point_flux(p, UR, x, y, direction)
        lam = max(abs(vn) + c, abs(vnR) + cR)
        H = oracle.llf(p, U, UR, x, y, direction)
        np.testing.assert_allclose(H, 0.5 * (F + FR) - 0.5 * lam * (UR - U), rtol=1e-14, atol=1e-15)


@pytest.mark.parametrize("direction", [0, 1])
def test_llf_bitwise_mirror_antisymmetry(direction):
    """h(UL,UR;n) = -h(UR,UL;-n): mirror the normal momentum, swap sides, result flips bitwise.
    A single-valued interface flux is what makes the scheme conservative."""
    rng = np.random.default_rng(7)
    p = W.make_params(nx=1, ny=1, order=1, eos=0, gamma=1.4)
    nrm = 1 + direction
    for _ in range(50):
        UL = np.array([1.0, 0.3, -0.2, 2.5]) + 0.1 * rng.normal(size=4)
        UR = np.array([1.1, -0.4, 0.1, 2.2]) + 0.1 * rng.normal(size=4)
        H = oracle.llf(p, UL, UR, 0.0, 0.0, direction)
        ML, MR = UL.copy(), UR.copy()
        ML[nrm] *= -1
        MR[nrm] *= -1
        Hm = oracle.llf(p, MR, ML, 0.0, 0.0, direction)
        sign = np.array([-1.0, -1.0, -1.0, -1.0])
        sign[nrm] = 1.0
        np.testing.assert_array_equal(Hm, sign * H)


def _potential(p, t, x, y):
    phi = -p["gm_star"] / math.sqrt(x * x + y * y + p["eps_star"] ** 2)
    if p["q_planet"]:
        a = p["omega_planet"] * t + p["phase0"]
        xp, yp = p["r_planet"] * math.cos(a), p["r_planet"] * math.sin(a)
        phi += -p["q_planet"] * p["gm_star"] / math.sqrt((x - xp) ** 2 + (y - yp) ** 2 + p["eps_planet"] ** 2)
    return phi


@pytest.mark.parametrize("q", [0.0, 3e-2])
def test_gravity_is_minus_grad_phi(q):
    p = W.make_params(nx=1, ny=1, order=1, gm_star=1.7, eps_star=0.02, q_planet=q, r_planet=0.9,
                      eps_planet=0.03, omega_planet=1.3, phase0=0.4)
    rng = np.random.default_rng(11)
    h = 1e-5
    for _ in range(30):
        x, y = rng.uniform(-2, 2, 2)
        t = rng.uniform(0, 5)
        g = oracle.gravity(p, t, x, y)
        gx = -(_potential(p, t, x + h, y) - _potential(p, t, x - h, y)) / (2 * h)
        gy = -(_potential(p, t, x, y + h) - _potential(p, t, x, y - h)) / (2 * h)
        np.testing.assert_allclose(g, [gx, gy], rtol=2e-6, atol=1e-8)


def test_planet_orbit_is_periodic_and_no_gravity_without_star():
    p = W.make_params(nx=1, ny=1, order=1, gm_star=1.0, eps_star=0.02, q_planet=1e-3, r_planet=1.0,
                      eps_planet=0.03, omega_planet=1.0, phase0=0.0)
    g0 = oracle.gravity(p, 0.0, 0.7, 0.2)
    g1 = oracle.gravity(p, 2 * math.pi, 0.7, 0.2)
    np.testing.assert_allclose(g0, g1, rtol=1e-13)
    gh = oracle.gravity(p, math.pi, 0.7, 0.2)
    assert abs(gh[0] - g0[0]) > 1e-6          # the planet did move in between
    # planet sits at (1, 0) at t = 0: its own pull at (1+d, 0) points in -x with the softened law
    d = 0.05
    star = -1.0 * (1 + d) / ((1 + d) ** 2 + 0.02 ** 2) ** 1.5
    pl = -1e-3 * d / (d * d + 0.03 ** 2) ** 1.5
    np.testing.assert_allclose(oracle.gravity(p, 0.0, 1 + d, 0.0), [star + pl, 0.0], rtol=1e-14, atol=1e-18)
    p["gm_star"] = 0.0
    np.testing.assert_array_equal(oracle.gravity(p, 0.3, 0.7, 0.2), [0.0, 0.0])
