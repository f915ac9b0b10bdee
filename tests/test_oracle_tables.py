"""Pins for oracle C1 (tables): PAPER.md:65 (orthonormal Legendre basis)
(Gauss-Legendre quadrature), PAPER.md:155 (zeroth mode = cell average)."""
import math

import numpy as np
import pytest
from numpy.polynomial import legendre as npleg

import oracle

ORDERS = [1, 2, 3, 4, 5]

# Closed forms of the Gauss-Legendre rules (Abramowitz & Stegun 25.4.29), ascending nodes.
CLOSED = {
    1: ([0.0], [2.0]),
    2: ([-1 / math.sqrt(3), 1 / math.sqrt(3)], [1.0, 1.0]),
    3: ([-math.sqrt(3 / 5), 0.0, math.sqrt(3 / 5)], [5 / 9, 8 / 9, 5 / 9]),
    4: ([-math.sqrt(3 / 7 + 2 / 7 * math.sqrt(6 / 5)), -math.sqrt(3 / 7 - 2 / 7 * math.sqrt(6 / 5)),
         math.sqrt(3 / 7 - 2 / 7 * math.sqrt(6 / 5)), math.sqrt(3 / 7 + 2 / 7 * math.sqrt(6 / 5))],
        [(18 - math.sqrt(30)) / 36, (18 + math.sqrt(30)) / 36,
         (18 + math.sqrt(30)) / 36, (18 - math.sqrt(30)) / 36]),
    5: ([-math.sqrt(5 + 2 * math.sqrt(10 / 7)) / 3, -math.sqrt(5 - 2 * math.sqrt(10 / 7)) / 3, 0.0,
         math.sqrt(5 - 2 * math.sqrt(10 / 7)) / 3, math.sqrt(5 + 2 * math.sqrt(10 / 7)) / 3],
        [(322 - 13 * math.sqrt(70)) / 900, (322 + 13 * math.sqrt(70)) / 900, 128 / 225,
         (322 + 13 * math.sqrt(70)) / 900, (322 - 13 * math.sqrt(70)) / 900]),
}


@pytest.mark.parametrize("m", ORDERS)
def test_closed_forms_and_numpy(m):
    t = oracle.tables(m)
    xi, w = CLOSED[m]
    np.testing.assert_allclose(t["xi"], xi, rtol=0, atol=2e-16)
    np.testing.assert_allclose(t["w"], w, rtol=0, atol=4e-16)
    x2, w2 = npleg.leggauss(m)
    np.testing.assert_allclose(t["xi"], x2, rtol=0, atol=3e-16)
    np.testing.assert_allclose(t["w"], w2, rtol=0, atol=6e-16)


@pytest.mark.parametrize("m", ORDERS)
def test_weights_sum_and_polynomial_exactness(m):
    t = oracle.tables(m)
    assert abs(t["w"].sum() - 2.0) < 1e-15
    for k in range(2 * m):          # exact up to degree 2m-1
        exact = 0.0 if k % 2 else 2.0 / (k + 1)
        assert abs((t["w"] * t["xi"] ** k).sum() - exact) < 2e-15
    # and NOT exact at degree 2m: the rule really has only m points
    assert abs((t["w"] * t["xi"] ** (2 * m)).sum() - 2.0 / (2 * m + 1)) > 1e-6


@pytest.mark.parametrize("m", ORDERS)
def test_orthonormal_basis_diagonal_mass(m):
    """(1/|K|) int phi_a phi_b = delta_ab with the m-point rule (reading G1)."""
    t = oracle.tables(m)
    M = np.einsum("q,qa,qb->ab", 0.5 * t["w"], t["B"], t["B"])
    np.testing.assert_allclose(M, np.eye(m), rtol=0, atol=1e-15)
    # phi_0 == 1: the zeroth mode is the cell average
    np.testing.assert_allclose(t["B"][:, 0], 1.0, rtol=0, atol=0)


@pytest.mark.parametrize("m", ORDERS)
def test_basis_values_derivatives_and_end_values(m):
    t = oracle.tables(m)
    for a in range(m):
        c = np.zeros(a + 1)
        c[a] = math.sqrt(2 * a + 1)
        np.testing.assert_allclose(t["B"][:, a], npleg.legval(t["xi"], c), rtol=0, atol=2e-15)
        np.testing.assert_allclose(t["D"][:, a], npleg.legval(t["xi"], npleg.legder(c)) if a else 0.0,
                                   rtol=0, atol=2e-14)
        assert t["Ep"][a] == math.sqrt(2 * a + 1)
        assert t["Em"][a] == (-1) ** a * math.sqrt(2 * a + 1)


@pytest.mark.parametrize("m", ORDERS)
def test_discrete_divergence_theorem(m):
    """sum_q w_q phi_a'(xi_q) = phi_a(1) - phi_a(-1): what makes free-stream preservation exact."""
    t = oracle.tables(m)
    np.testing.assert_allclose(t["w"] @ t["D"], t["Ep"] - t["Em"], rtol=0, atol=4e-15)
