"""Pins for oracle/sark.py (no GPU): PAPER.md:L136 (reduction to the base RK), eq. 14 (L142, with reading R5),
the printed-formula values (golden file), and exactness / order on a scalar stiff ODE."""
import os

import mpmath
import numpy as np
import pytest

from oracle import sark

GOLD = os.path.join(os.path.dirname(__file__), "golden", "sark_coefficients.txt")


def test_golden_values():
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        v = [float(x) for x in line.split()]
        a, b = sark.coefficients(v[0])
        got = [a[1][0], a[2][0], a[2][1], a[3][0], a[3][2], b[0], b[1], b[3]]
        assert np.allclose(got, v[1:], rtol=4e-16, atol=0)
        assert b[2] == b[1] and a[3][1] == 0.0


@pytest.mark.parametrize("gamma", [-1e-6, -1e-3, -0.04, -0.5, -3.0, -40.0])
def test_row_sums_eq14(gamma):
    """sum_j a~_ij = (e^{c_i g} - 1)/g, sum_j b~_j = (e^g - 1)/g  (eq. 14 without the spurious 1/c_i, reading R5;
    this is also what the paper's own GCL argument, L175-184, needs)."""
    mpmath.mp.dps = 40
    a, b = sark.coefficients(gamma)
    g = mpmath.mpf(gamma)
    for i, ci in ((1, 0.5), (2, 0.5), (3, 1.0)):
        exact = (mpmath.e ** (ci * g) - 1) / g
        assert abs(sum(a[i]) - float(exact)) < 4e-16
    assert abs(sum(b) - float((mpmath.e ** g - 1) / g)) < 4e-16


def test_limit_is_classic_rk4():
    """PAPER.md:L136 + reading R4: as 1/tau -> 0 the scheme is the classic RK4 (Table 1, blank in PAPER.md)."""
    a, b = sark.coefficients(-1e-9)
    assert np.allclose(a, sark.RK4_A, atol=1e-9)
    assert np.allclose(b, sark.RK4_B, atol=1e-9)
    a0, b0 = sark.coefficients(0.0)
    assert a0 == [list(r) for r in sark.RK4_A] and b0 == list(sark.RK4_B)
    # classic RK4 consistency (eq. 13)
    assert abs(sum(sark.RK4_B) - 1) < 1e-16
    for i in range(4):
        assert abs(sum(sark.RK4_A[i]) - sark.RK4_C[i]) < 1e-16


def scalar_sark(lam, f, q0, dt, nsteps):
    """q' = -lam q + f(t) with the recurrence of PAPER.md:L132-134, coefficients from the oracle."""
    a, b = sark.coefficients(-dt * lam)
    c = sark.RK4_C
    q, t = q0, 0.0
    for _ in range(nsteps):
        F = []
        for i in range(4):
            F.append(f(t + c[i] * dt))          # forcing independent of q: F_ni = f(t_n + c_i dt)
        q = q * np.exp(-lam * dt) + dt * sum(b[j] * F[j] for j in range(4))
        t += dt
    return q


def test_scalar_constant_forcing_is_exact():
    lam, alpha, q0 = 250.0, 3.0, 0.7
    for dt in (0.1, 0.01):
        n = int(round(1.0 / dt))
        exact = q0 * np.exp(-lam) + alpha / lam * (1 - np.exp(-lam))
        assert abs(scalar_sark(lam, lambda t: alpha, q0, dt, n) - exact) < 1e-14


def test_scalar_fourth_order():
    lam, q0 = 2.0, 1.0
    f = lambda t: np.sin(3 * t)
    # exact: q = e^{-lam t} q0 + int_0^t e^{-lam (t-s)} sin(3 s) ds
    exact = float(mpmath.e ** (-lam) * q0 + mpmath.quad(lambda s: mpmath.e ** (-lam * (1 - s)) * mpmath.sin(3 * s), [0, 1]))
    errs = [abs(scalar_sark(lam, f, q0, 1.0 / n, n) - exact) for n in (8, 16, 32)]
    rates = [np.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert all(r > 3.7 for r in rates), (errs, rates)
