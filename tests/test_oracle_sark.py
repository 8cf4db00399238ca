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


# ------------------------------------------------------------------ the stage recurrence of sark.step_debug itself
class _LinearSystem:
    """A stand-in for oracle.rhs.Problem with F(q, t) = M q + g(t), M dense: every field feeds every other, so each
    F_nj differs from the others and from stage to stage (unlike free stream / uniform relaxation, where all F_nj are
    equal and only the row sums of a~ are exercised)."""
    dim, sigma = 2, None

    def __init__(self, tau, seed=3):
        rng = np.random.default_rng(seed)
        self.tau = tau
        self.M = rng.uniform(-1, 1, size=(6, 6))
        self.gv = rng.uniform(-1, 1, size=(6, 3))

    def g(self, t):
        return self.gv[:, 0] * np.sin(3 * t) + self.gv[:, 1] * np.cos(2 * t) + self.gv[:, 2] * t

    def rhs(self, q, t, verts=None):
        return np.einsum("fg,kgi->kfi", self.M, q) + self.g(t)[None, :, None]


@pytest.mark.parametrize("tau", [0.1, 0.05])
def test_step_recurrence_is_fourth_order_on_a_coupled_stiff_system(tau):
    """PAPER.md:L132-134 with the coefficients of L148: q' = -Lambda q + M q + g(t), Lambda = diag(0,0,0,1/tau x3),
    integrated by oracle.sark.step with |gamma| = dt/tau between 2 and 0.125, against an adaptive high-order
    integration of the same ODE (scipy DOP853, rtol 1e-13).  The error must fall 16-fold per halving of dt, for the
    stiff fields on their own too.  a~_20 and a~_21 applied to the wrong F_nj (or a wrong exponent e^{-Lambda c_i dt})
    leave free stream and uniform relaxation intact but drop this to second order (ratio 4)."""
    from scipy.integrate import solve_ivp
    from oracle import physics
    P = _LinearSystem(tau)
    lam = physics.stiff_mask(2) / tau
    q0 = np.linspace(0.5, 1.5, 6)
    T = 0.8
    sol = solve_ivp(lambda t, y: -lam * y + P.M @ y + P.g(t), (0, T), q0, method="DOP853", rtol=1e-13, atol=1e-15)
    exact = sol.y[:, -1]
    errs = np.array([np.abs(sark.step(P, q0[None, :, None].copy(), 0.0, T / n, n)[0, :, 0] - exact) for n in (8, 16, 32, 64)])
    for sel in (slice(None), slice(3, 6)):
        e = errs[:, sel].max(axis=1)
        assert all(e[i] / e[i + 1] >= 14.0 for i in range(3)), e
    assert errs[-1].max() < 1e-7                             # error constant of a 4th-order scheme, not just its slope


def test_step_temporal_self_convergence_on_a_moving_mesh(refs):
    """oracle.sark.step on the real operator (2-D, N=2, SINES_PRODUCT motion, finite tau with gamma = -1 at the
    coarsest dt, second moments away from equilibrium): errors at dt, dt/2, dt/4 against the dt/8 run fall by >= 14
    per halving (geometry re-evaluated at every stage time, L152-154)."""
    from helpers import oracle_problem
    from workloads import configs
    ref = refs(2, 2)
    cfg = configs.config2(ref.lam, n=4)
    cfg["N"] = 2
    cfg = configs._finish(cfg, ref.lam)
    dt0 = cfg["dt"]
    cfg["tau"] = dt0
    P = oracle_problem(cfg, ref)
    q0 = cfg["q0"].copy()
    q0[:, 3:] += 0.02 * np.sin(configs.node_coordinates(cfg["X0"], cfg["EToV"], ref.lam)[..., 0])[:, None, :]
    T = 8 * dt0
    outs = [sark.step(P, q0, 0.1, T / n, n) for n in (8, 16, 32, 64)]
    for sel in (slice(None), slice(3, 6)):
        e = [np.abs(o - outs[-1])[:, sel].max() for o in outs[:-1]]
        assert e[0] / e[1] >= 14.0 and e[1] / e[2] >= 14.0, e
        assert e[2] > 1e-13                                  # still above round-off: the ratios mean something
