"""Pins of oracle/coords.py (no GPU): mesh coordinates advanced by the solver's RK4 (NEXT-2).

  * the integrated vertex positions converge to the closed-form law x(t) = X0 + disp(X0, t) at 4th order
    (dx/dt = v(X0, t) is a quadrature; classic RK4 reduces to Simpson's rule, error per step ~ dt^5 v''''/2880)
  * a velocity that is constant in time is integrated exactly, stage positions included
  * free-stream preservation on the integrated mesh, every stage (Table 2: that run integrated
    dx/dt = v_G)
  * with the motion switched off the integrated-coordinate step equals the closed-form step bit for bit
"""
import numpy as np
import pytest

from oracle import coords, motion, sark
from workloads import configs
from helpers import oracle_problem


def _integrate(P, T, nsteps):
    x = P.X0.copy()
    dt = T / nsteps
    for n in range(nsteps):
        _, x = coords.stage_vertices(P, x, n * dt, dt)
    return x


@pytest.mark.parametrize("dim", [2, 3])
def test_positions_converge_to_closed_form_at_fourth_order(dim, refs):
    ref = refs(dim, 3)
    cfg = configs.config1(ref.lam, n=4) if dim == 2 else configs.config4(ref.lam, n=3)
    P = oracle_problem(cfg, ref)
    T = 0.3
    exact = motion.vertices(P.motion_kind, P.motion_params, P.X0, T)[0]
    errs = [np.abs(_integrate(P, T, n) - exact).max() for n in (4, 8, 16)]
    assert errs[0] > 1e-12                              # not trivially exact
    rates = [np.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert all(3.8 < r < 4.3 for r in rates), (errs, rates)
    # Simpson's error constant: |err| <= T dt^4 max|d^4 v/dt^4| / 2880, v = A om cos(om t) shape
    A, per = cfg["motion_params"][0], cfg["motion_params"][1]
    om = 2 * np.pi / per
    bound = T * (T / 16) ** 4 * A * om ** 5 / 2880
    assert errs[2] <= 1.05 * bound


def test_velocity_constant_in_time_is_exact(refs):
    """PLUNGE_BLEND with omega -> 0 has no closed constant-velocity form, so use the law-free path: a Problem whose
    law is NONE and explicit stage velocities."""
    ref = refs(2, 3)
    cfg = configs.config1(ref.lam, n=4)
    P = oracle_problem(cfg, ref)
    rng = np.random.default_rng(199)
    v = rng.standard_normal(P.X0.shape)
    x_n = P.X0 + 0.01 * rng.standard_normal(P.X0.shape)
    dt = 0.037

    class Const:                                     # same interface as the Problem fields coords.velocity reads
        motion_kind, motion_params, X0 = motion.NONE, None, P.X0
    verts, x_next = coords.stage_vertices(Const, x_n, 0.2, dt)
    assert all(np.array_equal(vv, np.zeros_like(v)) for _, vv in verts)
    assert np.array_equal(x_next, x_n)
    # constant non-zero velocity through the recurrence itself
    k = [v, v, v, v]
    x1 = x_n + dt * sark.RK4_A[1][0] * k[0]
    x_end = x_n + dt * sum(b * kk for b, kk in zip(sark.RK4_B, k))
    assert np.allclose(x1, x_n + 0.5 * dt * v, rtol=0, atol=1e-16)
    assert np.allclose(x_end, x_n + dt * v, rtol=0, atol=2e-16)


@pytest.mark.parametrize("dim", [2, 3])
def test_free_stream_preserved_on_integrated_mesh(dim, refs):
    ref = refs(dim, 3)
    if dim == 2:
        cfg = configs.config1(ref.lam)
        nsteps = 30
    else:
        from oracle import physics
        cfg = configs.config4(ref.lam, n=3)
        cfg["q0"] = np.broadcast_to(
            physics.equilibrium_state(3, np.array(1.0), np.array([0.1, 0.05, -0.02]), 1.0)[None, :, None],
            (cfg["K"], 10, ref.Np)).copy()
        nsteps = 10
    P = oracle_problem(cfg, ref)
    q0 = cfg["q0"]
    stages, _, x1 = coords.step_debug(P, q0, P.X0.copy(), 0.0, cfg["dt"])
    for s in stages:
        assert np.abs(s - q0).max() < 1e-14
    q, x = coords.step(P, q0, P.X0.copy(), 0.0, cfg["dt"], nsteps)
    assert np.abs(q - q0).max() < 1e-13
    assert np.abs(x - P.X0).max() > 1e-3              # the mesh really moved
    exact = motion.vertices(P.motion_kind, P.motion_params, P.X0, nsteps * cfg["dt"])[0]
    assert np.abs(x - exact).max() < 1e-9             # and follows the law to time-integration accuracy


def test_static_mesh_equals_closed_form_step(refs):
    ref = refs(2, 3)
    cfg = configs.config1(ref.lam, n=4)
    cfg["motion_kind"], cfg["motion_params"] = motion.NONE, None
    P = oracle_problem(cfg, ref)
    rng = np.random.default_rng(199)
    q0 = cfg["q0"] * (1 + 1e-3 * rng.standard_normal(cfg["q0"].shape))
    a, _ = sark.step_debug(P, q0, 0.1, cfg["dt"])
    b, _, x1 = coords.step_debug(P, q0, P.X0.copy(), 0.1, cfg["dt"])
    assert np.array_equal(x1, P.X0)
    for sa, sb in zip(a, b):
        assert np.array_equal(sa, sb)


# ------------------------------------------------------------------ caller-supplied stage velocities (NEXT-2, general)
def test_stage_velocities_of_the_law_reproduce_the_law_bit_for_bit(refs):
    ref = refs(2, 3)
    cfg = configs.config1(ref.lam, n=4)
    P = oracle_problem(cfg, ref)
    rng = np.random.default_rng(3)
    q = cfg["q0"] * (1.0 + 1e-3 * rng.standard_normal(cfg["q0"].shape))
    t0, dt = 0.2, cfg["dt"]
    ks = [motion.vertices(P.motion_kind, P.motion_params, P.X0, t0 + c * dt)[1] for c in sark.RK4_C]
    x_n = motion.vertices(P.motion_kind, P.motion_params, P.X0, t0)[0]
    a, _, xa = coords.step_debug(P, q, x_n, t0, dt)
    b, _, xb = coords.step_debug(P, q, x_n, t0, dt, stage_velocities=ks)
    assert np.array_equal(xa, xb) and all(np.array_equal(u, v) for u, v in zip(a, b))


def test_position_dependent_velocity_rigid_rotation_is_fourth_order():
    """dx/dt = Omega x x depends on the positions, so k_2 != k_3: the caller (here: the test, standing in for a
    structure solver) evaluates its velocity at the stage positions it derives itself and hands the four
    k_i over.  x_{n+1} must be the classic RK4 update (L152: "the same Runge-Kutta integration scheme"), whose
    amplification of a rotation by angle h is the degree-4 Taylor polynomial of e^{ih} -- a closed form."""
    class Bare:      # stage_vertices needs no Problem when the velocities are supplied
        pass
    om = 1.3
    x0 = np.array([[1.0, 0.0], [0.3, -0.7], [-2.0, 0.5]])
    rot = lambda x: om * np.stack([-x[:, 1], x[:, 0]], axis=1)
    T = 0.9
    errs = []
    for n in (4, 8, 16):
        dt, x = T / n, x0.copy()
        for _ in range(n):
            k1 = rot(x); k2 = rot(x + 0.5 * dt * k1); k3 = rot(x + 0.5 * dt * k2); k4 = rot(x + dt * k3)
            verts, x_next = coords.stage_vertices(Bare(), x, 0.0, dt, stage_velocities=(k1, k2, k3, k4))
            # the stage positions the oracle hands to the field update are the ones the velocities were evaluated at
            assert np.allclose(verts[1][0], x + 0.5 * dt * k1, atol=1e-15) and np.allclose(verts[2][0], x + 0.5 * dt * k2, atol=1e-15)
            assert np.allclose(verts[3][0], x + dt * k3, atol=1e-15) and np.array_equal(verts[2][1], k3)
            z, h = x[:, 0] + 1j * x[:, 1], om * dt
            amp = 1 + 1j * h + (1j * h) ** 2 / 2 + (1j * h) ** 3 / 6 + (1j * h) ** 4 / 24
            assert np.allclose(x_next[:, 0] + 1j * x_next[:, 1], amp * z, rtol=0, atol=1e-14)
            x = x_next
        exact = (x0[:, 0] + 1j * x0[:, 1]) * np.exp(1j * om * T)
        errs.append(np.abs(x[:, 0] + 1j * x[:, 1] - exact).max())
    rates = [np.log2(errs[i] / errs[i + 1]) for i in range(2)]
    assert all(3.8 < r < 4.3 for r in rates), (errs, rates)
