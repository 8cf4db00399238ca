"""Pins of oracle/cubature.py (no GPU): the cubature-projected relaxation P N~(I q) of PAPER.md:L84-107, L197 (NEXT-1).

Nothing here re-types P = M^-1 I^T diag(w):
  * Galerkin property against closed forms: for monomials g (degree <= N) and f (degree <= 2N),
    g^T M (P f(x^c)) = int g f, the integral from Dirichlet's formula -- pins points, weights, I, M^-1 together
  * P I = identity (a rule exact to degree 2N reproduces the polynomial space)
  * the projection preserves the integral: 1^T M (P f) = sum_c w_c f_c
  * it is the L2-best approximation: closer to an under-resolved f in L2 than the nodal interpolant (de-aliasing, L84)
  * where N~(q) is itself a polynomial of degree <= N (uniform density, velocity of degree <= N/2) the cubature and
    the collocated relaxation (reading R8) agree to round-off; a uniform state gives the same F in both modes
  * free stream and exact uniform relaxation hold in cubature mode on a moving mesh (L154-184, L123)
"""
import numpy as np
import pytest

from oracle import cubature, physics, sark
from oracle.quadrature import simplex_rule
from workloads import configs
from helpers import oracle_problem
from test_oracle_operators import mono, monomials, unit_monomial_integral

PAIRS = [(2, 1), (2, 3), (2, 4), (3, 2), (3, 3), (3, 4)]


@pytest.mark.parametrize("dim,N", PAIRS)
def test_projection_is_galerkin_against_closed_form_integrals(dim, N, refs):
    ref = refs(dim, N)
    cub = cubature.Cubature(ref)
    assert cub.degree == 3 * N and np.all(cub.w > 0)
    assert abs(cub.w.sum() - (2.0 if dim == 2 else 4.0 / 3.0)) < 1e-14
    worst = 0.0
    for ef in monomials(dim, 2 * N):
        pf = cub.P @ mono(cub.x, ef)                       # nodal values of the projection of f
        for eg in monomials(dim, N):
            lhs = mono(ref.x, eg) @ ref.M @ pf
            rhs = unit_monomial_integral(dim, tuple(a + b for a, b in zip(ef, eg)))
            worst = max(worst, abs(lhs - rhs))
    assert worst < 2e-14


@pytest.mark.parametrize("dim,N", PAIRS)
def test_projection_reproduces_polynomials_and_preserves_integrals(dim, N, refs):
    ref = refs(dim, N)
    cub = cubature.Cubature(ref)
    assert np.abs(cub.P @ cub.I - np.eye(ref.Np)).max() < 5e-13
    rng = np.random.default_rng(199)
    f = rng.standard_normal(cub.Nc)
    assert abs(ref.w @ (cub.P @ f) - cub.w @ f) < 1e-13     # 1^T M P f = sum w f


@pytest.mark.parametrize("dim,N", [(2, 3), (3, 3)])
def test_projection_is_closer_in_L2_than_interpolation(dim, N, refs):
    ref = refs(dim, N)
    cub = cubature.Cubature(ref)
    xf, wf = simplex_rule(dim, 24)
    If = np.asarray(ref.lagrange(xf), dtype=float)

    def f(x):                                               # rational, like q2 q3 / q1: not in the polynomial space
        return np.sin(2.5 * x[:, 0] + 1.0) * np.cos(1.5 * x[:, -1]) / (1.3 + 0.4 * x[:, 0])
    err_proj = np.sqrt(wf @ (If @ (cub.P @ f(cub.x)) - f(xf)) ** 2)
    err_intp = np.sqrt(wf @ (If @ f(ref.x) - f(xf)) ** 2)
    assert err_proj < err_intp
    # and the projection residual is L2-orthogonal to the polynomial space up to the rule's own exactness
    resid = If @ (cub.P @ f(cub.x)) - f(xf)
    assert np.abs(If.T @ (wf * resid)).max() < 2e-3 * err_intp


@pytest.mark.parametrize("dim", [2, 3])
def test_equals_collocation_where_the_term_is_a_polynomial(dim, refs):
    N = 4
    ref = refs(dim, N)
    cub = cubature.Cubature(ref)
    rng = np.random.default_rng(199)
    K, Nf = 3, physics.nfields(dim)
    q = np.zeros((K, Nf, ref.Np))
    q[:, 0, :] = 1.7                                        # uniform density
    for k in range(K):
        for d in range(dim):                                # velocity fields of degree N/2 = 2
            for e in monomials(dim, N // 2):
                q[k, 1 + d, :] += rng.standard_normal() * mono(ref.x, e)
    q[:, 1 + dim:, :] = rng.standard_normal((K, Nf - 1 - dim, ref.Np))   # second moments do not enter N~
    a = cubature.relaxation(cub, dim, q, 1e-2)
    b = physics.N_tilde(dim, q, 1e-2)
    assert np.abs(b).max() > 1.0
    assert np.abs(a - b).max() < 1e-12 * np.abs(b).max()
    # a non-polynomial term does differ (the mode is not a no-op)
    q[:, 0, :] = 1.7 + 0.3 * mono(ref.x, (N,) + (0,) * (dim - 1))
    assert np.abs(cubature.relaxation(cub, dim, q, 1e-2) - physics.N_tilde(dim, q, 1e-2)).max() > 1e-6


@pytest.mark.parametrize("dim", [2, 3])
def test_free_stream_and_uniform_relaxation_in_cubature_mode(dim, refs):
    ref = refs(dim, 3)
    cfg = configs.config1(ref.lam, n=4) if dim == 2 else configs.config4(ref.lam, n=3)
    cfg["relax"] = "cubature"
    Nf = physics.nfields(dim)
    u = np.array([0.1, 0.05, -0.02][:dim])
    q0 = np.broadcast_to(physics.equilibrium_state(dim, np.array(1.0), u, 1.0)[None, :, None], (cfg["K"], Nf, ref.Np)).copy()
    P = oracle_problem(cfg, ref)
    assert P.cub is not None
    stages, _ = sark.step_debug(P, q0, 0.13, cfg["dt"])
    for s in stages:
        assert np.abs(s - q0).max() < 1e-14                 # free stream, every stage
    # uniform non-equilibrium state: q_k(t) = q_k^eq + (q_k(0) - q_k^eq) e^{-t/tau} exactly (L123)
    q1 = q0.copy()
    q1[:, 1 + dim, :] += 0.01
    tau, dt, n = cfg["tau"], cfg["dt"], 5
    q = sark.step(P, q1, 0.0, dt, n)
    expect = q0[0, 1 + dim, 0] + 0.01 * np.exp(-n * dt / tau)
    assert np.abs(q[:, 1 + dim, :] - expect).max() < 1e-13
    # same F as the collocated mode on a uniform state
    cfg2 = dict(cfg)
    cfg2["relax"] = "collocation"
    assert np.abs(P.rhs(q1, 0.2) - oracle_problem(cfg2, ref).rhs(q1, 0.2)).max() < 1e-10 * np.abs(P.rhs(q1, 0.2)).max()
