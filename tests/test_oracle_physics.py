"""Pins for oracle/physics.py (no GPU): the moment system the paper leaves blank is pinned by
what the paper does print — equilibrium moments (L43), macroscopic relations (L47, L51) — and by the mathematics
(Gauss-Hermite characteristic speeds, symmetry, 3-D -> 2-D reduction)."""
import numpy as np
import pytest

from oracle import physics


def test_2d_matrices_match_reading_R1():
    """DESIGN.md R1 (written out equation by equation from the Hermite recurrence):
    d q1 + c(dx q2 + dy q3); d q2 + c(dx(q1 + r2 q5) + dy q4); d q3 + c(dx q4 + dy(q1 + r2 q6));
    d q4 + c(dx q3 + dy q2); d q5 + c r2 dx q2; d q6 + c r2 dy q3."""
    r2 = np.sqrt(2.0)
    Ax = np.zeros((6, 6)); Ay = np.zeros((6, 6))
    Ax[0, 1] = 1; Ax[1, 0] = 1; Ax[1, 4] = r2; Ax[2, 3] = 1; Ax[3, 2] = 1; Ax[4, 1] = r2
    Ay[0, 2] = 1; Ay[1, 3] = 1; Ay[2, 0] = 1; Ay[2, 5] = r2; Ay[3, 1] = 1; Ay[5, 2] = r2
    A = physics.stream_matrices(2)
    assert np.array_equal(A[0], Ax) and np.array_equal(A[1], Ay)


@pytest.mark.parametrize("dim", [2, 3])
def test_characteristic_speeds(dim):
    """A_n = sum n_d A^_d is symmetric with spectrum {0, +-1, +-sqrt3} (the Gauss-Hermite abscissae of the 3-point rule
    a degree-2 Hermite closure induces) for EVERY unit normal: rotation invariance of the closure."""
    rng = np.random.default_rng(3)
    A = physics.stream_matrices(dim)
    nf = physics.nfields(dim)
    for _ in range(20):
        n = rng.standard_normal(dim); n /= np.linalg.norm(n)
        An = sum(n[d] * A[d] for d in range(dim))
        assert np.array_equal(An, An.T)
        ev = np.sort(np.linalg.eigvalsh(An))
        expect = np.sort(np.concatenate([[-np.sqrt(3), np.sqrt(3)], [-1] * (dim - 1), [1] * (dim - 1),
                                         np.zeros(nf - 2 * dim)]))
        assert np.allclose(ev, expect, atol=1e-13)


def test_3d_reduces_to_2d():
    """With no z-dependence and no z-momentum the 3-D system restricted to (q1,q2,q3,q5,q8,q9) is the 2-D system."""
    A3, A2 = physics.stream_matrices(3), physics.stream_matrices(2)
    sel = [0, 1, 2, 4, 7, 8]                      # (000,100,010,110,200,020) <-> (00,10,01,11,20,02)
    for d in range(2):
        assert np.array_equal(A3[d][np.ix_(sel, sel)], A2[d])
    assert physics.stiff_mask(3).tolist() == [0, 0, 0, 0, 1, 1, 1, 1, 1, 1]
    assert physics.stiff_mask(2).tolist() == [0, 0, 0, 1, 1, 1]      # Lambda of PAPER.md:L115


@pytest.mark.parametrize("dim", [2, 3])
def test_collision_term_printed_form(dim):
    rng = np.random.default_rng(4)
    q = rng.uniform(0.5, 1.5, size=(3, physics.nfields(dim), 7))
    tau = 0.013
    N = physics.N_full(dim, q, tau)
    if dim == 2:
        # PAPER.md:L43 verbatim
        q1, q2, q3, q4, q5, q6 = [q[:, i, :] for i in range(6)]
        exp = -1 / tau * np.stack([0 * q1, 0 * q1, 0 * q1, q4 - q2 * q3 / q1, q5 - q2 ** 2 / (q1 * np.sqrt(2)),
                                   q6 - q3 ** 2 / (q1 * np.sqrt(2))], axis=1)
        assert np.allclose(N, exp, rtol=1e-14)
    assert np.all(N[:, :dim + 1, :] == 0)                  # mass and momentum are collision invariants
    # N = N~ - Lambda q (eq. 10)
    lam = physics.stiff_mask(dim)[None, :, None] / tau
    assert np.allclose(N, physics.N_tilde(dim, q, tau) - lam * q, rtol=1e-14)
    # N(q_eq) = 0 (L158)
    rho = rng.uniform(0.9, 1.1, size=5); u = rng.uniform(-0.2, 0.2, size=(5, dim))
    qe = physics.equilibrium_state(dim, rho, u, 1.7)[:, :, None]
    assert np.abs(physics.N_full(dim, qe, tau)).max() < 1e-13
    assert np.allclose(qe[:, 1, 0] * np.sqrt(1.7), rho * u[:, 0])     # rho u = sqrt(RT) q2 (L47)


def test_equilibrium_has_zero_deviatoric_stress():
    """sigma_11 = -RT(sqrt2 q5 - q2^2/q1) etc. vanish at equilibrium — pins the sqrt2 normalisation."""
    q = physics.equilibrium_state(2, np.array([1.3]), np.array([[0.3, -0.2]]), 2.0)[0]
    q1, q2, q3, q4, q5, q6 = q
    assert abs(np.sqrt(2) * q5 - q2 ** 2 / q1) < 1e-15
    assert abs(np.sqrt(2) * q6 - q3 ** 2 / q1) < 1e-15
    assert abs(q4 - q2 * q3 / q1) < 1e-15


@pytest.mark.parametrize("dim", [2, 3])
def test_upwind_split(dim):
    """eq. 7: A_n = A_n^+ + A_n^-, A^- negative semidefinite, A^+ positive semidefinite; and the closed form the
    library uses, |A_n| = c (a A^2 + b A^4) with a = (9-sqrt3)/6, b = (sqrt3-3)/6 (exact on the spectrum)."""
    rng = np.random.default_rng(8)
    c = 1.3
    n = rng.standard_normal((6, dim)); n /= np.linalg.norm(n, axis=1)[:, None]
    An = physics.normal_matrix(dim, c, n)
    Am = physics.upwind_minus(An)
    Ap = An - Am
    assert np.all(np.linalg.eigvalsh(Am) < 1e-13) and np.all(np.linalg.eigvalsh(Ap) > -1e-13)
    absA = Ap - Am
    Ah = An / c
    a, b = (9 - np.sqrt(3)) / 6, (np.sqrt(3) - 3) / 6
    closed = c * (a * Ah @ Ah + b * Ah @ Ah @ Ah @ Ah)
    assert np.abs(absA - closed).max() < 1e-13
