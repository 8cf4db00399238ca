"""Cubature-projected nonlinear relaxation P N~(I q) (oracle; test infrastructure only).

PAPER.md:L84-86: "To evaluate the integral terms containing the nonlinear term N(q^e), we use a cubature based
integration to reduce aliasing errors.  We select a nodal set of N_c cubature nodes on the reference element and
associated weights w_i^c ... map to the reference element with an interpolation operator I_ij = phi_j(x_i^c)";
L98-107 (eqs. 8-9): the term  M^-1 I^T diag(w) N(I q) = P N(I q),  P = M^-1 I^T diag(w)  (L103);
L197 (cubature kernel): interpolate with I, evaluate the nonlinear term at the cubature nodes, project with P.

Readings (R8, R20):
  * eq. 9 prints "J^e P N(I q)".  P as defined on L103 contains (M^e)^-1 = (J^e M^)^-1 while the integral over D^e
    carries J^e, so the two cancel: on the reference element P = M^^-1 I^T diag(w) and no J appears.
  * the paper fixes neither the rule nor N_c.  Taken here: the conical-product Gauss-Jacobi rule of
    oracle/quadrature.py, exact to total degree 3N (a product of three degree-N polynomials, the order of the
    rational integrand's leading terms).
  * SARK integrates -Lambda q exactly (L113-117), so only N~ (L115) goes through the cubature; the linear part would
    be reproduced exactly anyway (P I = identity for a rule exact to degree 2N).

This is SURVEY.md 8(f) NEXT-1; collocation at the interpolation nodes (I = P = identity) stays the default (R8).
Pinned in tests/test_oracle_cubature.py.
"""
import numpy as np

from . import physics as _physics
from .quadrature import simplex_rule


def cubature_degree(N):
    return 3 * N


class Cubature:
    """Points, weights, interpolation matrix I [Nc, Np] and projection P [Np, Nc] of a ReferenceElement."""

    def __init__(self, ref, degree=None):
        self.degree = cubature_degree(ref.N) if degree is None else degree
        self.x, self.w = simplex_rule(ref.dim, self.degree)          # L84: cubature nodes and weights
        self.Nc = self.w.size
        self.I = np.asarray(ref.lagrange(self.x), dtype=np.float64)  # L86: I_ij = phi_j(x_i^c)
        self.P = ref.Minv @ self.I.T @ np.diag(self.w)               # L103: P = M^-1 I^T diag(w)


def relaxation(cub, dim, q, tau):
    """P N~(I q) for q[K, Nf, Np] -> [K, Nf, Np] (eq. 9, last term; L197)."""
    qc = np.einsum("cj,kfj->kfc", cub.I, q)                          # interpolate to the cubature nodes
    nc = _physics.N_tilde(dim, qc, tau)                              # nonlinear term at the cubature nodes
    return np.einsum("ic,kfc->kfi", cub.P, nc)                       # project back


def relaxation_abs(cub, dim, q, tau):
    """Bound on the absolute values of the terms summed by ``relaxation`` (R15): |P| applied to the
    nonlinear term evaluated on |I||q| with the true interpolated density in the denominator, scaled by the
    conditioning of that density's interpolation sum."""
    qc = np.einsum("cj,kfj->kfc", cub.I, q)
    ac = np.einsum("cj,kfj->kfc", np.abs(cub.I), np.abs(q))
    aq = ac.copy()
    aq[:, 0, :] = np.abs(qc[:, 0, :])
    na = np.abs(_physics.N_tilde(dim, aq, tau)) * (ac[:, :1, :] / np.abs(qc[:, :1, :]))
    return np.einsum("ic,kfc->kfi", np.abs(cub.P), na)
