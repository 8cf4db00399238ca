"""Quadrature on the reference simplices (oracle; test infrastructure only).

Reference simplices (the paper's reference element D^ of Fig. 1):
  dim 1: [-1, 1]                                      measure 2
  dim 2: vertices (-1,-1), (1,-1), (-1,1)             measure 2
  dim 3: vertices (-1,-1,-1), (1,-1,-1), (-1,1,-1), (-1,-1,1)   measure 4/3

The rules are conical products of Gauss-Jacobi rules (collapsed coordinates), exact for polynomials of total
degree <= ``degree``.  They exist so that the element matrices can be written exactly as PAPER.md:L94 defines them,
M_ij = int phi_j phi_i etc., with the integral evaluated by a rule that is exact for the integrand.
Pinned in tests/test_oracle_operators.py against the closed-form Dirichlet integrals of monomials.
"""
import numpy as np
from scipy.special import roots_jacobi


def simplex_rule(dim, degree):
    """Points x[nq, dim] and weights w[nq] on the reference ``dim``-simplex, exact to total degree ``degree``."""
    n = degree // 2 + 1  # n-point Gauss-Jacobi is exact to degree 2n-1 >= degree
    a, wa = roots_jacobi(n, 0.0, 0.0)
    if dim == 1:
        return a[:, None].copy(), wa.copy()
    b, wb = roots_jacobi(n, 1.0, 0.0)  # weight (1-b)
    if dim == 2:
        # r = (1+a)(1-b)/2 - 1, s = b;  dr ds = (1-b)/2 da db
        A, B = np.meshgrid(a, b, indexing="ij")
        W = np.outer(wa, wb) / 2.0
        r = (1 + A) * (1 - B) / 2 - 1
        s = B
        return np.stack([r.ravel(), s.ravel()], axis=1), W.ravel()
    if dim == 3:
        c, wc = roots_jacobi(n, 2.0, 0.0)  # weight (1-c)^2
        # r = (1+a)(1-b)(1-c)/4 - 1, s = (1+b)(1-c)/2 - 1, t = c;  dr ds dt = (1-b)(1-c)^2/8 da db dc
        A, B, C = np.meshgrid(a, b, c, indexing="ij")
        W = wa[:, None, None] * wb[None, :, None] * wc[None, None, :] / 8.0
        r = (1 + A) * (1 - B) * (1 - C) / 4 - 1
        s = (1 + B) * (1 - C) / 2 - 1
        t = C
        return np.stack([r.ravel(), s.ravel(), t.ravel()], axis=1), W.ravel()
    raise ValueError("dim must be 1, 2 or 3")
