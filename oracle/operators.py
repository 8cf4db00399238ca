"""Reference-element operators (oracle; test infrastructure only).

Written exactly as PAPER.md:L94 defines them, with integrals evaluated by exact quadrature (oracle/quadrature.py):

    M_ij   = int_D^ l_j l_i                 (mass)
    M^f_ij = int_face l_j l_i               (surface mass of face f, on the face's own reference simplex of measure 2)
    S^a_ij = int_D^ l_i d l_j / d a         (stiffness in the reference direction a = r, s, t; see note)
    D_a    = M^-1 S^a,  LIFT = M^-1 M^f

l_i are the Lagrange polynomials of the Warp & Blend nodes (L75).  They are evaluated as l(x) = V^-T phi(x) with the
plain product-Legendre basis phi_abc = P_a(r) P_b(s) P_c(t), a+b+c <= N (any basis of P_N gives the same l_i).

Note on S: L94 prints "S = int phi_j d phi_i/dx"; for D = M^-1 S to differentiate the interpolant (as eq. 9 uses it)
the derivative must fall on the trial function l_j, which is what is coded.  The test pins D against the analytic
derivative of every monomial, and against V_a V^-1, so the reading cannot be off by a transpose.

The library (csrc/) builds its operators another way (orthonormal Koornwinder Vandermonde, M = (V V^T)^-1); the two
share nothing and are compared to 1e-12 in tests/test_host_operators.py.
"""
import numpy as np
from numpy.polynomial import legendre as npleg

from . import nodes as _nodes
from .quadrature import simplex_rule

# Local vertex numbers of each face.  2-D: f1 v1->v2, f2 v2->v3, f3 v3->v1.
# 3-D: f1 t=-1 (v1,v2,v3), f2 s=-1 (v1,v2,v4), f3 r+s+t=-1 (v2,v3,v4), f4 r=-1 (v1,v3,v4).
FACE_VERTS = {
    2: np.array([[0, 1], [1, 2], [2, 0]]),
    3: np.array([[0, 1, 2], [0, 1, 3], [1, 2, 3], [0, 2, 3]]),
}


def _exponents(dim, N):
    if dim == 1:
        return [(a,) for a in range(N + 1)]
    if dim == 2:
        return [(a, b) for a in range(N + 1) for b in range(N + 1 - a)]
    return [(a, b, c) for a in range(N + 1) for b in range(N + 1 - a) for c in range(N + 1 - a - b)]


XP = np.longdouble     # the element matrices are accumulated in extended precision and rounded once to fp64


def _leg(n, x, deriv=0):
    c = np.zeros(n + 1)
    c[n] = 1.0
    if deriv:
        c = npleg.legder(c, deriv)
    return npleg.legval(np.asarray(x, dtype=XP), c.astype(XP))


def _inverse(A):
    """A^-1 in extended precision: fp64 LAPACK inverse, then two Newton-Schulz corrections X <- X + X (I - A X)."""
    A = np.asarray(A, dtype=XP)
    X = np.linalg.inv(A.astype(np.float64)).astype(XP)
    eye = np.eye(A.shape[0], dtype=XP)
    for _ in range(3):
        X = X + X @ (eye - A @ X)
    return X


def basis(dim, N, x):
    """phi[npts, Np] of the product-Legendre basis at points x[npts, dim]."""
    ex = _exponents(dim, N)
    out = np.empty((x.shape[0], len(ex)), dtype=XP)
    for m, e in enumerate(ex):
        v = np.ones(x.shape[0], dtype=XP)
        for d in range(dim):
            v = v * _leg(e[d], x[:, d])
        out[:, m] = v
    return out


def basis_grad(dim, N, x, a):
    """d phi / d x_a [npts, Np]."""
    ex = _exponents(dim, N)
    out = np.empty((x.shape[0], len(ex)), dtype=XP)
    for m, e in enumerate(ex):
        v = np.ones(x.shape[0], dtype=XP)
        for d in range(dim):
            v = v * _leg(e[d], x[:, d], deriv=1 if d == a else 0)
        out[:, m] = v
    return out


class ReferenceElement:
    """All constant per-(dim, N) data of the discretisation."""

    def __init__(self, dim, N, alpha=None):
        self.dim, self.N = dim, N
        self.Nfaces = dim + 1
        self.lattice = _nodes.lattice(dim, N)                       # [Np, dim+1] integers
        self.lam = _nodes.warp_blend_barycentric(dim, N, alpha)     # [Np, dim+1]; L192 interpolation matrix
        self.x = self.lam @ _nodes.REF_VERTICES[dim]                # [Np, dim]
        self.Np = self.x.shape[0]
        V = basis(dim, N, self.x)
        self.V = V
        invV = _inverse(V)
        self.invV = invV

        def lagrange(pts):          # l_j(pts): [npts, Np], extended precision
            return basis(dim, N, pts) @ invV

        def lagrange_grad(pts, a):
            return basis_grad(dim, N, pts, a) @ invV

        self.lagrange = lagrange
        self.lagrange_grad = lagrange_grad

        # --- volume matrices, exact quadrature of degree 2N (L94)
        xq, wq = simplex_rule(dim, 2 * N)
        wq = wq.astype(XP)
        L = lagrange(xq)
        M = L.T @ (wq[:, None] * L)
        S = [L.T @ (wq[:, None] * lagrange_grad(xq, a)) for a in range(dim)]
        Minv = _inverse(M)
        self.M = M.astype(np.float64)
        self.S = [s.astype(np.float64) for s in S]
        self.Minv = Minv.astype(np.float64)
        self.D = [(Minv @ s).astype(np.float64) for s in S]          # L103
        self.w = M.sum(axis=0).astype(np.float64)                    # nodal quadrature weights 1^T M

        # --- faces
        fv = FACE_VERTS[dim]
        self.face_verts = fv
        self.fmask = []
        for f in range(self.Nfaces):
            opposite = [v for v in range(dim + 1) if v not in fv[f]][0]
            self.fmask.append(np.nonzero(self.lattice[:, opposite] == 0)[0])
        self.fmask = np.array(self.fmask)                            # [Nfaces, Nfp], ascending node index
        self.Nfp = self.fmask.shape[1]

        # surface mass of each face, on the face's reference (dim-1)-simplex of measure 2 (L94), then LIFT (L103)
        uq, wuq = simplex_rule(dim - 1, 2 * N)
        vref = _nodes.REF_VERTICES[dim]
        fref = _nodes.REF_VERTICES[dim - 1]                          # vertices of the face's reference simplex
        wuq = wuq.astype(XP)
        self.Mf = []
        LIFT = np.zeros((self.Np, self.Nfaces * self.Nfp))
        for f in range(self.Nfaces):
            # barycentric coordinates of uq in the face simplex, then map to the volume reference coordinates
            A = np.vstack([fref.T, np.ones(dim)])                    # [dim, dim]
            lamf = np.linalg.solve(A, np.vstack([uq.T, np.ones(uq.shape[0])])).T   # [nq, dim]
            pts = lamf @ vref[fv[f]]
            Lf = lagrange(pts)                                       # [nq, Np]
            Mf = Lf.T @ (wuq[:, None] * Lf)                          # [Np, Np], zero off the face
            self.Mf.append(Mf.astype(np.float64))
            LIFT[:, f * self.Nfp:(f + 1) * self.Nfp] = (Minv @ Mf)[:, self.fmask[f]].astype(np.float64)
        self.LIFT = LIFT

        # lattice tuple -> node index (used by the face matching in mesh.py)
        self.node_of = {tuple(int(v) for v in row): i for i, row in enumerate(self.lattice)}
