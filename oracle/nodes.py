"""Interpolation nodes on the reference simplex (oracle; test infrastructure only).

PAPER.md:L75 — "Lagrange polynomials interpolated at the Warp & Blend nodes [34]".  Ref. [34] (Warburton 2006) is not
in the container; what is restated here is its published construction in barycentric form:

  * start from the equispaced lattice of order N, barycentric coordinates lambda = (i_0, ..., i_d)/N;
  * the 1-D warp w(r) is the degree-N interpolant, through the N+1 equispaced points of [-1,1], of the displacement
    that carries them to the Legendre-Gauss-Lobatto points;
  * every edge (a,b) of the simplex pushes a node along the edge direction by
        4 lambda_a lambda_b * w(rho)/(1-rho^2) * (1 + (alpha*lambda_rest)^2),   rho = lambda_b - lambda_a,
    with lambda_rest = 1 - lambda_a - lambda_b; a displacement of size c along edge a->b in the edge's [-1,1]
    coordinate changes lambda_b by +c/2 and lambda_a by -c/2.

In 2-D this is the construction of [34] exactly.  In 3-D it reproduces, on every face, the 2-D Warp & Blend set of
that face (edges that do not lie in the face have lambda_a*lambda_b = 0 there) and is symmetric under all vertex
permutations; for N <= 4 the only node not on a face is the centroid (N = 4), so the set coincides with the one the
configs need.  For N >= 5 in 3-D the interior nodes are this build's extension (reading R10).

alpha: optimised blend parameters published in [34]; recalled, unverifiable here, and immaterial for N = 3
(SURVEY R10).  They are constants of the build; the library carries its own copy.
"""
import numpy as np
from scipy.special import roots_jacobi

ALPHA_2D = {1: 0.0, 2: 0.0, 3: 1.4152, 4: 0.1001, 5: 0.2751, 6: 0.9800, 7: 1.0999, 8: 1.2832}
ALPHA_3D = {1: 0.0, 2: 0.0, 3: 0.0, 4: 0.1002, 5: 1.1332, 6: 1.5608, 7: 1.3413, 8: 1.2577}

REF_VERTICES = {
    1: np.array([[-1.0], [1.0]]),
    2: np.array([[-1.0, -1.0], [1.0, -1.0], [-1.0, 1.0]]),
    3: np.array([[-1.0, -1.0, -1.0], [1.0, -1.0, -1.0], [-1.0, 1.0, -1.0], [-1.0, -1.0, 1.0]]),
}


def lgl_points(N):
    """Legendre-Gauss-Lobatto points of order N on [-1,1]: +-1 and the zeros of P_N' = zeros of P_{N-1}^{(1,1)}."""
    if N == 1:
        return np.array([-1.0, 1.0])
    x, _ = roots_jacobi(N - 1, 1.0, 1.0)
    return np.concatenate([[-1.0], np.sort(x), [1.0]])


def warp_1d(N, rho):
    """w(rho): Lagrange interpolant through the equispaced points of the LGL-minus-equispaced displacement."""
    req = np.linspace(-1.0, 1.0, N + 1)
    disp = lgl_points(N) - req
    rho = np.asarray(rho, dtype=float)
    w = np.zeros_like(rho)
    for i in range(N + 1):
        li = np.ones_like(rho)
        for j in range(N + 1):
            if j != i:
                li *= (rho - req[j]) / (req[i] - req[j])
        w += disp[i] * li
    return w


def lattice(dim, N):
    """Integer barycentric lattice, one row (i_0, ..., i_dim) per node, sum = N.

    Order: the index attached to vertex 1 runs fastest, then vertex 2, then vertex 3; i_0 = N - rest.
    """
    rows = []
    if dim == 1:
        for i in range(N + 1):
            rows.append((N - i, i))
    elif dim == 2:
        for j in range(N + 1):
            for i in range(N + 1 - j):
                rows.append((N - i - j, i, j))
    else:
        for k in range(N + 1):
            for j in range(N + 1 - k):
                for i in range(N + 1 - j - k):
                    rows.append((N - i - j - k, i, j, k))
    return np.array(rows, dtype=np.int64)


def warp_blend_barycentric(dim, N, alpha=None):
    """Barycentric coordinates lam[Np, dim+1] of the Warp & Blend nodes."""
    if alpha is None:
        alpha = {1: 0.0}.get(dim, None)
        if dim == 2:
            alpha = ALPHA_2D[N]
        elif dim == 3:
            alpha = ALPHA_3D[N]
    lat = lattice(dim, N)
    lam0 = lat.astype(float) / N
    lam = lam0.copy()
    nv = dim + 1
    for a in range(nv):
        for b in range(a + 1, nv):
            la, lb = lam0[:, a], lam0[:, b]
            rho = lb - la
            denom = 1.0 - rho * rho
            # w(rho)/(1-rho^2): w vanishes at rho = +-1, where the blend 4 la lb vanishes as well -> push 0 there
            interior = np.abs(denom) > 1e-12
            scaled = np.zeros_like(rho)
            scaled[interior] = warp_1d(N, rho[interior]) / denom[interior]
            rest = 1.0 - la - lb
            push = 4.0 * la * lb * scaled * (1.0 + (alpha * rest) ** 2)
            lam[:, b] += 0.5 * push
            lam[:, a] -= 0.5 * push
    return lam


def warp_blend_nodes(dim, N, alpha=None):
    """Reference coordinates x[Np, dim] of the nodes, lattice order."""
    lam = warp_blend_barycentric(dim, N, alpha)
    return lam @ REF_VERTICES[dim]
