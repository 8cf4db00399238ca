"""Geometric factors of affine simplices (oracle; test infrastructure only).

PAPER.md:L88-92: G^e = [x_r x_s; y_r y_s], J^e = det G^e; L193: "the elemental Jacobian, spatial derivative
matrices, and interfacial face normals" are constant per element and determined by the vertices.

With the reference simplex of oracle/nodes.py (vertices at -1/+1) the affine map is
x(xi) = sum_v lambda_v(xi) x_v, so x_r = (x_2 - x_1)/2, x_s = (x_3 - x_1)/2, x_t = (x_4 - x_1)/2.

The face quantities are computed from first principles, not from the metric identities the library uses:
  unit outward normal  = the unit vector orthogonal to the face (edge rotated by 90 degrees / cross product of two
                         face edges), oriented away from the opposite vertex;
  sJ                   = physical face measure / measure of the face's reference simplex (2 for an edge [-1,1] and for
                         the reference triangle), so that int_face g = sJ * int_refface g;
  Fscale               = sJ / J (the factor in front of LIFT once M^-1 = (J M^)^-1 is applied; L103).
"""
import numpy as np

from .operators import FACE_VERTS


def factors(dim, xv, EToV):
    """xv[Nv, dim] moved vertices, EToV[K, dim+1].

    Returns dict: J[K]; G[K, dim, dim] with G[:, d, a] = d x_d / d xi_a; Ginv[K, a, d] = d xi_a / d x_d;
    nhat[K, Nfaces, dim]; sJ[K, Nfaces]; Fscale[K, Nfaces].
    """
    X = xv[EToV]                                    # [K, dim+1, dim]
    K = X.shape[0]
    G = np.empty((K, dim, dim))
    for a in range(dim):
        G[:, :, a] = 0.5 * (X[:, a + 1, :] - X[:, 0, :])
    J = np.linalg.det(G)
    Ginv = np.linalg.inv(G)                         # rows a: (a_x, a_y, a_z)
    fv = FACE_VERTS[dim]
    Nfaces = dim + 1
    nhat = np.empty((K, Nfaces, dim))
    sJ = np.empty((K, Nfaces))
    for f in range(Nfaces):
        P = X[:, fv[f], :]                          # [K, dim, dim] the face's vertices
        opp = [v for v in range(dim + 1) if v not in fv[f]][0]
        if dim == 2:
            e = P[:, 1, :] - P[:, 0, :]
            n = np.stack([e[:, 1], -e[:, 0]], axis=1)
            measure = np.sqrt(np.sum(e * e, axis=1))            # edge length
        else:
            n = np.cross(P[:, 1, :] - P[:, 0, :], P[:, 2, :] - P[:, 0, :])
            measure = 0.5 * np.sqrt(np.sum(n * n, axis=1))      # triangle area
        # orient away from the opposite vertex
        s = np.sign(np.sum(n * (P[:, 0, :] - X[:, opp, :]), axis=1))
        n = n * s[:, None]
        nhat[:, f, :] = n / np.sqrt(np.sum(n * n, axis=1))[:, None]
        sJ[:, f] = measure / 2.0
    return dict(J=J, G=G, Ginv=Ginv, nhat=nhat, sJ=sJ, Fscale=sJ / J[:, None])
