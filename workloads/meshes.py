"""Seeded, synthetic mesh generators shared by the tests, bench.py, the oracle-side tests and the CUDA-side tests.

This module holds NONE of the method's arithmetic: it only produces inputs (vertex coordinates, element-to-vertex
tables, periodic vertex identification, boundary tags, damping profiles).  Neither oracle/ nor the CUDA package
imports it; tests and bench.py hand its outputs to both.

All meshes are straight-sided, conforming, positively oriented simplices.  They stand in for the
paper's meshes, which are not available.
"""
import itertools

import numpy as np


def _morton_order(shape):
    """Cells of an n-d grid in Z-order (bit interleave), so consecutive elements are spatial neighbours."""
    grids = np.meshgrid(*[np.arange(n) for n in shape], indexing="ij")
    idx = [g.ravel().astype(np.uint64) for g in grids]
    nbits = max(int(np.ceil(np.log2(max(shape)))), 1)
    code = np.zeros(idx[0].shape, dtype=np.uint64)
    nd = len(shape)
    for b in range(nbits):
        for d in range(nd):
            code |= ((idx[d] >> np.uint64(b)) & np.uint64(1)) << np.uint64(b * nd + d)
    order = np.argsort(code, kind="stable")
    return [i[order].astype(np.int64) for i in idx]


def periodic_square(n, lo=0.0, hi=1.0, periodic=True, morton=True):
    """[lo,hi]^2, n x n quads, each split along the same diagonal into two CCW triangles (2 n^2 elements).

    Returns X0[(n+1)^2, 2], EToV[2n^2, 3], vertex_equiv[(n+1)^2] (or None)."""
    xs = np.linspace(lo, hi, n + 1)
    vid = lambda i, j: i + (n + 1) * j
    X0 = np.array([[xs[i], xs[j]] for j in range(n + 1) for i in range(n + 1)])
    if morton:
        ci, cj = _morton_order((n, n))
    else:
        cj, ci = [a.ravel() for a in np.meshgrid(np.arange(n), np.arange(n), indexing="ij")]
    tris = []
    for i, j in zip(ci, cj):
        a, b, c, d = vid(i, j), vid(i + 1, j), vid(i + 1, j + 1), vid(i, j + 1)
        tris.append((a, b, c))
        tris.append((a, c, d))
    EToV = np.array(tris, dtype=np.int32)
    equiv = None
    if periodic:
        equiv = np.array([vid(i % n, j % n) for j in range(n + 1) for i in range(n + 1)], dtype=np.int32)
    return X0, EToV, equiv


def periodic_cube(n, lo=0.0, hi=1.0, periodic=True, morton=True):
    """[lo,hi]^3, n^3 hexes, each split into the 6 Kuhn tetrahedra that share the hex's main diagonal.

    The split is translation invariant, hence conforming and periodic-conforming.  Vertices of every tet are ordered
    so that the Jacobian is positive.  Returns X0[(n+1)^3, 3], EToV[6 n^3, 4], vertex_equiv or None."""
    xs = np.linspace(lo, hi, n + 1)
    m = n + 1
    vid = lambda i, j, k: i + m * (j + m * k)
    kk, jj, ii = np.meshgrid(np.arange(m), np.arange(m), np.arange(m), indexing="ij")
    X0 = np.stack([xs[ii.ravel()], xs[jj.ravel()], xs[kk.ravel()]], axis=1)
    if morton:
        ci, cj, ck = _morton_order((n, n, n))
    else:
        ck, cj, ci = [a.ravel() for a in np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")]
    unit = np.eye(3, dtype=np.int64)
    perms = list(itertools.permutations(range(3)))

    def parity(p):
        inv = sum(1 for a in range(3) for b in range(a + 1, 3) if p[a] > p[b])
        return inv % 2

    # per permutation: the 4 corner offsets walked along the axes in that order
    offs = []
    for p in perms:
        o = [np.zeros(3, dtype=np.int64)]
        for a in p:
            o.append(o[-1] + unit[a])
        o = np.array(o)
        if parity(p) == 1:
            o = o[[0, 2, 1, 3]]
        offs.append(o)
    offs = np.array(offs)                                      # [6, 4, 3]
    base = np.stack([ci, cj, ck], axis=1)                      # [n^3, 3]
    corners = base[:, None, None, :] + offs[None, :, :, :]     # [n^3, 6, 4, 3]
    EToV = (corners[..., 0] + m * (corners[..., 1] + m * corners[..., 2])).reshape(-1, 4).astype(np.int32)
    equiv = None
    if periodic:
        equiv = (ii.ravel() % n + m * ((jj.ravel() % n) + m * (kk.ravel() % n))).astype(np.int32)
    return X0, EToV, equiv


def naca00_halfthickness(x, thickness=0.12):
    """NACA 00xx half-thickness polynomial with the closed trailing edge coefficient (-0.1036)."""
    return 5.0 * thickness * (0.2969 * np.sqrt(x) - 0.1260 * x - 0.3516 * x ** 2 + 0.2843 * x ** 3 - 0.1036 * x ** 4)


def airfoil_ogrid(ntheta=300, nr=100, R=20.0, pml_width=2.0, sigma_max=10.0, thickness=0.12):
    """O-grid of 2*ntheta*nr straight-sided triangles around a NACA 00xx profile of chord 1 (config 3).

    Inner ring: vertices on the airfoil, cosine-spaced; outer ring: circle of radius R about the mid-chord; rings in
    between blend geometrically.  Tags: 1 (wall) on the airfoil, 2 (far field) on the outer circle.  pml_sigma > 0
    for elements whose centroid radius exceeds R - pml_width (quadratic ramp, same value for both components).
    Returns X0, EToV, EToB[K,3] int8, pml_sigma[K,2], centre(2,)."""
    centre = np.array([0.5, 0.0])
    th = 2.0 * np.pi * np.arange(ntheta) / ntheta
    # airfoil point for parameter theta: x = (1+cos th)/2, upper surface for th in (0,pi), lower for (pi,2pi)
    xa = 0.5 * (1.0 + np.cos(th))
    ya = naca00_halfthickness(xa, thickness) * np.where(np.sin(th) >= 0, 1.0, -1.0)
    inner = np.stack([xa, ya], axis=1)
    outer = centre[None, :] + R * np.stack([np.cos(th), np.sin(th)], axis=1)
    # geometric radial stretching s_j in [0,1]
    ratio = 1.06
    s = np.cumsum(np.concatenate([[0.0], ratio ** np.arange(nr)]))
    s = s / s[-1]
    X0 = np.empty(((nr + 1) * ntheta, 2))
    for j in range(nr + 1):
        # blend exponent keeps the first layers body-fitted and the last ones circular
        X0[j * ntheta:(j + 1) * ntheta] = (1.0 - s[j]) * inner + s[j] * outer
    vid = lambda i, j: (i % ntheta) + ntheta * j
    tris, tags = [], []
    for j in range(nr):
        for i in range(ntheta):
            a, b, c, d = vid(i, j), vid(i, j + 1), vid(i + 1, j + 1), vid(i + 1, j)
            # (a,b,c,d) runs radially outwards first: orientation fixed below by a signed-area test
            tris.append((a, d, c)); tags.append((1 if j == 0 else 0, 0, 0))
            tris.append((a, c, b)); tags.append((0, 2 if j == nr - 1 else 0, 0))
    EToV = np.array(tris, dtype=np.int32)
    EToB = np.array(tags, dtype=np.int8)
    # orientation: make every triangle CCW, permuting tags consistently (faces: v1v2, v2v3, v3v1)
    P = X0[EToV]
    area = 0.5 * ((P[:, 1, 0] - P[:, 0, 0]) * (P[:, 2, 1] - P[:, 0, 1]) - (P[:, 2, 0] - P[:, 0, 0]) * (P[:, 1, 1] - P[:, 0, 1]))
    flip = area < 0
    EToV[flip] = EToV[flip][:, [0, 2, 1]]
    EToB[flip] = EToB[flip][:, [2, 1, 0]]
    rc = np.sqrt(np.sum((X0[EToV].mean(axis=1) - centre[None, :]) ** 2, axis=1))
    u = np.clip((rc - (R - pml_width)) / pml_width, 0.0, 1.0)
    sig = sigma_max * u ** 2
    pml_sigma = np.stack([sig, sig], axis=1)
    return X0, EToV, EToB, pml_sigma, centre


def _inside_body(p, length=1.0, half_height=0.14, half_width=0.10):
    """Ellipsoid of length 1 with the nose at x = 0 (config 5 stand-in for the fish body); the
    default half-axes are the maxima of the paper's profiles R(x), r(x) (eq. 22): 0.14 L and ~0.10 L.  A thinner body
    (round 1 used 0.10 / 0.06) contains no hex centre of the full-size 0.12-wide grid: the wall would vanish."""
    return ((p[..., 0] - 0.5 * length) / (0.5 * length)) ** 2 + (p[..., 1] / half_height) ** 2 + (p[..., 2] / half_width) ** 2 < 1.0


def swimmer_box(nx=100, ny=50, nz=50, lo=(-4.0, -3.0, -3.0), hi=(8.0, 3.0, 3.0), pml_width=0.5, sigma_max=10.0,
                half_height=0.14, half_width=0.10):
    """Box of nx*ny*nz hexes x 6 Kuhn tets with the hexes whose centre lies inside the ellipsoidal body removed
    (stair-step body surface: no mesher is available; DESIGN.md input recipe, config 5).

    Tags: 1 (wall) on faces exposed by the removal, 2 (far field) on the outer box faces.  pml_sigma[K,3]: in a shell
    of width pml_width on all six outer faces, per direction, quadratic ramp.
    Returns X0, EToV, EToB[K,4] int8, pml_sigma[K,3]."""
    lo, hi = np.array(lo, float), np.array(hi, float)
    n = (nx, ny, nz)
    m = (nx + 1, ny + 1, nz + 1)
    xs = [np.linspace(lo[d], hi[d], m[d]) for d in range(3)]
    vid = lambda i, j, k: i + m[0] * (j + m[1] * k)
    kk, jj, ii = np.meshgrid(np.arange(m[2]), np.arange(m[1]), np.arange(m[0]), indexing="ij")
    X0 = np.stack([xs[0][ii.ravel()], xs[1][jj.ravel()], xs[2][kk.ravel()]], axis=1)
    ci, cj, ck = _morton_order(n)
    centre = np.stack([0.5 * (xs[0][ci] + xs[0][ci + 1]), 0.5 * (xs[1][cj] + xs[1][cj + 1]),
                       0.5 * (xs[2][ck] + xs[2][ck + 1])], axis=1)
    keep = ~_inside_body(centre, half_height=half_height, half_width=half_width)
    ci, cj, ck = ci[keep], cj[keep], ck[keep]
    unit = np.eye(3, dtype=np.int64)
    offs = []
    for p in itertools.permutations(range(3)):
        o = [np.zeros(3, dtype=np.int64)]
        for a in p:
            o.append(o[-1] + unit[a])
        o = np.array(o)
        inv = sum(1 for a in range(3) for b in range(a + 1, 3) if p[a] > p[b])
        if inv % 2 == 1:
            o = o[[0, 2, 1, 3]]
        offs.append(o)
    offs = np.array(offs)
    base = np.stack([ci, cj, ck], axis=1)
    corners = base[:, None, None, :] + offs[None, :, :, :]
    EToV = (corners[..., 0] + m[0] * (corners[..., 1] + m[1] * corners[..., 2])).reshape(-1, 4).astype(np.int32)
    K = EToV.shape[0]
    # boundary tags: a face is a boundary face iff its sorted vertex triple occurs once
    FV = np.array([[0, 1, 2], [0, 1, 3], [1, 2, 3], [0, 2, 3]])
    fkey = np.sort(EToV[:, FV], axis=2).reshape(K * 4, 3).astype(np.int64)
    code = fkey[:, 0] + X0.shape[0] * (fkey[:, 1] + X0.shape[0] * fkey[:, 2])
    _, inv, cnt = np.unique(code, return_inverse=True, return_counts=True)
    single = (cnt[inv] == 1).reshape(K, 4)
    fc = X0[EToV[:, FV]].mean(axis=2)                          # face centroids [K,4,3]
    eps = 1e-9
    on_outer = np.zeros((K, 4), dtype=bool)
    for d in range(3):
        on_outer |= (np.abs(fc[..., d] - lo[d]) < eps) | (np.abs(fc[..., d] - hi[d]) < eps)
    EToB = np.zeros((K, 4), dtype=np.int8)
    EToB[single & on_outer] = 2
    EToB[single & ~on_outer] = 1
    ec = X0[EToV].mean(axis=1)
    pml_sigma = np.zeros((K, 3))
    for d in range(3):
        dist = np.minimum(ec[:, d] - lo[d], hi[d] - ec[:, d])
        u = np.clip((pml_width - dist) / pml_width, 0.0, 1.0)
        pml_sigma[:, d] = sigma_max * u ** 2
    return X0, EToV, EToB, pml_sigma
