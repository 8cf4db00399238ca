"""Pins for oracle/quadrature.py, oracle/nodes.py, oracle/operators.py against closed forms (no GPU).

Nothing here re-types an oracle formula: quadrature is pinned by Dirichlet's integral formula, nodes by the known
Legendre-Gauss-Lobatto abscissae and by symmetry, D / M / LIFT by analytic calculus on monomials.
"""
import itertools
from math import factorial

import numpy as np
import pytest

from oracle import nodes
from oracle.operators import FACE_VERTS, ReferenceElement
from oracle.quadrature import simplex_rule

PAIRS = [(2, 1), (2, 2), (2, 3), (2, 4), (2, 5), (3, 1), (3, 2), (3, 3), (3, 4)]


def unit_monomial_integral(dim, expo):
    """int over the reference simplex of prod ((1+x_d)/2)^e_d = 2^dim * prod e_d! / (sum e + dim)!  (Dirichlet)."""
    num = 1
    for e in expo:
        num *= factorial(e)
    return 2.0 ** dim * num / factorial(sum(expo) + dim)


def monomials(dim, deg):
    return [e for e in itertools.product(range(deg + 1), repeat=dim) if sum(e) <= deg]


def mono(x, e):
    v = np.ones(x.shape[0])
    for d, p in enumerate(e):
        v = v * ((1.0 + x[:, d]) / 2.0) ** p
    return v


def dmono(x, e, a):
    v = np.ones(x.shape[0])
    for d, p in enumerate(e):
        if d == a:
            v = v * (0.5 * p * ((1.0 + x[:, d]) / 2.0) ** (p - 1) if p > 0 else 0.0)
        else:
            v = v * ((1.0 + x[:, d]) / 2.0) ** p
    return v


@pytest.mark.parametrize("dim", [1, 2, 3])
@pytest.mark.parametrize("deg", [1, 4, 8])
def test_quadrature_exact_on_monomials(dim, deg):
    x, w = simplex_rule(dim, deg)
    assert np.all(w > 0)
    for e in monomials(dim, deg):
        assert abs(w @ mono(x, e) - unit_monomial_integral(dim, e)) < 5e-15


def test_lgl_points_known_values():
    # Legendre-Gauss-Lobatto abscissae (Abramowitz & Stegun 25.4.32): N=3: +-1, +-1/sqrt5; N=4: 0, +-sqrt(3/7), +-1
    assert np.allclose(nodes.lgl_points(3), [-1, -1 / np.sqrt(5), 1 / np.sqrt(5), 1], atol=1e-15)
    assert np.allclose(nodes.lgl_points(4), [-1, -np.sqrt(3 / 7), 0, np.sqrt(3 / 7), 1], atol=1e-15)
    assert np.allclose(nodes.lgl_points(2), [-1, 0, 1], atol=1e-15)


@pytest.mark.parametrize("dim,N", PAIRS)
def test_nodes_symmetric_and_lgl_on_edges(dim, N):
    lam = nodes.warp_blend_barycentric(dim, N)
    Np = lam.shape[0]
    assert Np == factorial(N + dim) // (factorial(N) * factorial(dim))
    assert np.allclose(lam.sum(axis=1), 1.0, atol=1e-15)
    assert lam.min() > -1e-15
    # the set is invariant under every permutation of the vertices
    key = lambda L: sorted(tuple(np.round(row, 12)) for row in L)
    base = key(lam)
    for p in itertools.permutations(range(dim + 1)):
        assert key(lam[:, p]) == base
    # nodes on the edge v0-v1 are the LGL points
    lat = nodes.lattice(dim, N)
    on_edge = np.all(lat[:, 2:] == 0, axis=1)
    rho = np.sort(lam[on_edge, 1] - lam[on_edge, 0])
    assert np.allclose(rho, nodes.lgl_points(N), atol=1e-14)
    # lattice order: vertex-1 index fastest
    assert tuple(lat[0]) == (N,) + (0,) * dim and tuple(lat[1])[1] == 1


def test_faces_of_3d_set_are_the_2d_sets():
    """3-D nodes restricted to a face = 2-D Warp & Blend set with the 3-D alpha."""
    for N in (3, 4):
        lam3 = nodes.warp_blend_barycentric(3, N)
        lat3 = nodes.lattice(3, N)
        face = lat3[:, 3] == 0
        lam2 = nodes.warp_blend_barycentric(2, N, alpha=nodes.ALPHA_3D[N])
        a = sorted(tuple(np.round(r[:3], 12)) for r in lam3[face])
        b = sorted(tuple(np.round(r, 12)) for r in lam2)
        assert a == b
        interior = np.all(lat3 > 0, axis=1)
        if N == 4:
            assert np.allclose(lam3[interior], 0.25)
        else:
            assert not interior.any()


@pytest.mark.parametrize("dim,N", PAIRS)
def test_D_differentiates_monomials(dim, N, refs):
    ref = refs(dim, N)
    for e in monomials(dim, N):
        for a in range(dim):
            err = np.abs(ref.D[a] @ mono(ref.x, e) - dmono(ref.x, e, a)).max()
            assert err < 2e-13, (e, a, err)
    # and nothing more: a degree N+1 monomial is NOT differentiated exactly (D is not accidentally something else)
    e = (N + 1,) + (0,) * (dim - 1)
    assert np.abs(ref.D[0] @ mono(ref.x, e) - dmono(ref.x, e, 0)).max() > 1e-6


@pytest.mark.parametrize("dim,N", PAIRS)
def test_mass_matrix_integrates_products(dim, N, refs):
    ref = refs(dim, N)
    assert np.allclose(ref.M, ref.M.T, atol=1e-15)
    mons = monomials(dim, N)
    for e in mons:
        assert abs(ref.w @ mono(ref.x, e) - unit_monomial_integral(dim, e)) < 1e-14
    for e1 in mons[::2]:
        for e2 in mons[::3]:
            exact = unit_monomial_integral(dim, tuple(a + b for a, b in zip(e1, e2)))
            assert abs(mono(ref.x, e1) @ ref.M @ mono(ref.x, e2) - exact) < 1e-14


@pytest.mark.parametrize("dim,N", PAIRS)
def test_stiffness_by_parts(dim, N, refs):
    """M D_a + (M D_a)^T = sum_f n_a^f M^f on the reference element (integration by parts), n^f = outward normal of
    the reference face scaled so that int_face = int over the face's reference simplex of measure 2."""
    ref = refs(dim, N)
    vref = nodes.REF_VERTICES[dim]
    for a in range(dim):
        lhs = ref.M @ ref.D[a]
        rhs = np.zeros_like(lhs)
        for f in range(dim + 1):
            P = vref[FACE_VERTS[dim][f]]
            if dim == 2:
                e = P[1] - P[0]
                n = np.array([e[1], -e[0]]) / 2.0                      # |edge|/2 * unit normal
            else:
                n = np.cross(P[1] - P[0], P[2] - P[0]) / 4.0           # area/2 * unit normal
            opp = [v for v in range(dim + 1) if v not in FACE_VERTS[dim][f]][0]
            if n @ (P[0] - vref[opp]) < 0:
                n = -n
            rhs += n[a] * ref.Mf[f]
        assert np.abs(lhs + lhs.T - rhs).max() < 1e-13


@pytest.mark.parametrize("dim,N", PAIRS)
def test_lift_reproduces_face_integrals(dim, N, refs):
    """1^T M LIFT_f g = int_refface g for every face polynomial g of degree <= N (SURVEY 8(c) check 1)."""
    ref = refs(dim, N)
    for f in range(dim + 1):
        fv = FACE_VERTS[dim][f]
        lamf = ref.lam[ref.fmask[f]][:, fv]                  # face-barycentric coordinates of the face nodes
        for e in monomials(dim - 1, N):
            # g = prod lam_{m+1}^e_m on the face; its integral over the reference face simplex (measure 2):
            # Dirichlet: (dim-1)! * prod e! / (sum e + dim - 1)! * measure
            g = np.ones(ref.Nfp)
            for m, p in enumerate(e):
                g = g * lamf[:, m + 1] ** p
            num = 1
            for p in e:
                num *= factorial(p)
            exact = 2.0 * factorial(dim - 1) * num / factorial(sum(e) + dim - 1)
            G = np.zeros(ref.Nfaces * ref.Nfp)
            G[f * ref.Nfp:(f + 1) * ref.Nfp] = g
            assert abs(ref.w @ (ref.LIFT @ G) - exact) < 1e-13


@pytest.mark.parametrize("dim,N", [(2, 3), (2, 4), (3, 3), (3, 4)])
def test_interpolation_matrix_is_barycentric(dim, N, refs):
    """the Np x Nvertices interpolation matrix reproduces any P1 function from its vertex values."""
    ref = refs(dim, N)
    vref = nodes.REF_VERTICES[dim]
    coef = np.arange(1, dim + 1) * 0.37
    f_vert = vref @ coef + 0.11
    assert np.allclose(ref.lam @ f_vert, ref.x @ coef + 0.11, atol=1e-15)
    assert ref.fmask.shape == (dim + 1, {2: N + 1, 3: (N + 1) * (N + 2) // 2}[dim])


def test_interior_orbit_of_order_4_matches_survey_values():
    """SURVEY 8(c)-S1 prints the only nodes of the four (dim, N) pairs of the configs that are not fixed by symmetry
    and the LGL edge points: the 3-node interior orbit of the 2-D N=4 set, barycentric (0.551583507555,
    0.224208246222, 0.224208246222) at alpha = 0.1001, and the same orbit on every face of the 3-D N=4 set,
    (0.551583572091, 0.224208213955, 0.224208213955) at alpha = 0.1002 (reading R10).  A wrong blend
    exponent, a dropped factor in 4 lambda_a lambda_b or another alpha moves these digits (alpha = 0 gives 0.551551)."""
    lam = nodes.warp_blend_barycentric(2, 4)
    lat = nodes.lattice(2, 4)
    interior = lam[np.all(lat > 0, axis=1)]
    assert interior.shape == (3, 3)
    for row in interior:
        assert np.allclose(np.sort(row), [0.224208246222, 0.224208246222, 0.551583507555], rtol=0, atol=2e-12)
    lam3 = nodes.warp_blend_barycentric(3, 4)
    lat3 = nodes.lattice(3, 4)
    for face in range(4):                                    # the face opposite vertex `face`
        on_face = lat3[:, face] == 0
        inner = on_face & (np.sum(lat3 > 0, axis=1) == 3)    # not on an edge of that face
        assert inner.sum() == 3
        for row in lam3[inner]:
            assert np.allclose(np.sort(row), [0.0, 0.224208213955, 0.224208213955, 0.551583572091], rtol=0, atol=2e-12)
    # sensitivity: the pinned digits separate alpha = 0.1001 from alpha = 0 and from a blend without the square
    lam0 = nodes.warp_blend_barycentric(2, 4, alpha=0.0)
    assert abs(np.sort(lam0[np.all(lat > 0, axis=1)][0])[-1] - 0.551583507555) > 1e-5
