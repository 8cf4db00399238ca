"""Pins for oracle/motion.py, oracle/geometry.py, oracle/mesh.py (no GPU)."""
import numpy as np
import pytest

from oracle import geometry, mesh, motion
from oracle.operators import FACE_VERTS
from workloads import configs, meshes

LAWS = [
    (2, motion.SINES_PRODUCT, [0.05, 1.0, np.pi, np.pi, 0.0, 0.3]),
    (3, motion.SINES_PRODUCT, [0.03, 0.7, 2.0, 3.0, 1.0, 0.1, 0.2, 0.3]),
    (2, motion.SINES_CROSS, [0.04, 1.3, 2 * np.pi, 0.4]),
    (3, motion.SINES_CROSS, [0.03, 1.0, 2 * np.pi, 0.0]),
    (2, motion.PLUNGE_BLEND, [0.25, np.pi, 0.2, 0.8, 1, 0.5, 0.5]),
    (3, motion.PLUNGE_BLEND, [0.1, 2.0, 0.1, 0.9, 2, 0.4, 0.5, 0.6]),
    (3, motion.CARANGIFORM, [0.02, -0.0825, 0.1625, 2 * np.pi / 0.95, 2 * np.pi, 0.5, 10.0, 1.0, 1, 1e-16]),
]


@pytest.mark.parametrize("dim,kind,params", LAWS)
@pytest.mark.parametrize("t", [0.0, 0.37, 1.6])
def test_velocity_is_time_derivative_of_position(dim, kind, params, t):
    rng = np.random.default_rng(5)
    X0 = rng.uniform(-0.5, 1.5, size=(200, dim))
    eps = 1e-5
    xp, _ = motion.vertices(kind, params, X0, t + eps)
    xm, _ = motion.vertices(kind, params, X0, t - eps)
    _, v = motion.vertices(kind, params, X0, t)
    if t == 0.0 and kind == motion.CARANGIFORM:
        xm = X0       # ramp is one-sided at t = 0: S = S' = 0
        assert np.abs(v).max() == 0.0
        return
    assert np.abs((xp - xm) / (2 * eps) - v).max() < 2e-8
    x0, _ = motion.vertices(kind, params, X0, 0.0)
    assert np.abs(x0 - X0).max() < 1e-15


def test_plunge_blend_limits_and_carangiform_cut():
    X0 = np.array([[0.5, 0.0], [0.5, 1.9], [0.5, 6.0], [0.5, 10.5], [30.0, 0.0]])
    p = [0.25, np.pi, 2.0, 10.0, 1, 0.5, 0.0]
    x, v = motion.vertices(motion.PLUNGE_BLEND, p, X0, 0.5)
    d = x[:, 1] - X0[:, 1]
    assert np.allclose(d[:2], 0.25) and 0 < d[2] < 0.25 and d[3] == 0 and d[4] == 0 and np.all(x[:, 0] == X0[:, 0])
    # far from the body the Gaussian blend is cut to exactly zero -> static mesh there
    pc = [0.02, -0.0825, 0.1625, 2 * np.pi / 0.95, 2 * np.pi, 0.5, 10.0, 1.0, 1, 1e-16]
    Xf = np.array([[0.5, 0.0, 0.0], [0.5, 2.45, 0.0], [1.2, 0.1, 0.0]])
    x, v = motion.vertices(motion.CARANGIFORM, pc, Xf, 2.3)
    assert x[1, 1] == Xf[1, 1] and v[1, 1] == 0.0
    # inside the rigid core B = 1 and t > T_ramp: h = A(x~) sin(k X - w t)   (L326, L353)
    A = 0.02 - 0.0825 * 0.5 + 0.1625 * 0.25
    assert abs((x[0, 1] - Xf[0, 1]) - A * np.sin(2 * np.pi / 0.95 * 0.5 - 2 * np.pi * 2.3)) < 1e-15
    assert np.all(x[:, 0] == Xf[:, 0]) and np.all(x[:, 2] == Xf[:, 2])


@pytest.mark.parametrize("dim", [2, 3])
def test_geometry_against_direct_formulas(dim):
    rng = np.random.default_rng(11)
    if dim == 2:
        X0, EToV, _ = meshes.periodic_square(4)
    else:
        X0, EToV, _ = meshes.periodic_cube(3)
    xv = X0 + 0.03 * rng.standard_normal(X0.shape)
    g = geometry.factors(dim, xv, EToV)
    P = xv[EToV]
    # measure = J * reference measure (2 or 4/3), from the Cayley-Menger-free direct determinant of edge vectors
    E = P[:, 1:, :] - P[:, :1, :]
    vol = np.linalg.det(E) / (2 if dim == 2 else 6)
    assert np.all(g["J"] > 0)
    assert np.allclose(g["J"] * (2.0 if dim == 2 else 4.0 / 3.0), vol, rtol=1e-13)
    # closed surface: sum_f sJ_f * (reference face measure 2) * n_f = 0
    assert np.abs(np.einsum("kf,kfd->kd", g["sJ"], g["nhat"])).max() < 1e-14
    assert np.allclose(np.linalg.norm(g["nhat"], axis=2), 1.0, atol=1e-15)
    # divergence theorem with the linear field x: sum_f |face| n_f . x_face_centroid = dim * volume
    fc = np.stack([P[:, FACE_VERTS[dim][f], :].mean(axis=1) for f in range(dim + 1)], axis=1)
    flux = np.einsum("kf,kfd,kfd->k", 2.0 * g["sJ"], g["nhat"], fc)
    assert np.allclose(flux, dim * vol, rtol=1e-12)
    # metrics are the inverse of the Jacobian matrix of x(xi) = sum_v lambda_v x_v
    assert np.allclose(np.einsum("kad,kdb->kab", g["Ginv"], g["G"]), np.eye(dim)[None], atol=1e-13)
    assert np.allclose(g["G"][:, :, 0], 0.5 * (P[:, 1] - P[:, 0]))
    assert np.allclose(g["Fscale"], g["sJ"] / g["J"][:, None])


@pytest.mark.parametrize("dim", [2, 3])
def test_dJdt_equals_J_div_vG(dim):
    """For a P1 velocity on an affine element dJ/dt = J div v_G exactly; the basis of the GCL (L154)."""
    if dim == 2:
        X0, EToV, _ = meshes.periodic_square(4)
        kind, p = motion.SINES_PRODUCT, [0.05, 1.0, np.pi, np.pi, 0.0, 0.0]
    else:
        X0, EToV, _ = meshes.periodic_cube(3)
        kind, p = motion.SINES_CROSS, [0.03, 1.0, 2 * np.pi, 0.0]
    t, eps = 0.21, 1e-5
    xv, vv = motion.vertices(kind, p, X0, t)
    g = geometry.factors(dim, xv, EToV)
    Jp = geometry.factors(dim, motion.vertices(kind, p, X0, t + eps)[0], EToV)["J"]
    Jm = geometry.factors(dim, motion.vertices(kind, p, X0, t - eps)[0], EToV)["J"]
    V = vv[EToV]
    # grad of the P1 field: sum_a (dxi_a/dx_d) * dv/dxi_a, dv/dxi_a = (v_{a+1} - v_1)/2
    div = sum(g["Ginv"][:, a, d] * 0.5 * (V[:, a + 1, d] - V[:, 0, d]) for a in range(dim) for d in range(dim))
    rate = g["J"] * div
    assert np.abs(rate).max() > 1e-3 * np.abs(g["J"]).max()          # the test is not vacuous
    assert np.abs((Jp - Jm) / (2 * eps) - rate).max() < 1e-7 * np.abs(rate).max()


@pytest.mark.parametrize("which", ["square", "cube", "airfoil", "swimmer"])
def test_connectivity_partners_coincide(which, refs):
    """vmapP found through vertex permutations must be the geometrically coincident node (checked by coordinates,
    which the matching itself never uses; periodic images differ by a lattice vector)."""
    if which == "square":
        ref = refs(2, 4); X0, EToV, eq = meshes.periodic_square(4); EToB = None; L = 1.0
    elif which == "cube":
        ref = refs(3, 4); X0, EToV, eq = meshes.periodic_cube(3); EToB = None; L = 1.0
    elif which == "airfoil":
        ref = refs(2, 3); X0, EToV, EToB, _, _ = meshes.airfoil_ogrid(24, 6); eq = None; L = None
    else:
        ref = refs(3, 3); X0, EToV, EToB, _ = meshes.swimmer_box(12, 6, 6, half_height=0.8, half_width=0.8); eq = None; L = None
    c = mesh.connect(ref, EToV, eq, EToB)
    K = EToV.shape[0]
    x = configs.node_coordinates(X0, EToV, ref.lam).reshape(K * ref.Np, -1)
    d = x[c["vmapP"]] - x[c["vmapM"]]
    if L is not None:
        d = d - L * np.round(d / L)
    assert np.abs(d).max() < 1e-12
    # symmetric neighbour relation, every interior face paired exactly once
    E, F = c["EToE"], c["EToF"]
    ee = np.arange(K)[:, None].repeat(ref.Nfaces, 1)
    ff = np.arange(ref.Nfaces)[None, :].repeat(K, 0)
    assert np.all(E[E, F] == ee) and np.all(F[E, F] == ff)
    if EToB is None:
        assert np.all((E != ee) | (F != ff))
    else:
        bnd = (E == ee) & (F == ff)
        assert np.all(bnd == (EToB != 0))
        assert np.all(c["vmapP"][bnd] == c["vmapM"][bnd])
        assert (EToB == 1).sum() > 0 and (EToB == 2).sum() > 0


def test_connectivity_rejects_short_periods_and_untagged_boundaries(refs):
    X0, EToV, eq = meshes.periodic_square(2)
    with pytest.raises(mesh.MeshError):
        mesh.connect(refs(2, 2), EToV, eq)
    X0, EToV, eq = meshes.periodic_square(3, periodic=False)
    with pytest.raises(mesh.MeshError):
        mesh.connect(refs(2, 2), EToV, None, None)


def test_generated_meshes_are_positive(refs):
    for X0, EToV, dim in [meshes.periodic_square(5)[:2] + (2,), meshes.periodic_cube(3)[:2] + (3,),
                          meshes.airfoil_ogrid(40, 10)[:2] + (2,), meshes.swimmer_box(12, 6, 6)[:2] + (3,)]:
        assert np.all(geometry.factors(dim, X0, EToV)["J"] > 0)
