"""Pins of oracle/forces.py (no GPU): wall-force integrals (PAPER.md:L308, L369 with L51, L53; NEXT-3).

Gauss's theorem on the closed wall surface of the synthetic bodies gives closed forms that share nothing with the
face-quadrature code: for p = p0 + a.x,  -int p n_b dS = -a V;  for sigma_ij = s0_ij + S_ijk x_k,
int sigma n_b dS = (S_ijj summed) V, with V the body's area / volume -- the polygon's shoelace area for the airfoil,
the number of removed hexes times the hex volume for the stair-step swimmer body.
"""
import numpy as np
import pytest

from oracle import forces, physics
from workloads import configs
from helpers import oracle_problem, swimmer_small


def _body_measure(name, cfg, P):
    if name == "airfoil":
        # the wall faces form a closed polygon: shoelace area from the wall edges (ordered by the face orientation)
        g = P.geometry(0.0)
        area = 0.0
        for f in range(3):
            for e in np.nonzero(P.EToB[:, f] == 1)[0]:
                v = P.EToV[e][list(P.ref.face_verts[f][:2])]
                a, b = g["xv"][v[0]], g["xv"][v[1]]
                area += 0.5 * (a[0] * b[1] - b[0] * a[1])     # fluid element is CCW, so the body is traversed clockwise
        return -area
    # swimmer: divergence theorem with the identity field x/3 over the wall triangles, independent of face quadrature
    g = P.geometry(0.0)
    vol = 0.0
    for f in range(4):
        for e in np.nonzero(P.EToB[:, f] == 1)[0]:
            v = P.EToV[e][list(P.ref.face_verts[f])]
            a, b, c = g["xv"][v[0]], g["xv"][v[1]], g["xv"][v[2]]
            nA = 0.5 * np.cross(b - a, c - a)
            nA *= np.sign(nA @ g["nhat"][e, f])               # outward from the fluid = into the body
            vol += -(a + b + c) @ nA / 9.0                    # int x.n_b dS / 3 with n_b = -n^
    return vol


@pytest.mark.parametrize("name", ["airfoil", "swimmer"])
def test_gauss_theorem_closed_forms(name, refs):
    if name == "airfoil":
        ref = refs(2, 4)
        cfg = configs.config3(ref.lam, ntheta=40, nr=8)
    else:
        ref = refs(3, 3)
        cfg = swimmer_small(ref.lam)
    dim, RT = cfg["dim"], cfg["RT"]
    P = oracle_problem(cfg, ref)
    V = _body_measure(name, cfg, P)
    assert V > 1e-3
    g = P.geometry(0.0)
    x = np.einsum("iv,kvd->kdi", ref.lam, g["xv"][P.EToV])     # node coordinates [K, dim, Np]
    rng = np.random.default_rng(199)
    a = rng.standard_normal(dim)
    S = rng.standard_normal((dim, dim, dim))
    S = 0.5 * (S + S.transpose(1, 0, 2))                      # symmetric in (i, j)
    s0 = rng.standard_normal((dim, dim)); s0 = 0.5 * (s0 + s0.T)
    Nf = physics.nfields(dim)
    q = np.zeros((cfg["K"], Nf, ref.Np))
    q[:, 0, :] = (2.0 + np.einsum("d,kdi->ki", a, x)) / RT     # p = 2 + a.x, momentum zero
    sig = s0[None, :, :, None] + np.einsum("ijd,kdn->kijn", S, x)
    for k, alpha in enumerate(physics.MULTI[dim]):             # second moments carrying sigma (L51 inverted, u = 0)
        if sum(alpha) != 2:
            continue
        nz = [d for d in range(dim) if alpha[d] > 0]
        if len(nz) == 1:
            q[:, k, :] = -sig[:, nz[0], nz[0], :] / RT / np.sqrt(2.0)
        else:
            q[:, k, :] = -sig[:, nz[0], nz[1], :] / RT
    Fp, Fv = forces.wall_force(P, q, 0.0)
    assert np.abs(Fp - (-a * V)).max() < 1e-12 * max(1.0, np.abs(a * V).max())
    assert np.abs(Fv - np.einsum("ijj->i", S) * V).max() < 1e-12 * max(1.0, V)


def test_equilibrium_has_no_viscous_force_and_uniform_pressure_no_net_force(refs):
    ref = refs(2, 4)
    cfg = configs.config3(ref.lam, ntheta=40, nr=8)
    P = oracle_problem(cfg, ref)
    Fp, Fv = forces.wall_force(P, cfg["q0"], 0.3)              # q0 = q_inf everywhere (Maxwellian, u = (0.1, 0))
    assert np.abs(Fv).max() < 1e-15 and np.abs(Fp).max() < 1e-13
    # no wall faces -> zeros
    ref1 = refs(2, 3)
    P1 = oracle_problem(configs.config1(ref1.lam, n=4), ref1)
    assert all(np.all(v == 0) for v in forces.wall_force(P1, configs.config1(ref1.lam, n=4)["q0"], 0.0))
