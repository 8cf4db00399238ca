"""Pressure and viscous force on wall faces (oracle; test infrastructure only).  SURVEY.md 8(f) NEXT-3.

PAPER.md:L308: c_D = F_D / (0.5 rho_inf u_inf^2 c); L369: C_p = F_p / (0.5 rho u^2 A), C_v = F_v / (0.5 rho u^2 A),
"the subscript p represents the pressure force contribution and v represents the viscous force contributions".
The paper does not print the surface integrals; they are the textbook traction integrals with the paper's own
macroscopic relations:

    p = rho RT = q1 RT                                                     (L53)
    sigma_11 = -RT (sqrt2 q5 - q2^2/q1),  sigma_12 = -RT (q4 - q2 q3/q1), ...   (L51; 3-D by the same rule in the
                                                                            field order of DESIGN.md reading R3)
    F_p = - int_wall p n_b dS,     F_v = int_wall sigma . n_b dS,   n_b = outward normal of the BODY = -n^

where n^ is the outward normal of the fluid element on the wall face.  The face integral uses the nodal face
quadrature of the discretisation itself: int_face g dS = sJ_f sum_m (1^T M^f)_m g_m on the face's reference simplex of
measure 2 (L94: M^ef), exact for g of degree <= N.  Reading R22.

Pinned in tests/test_oracle_forces.py: Gauss's theorem on the closed wall surface with constant and linear p and
sigma (closed forms: zero, and gradient times the body's volume), zero viscous force at equilibrium (L51).
"""
import numpy as np

from . import physics as _physics
from .rhs import WALL


def pressure_and_stress(dim, q, RT):
    """q[..., Nf, n] -> p[..., n], sigma[..., dim, dim, n] (L51, L53)."""
    p = RT * q[..., 0, :]
    sig = np.zeros(q.shape[:-2] + (dim, dim, q.shape[-1]))
    for k, alpha in enumerate(_physics.MULTI[dim]):
        if sum(alpha) != 2:
            continue
        nz = [d for d in range(dim) if alpha[d] > 0]
        if len(nz) == 1:
            i = j = nz[0]
            m = np.sqrt(2.0) * q[..., k, :]
        else:
            i, j = nz
            m = q[..., k, :]
        s = -RT * (m - q[..., 1 + i, :] * q[..., 1 + j, :] / q[..., 0, :])
        sig[..., i, j, :] = s
        sig[..., j, i, :] = s
    return p, sig


def face_weights(ref):
    """(1^T M^f) restricted to the nodes of each face: [Nfaces, Nfp]."""
    return np.array([ref.Mf[f].sum(axis=0)[ref.fmask[f]] for f in range(ref.Nfaces)])


def wall_force(problem, q, t, tag=WALL):
    """(F_p[dim], F_v[dim]) on the faces tagged ``tag`` at time t."""
    ref, dim = problem.ref, problem.dim
    g = problem.geometry(t)
    wf = face_weights(ref)
    Fp, Fv = np.zeros(dim), np.zeros(dim)
    if problem.EToB is None:
        return Fp, Fv
    for f in range(ref.Nfaces):
        elems = np.nonzero(problem.EToB[:, f] == tag)[0]
        if elems.size == 0:
            continue
        qf = q[elems][:, :, ref.fmask[f]]                      # [n, Nf, Nfp]
        p, sig = pressure_and_stress(dim, qf, problem.RT)
        nb = -g["nhat"][elems, f, :]                           # outward normal of the body
        sJ = g["sJ"][elems, f]
        Fp += -np.einsum("e,m,em,ed->d", sJ, wf[f], p, nb)
        Fv += np.einsum("e,m,eijm,ej->i", sJ, wf[f], sig, nb)
    return Fp, Fv
