"""Semi-analytic Runge-Kutta (SARK4) time stepping (oracle; test infrastructure only).

PAPER.md:L111-148.  dq/dt = -Lambda q + F(q) (eq. 11), Lambda = diag(0,..,0, 1/tau,..) (L115);

    q_ni   = q_n e^{-Lambda dt_i} + dt sum_{j<i} a~_ij F_nj          (L132)
    q_n+1  = q_n e^{-Lambda dt}   + dt sum_j   b~_j  F_nj           (L134)

with dt_i = c_i dt, c = (0, 1/2, 1/2, 1) of the classic RK4 (Table 1 is blank in PAPER.md:L119; reading R4: the
printed a~, b~ have exactly the classic RK4 tableau as their gamma -> 0 limit, test_oracle_sark pins it), and
gamma = -dt/tau (L144).  Fields with Lambda = 0 use the gamma -> 0 limit, i.e. classic RK4 itself (L121, L136).

The coefficients are the formulas PRINTED at PAPER.md:L148, evaluated in 60-digit decimal arithmetic and rounded
once to fp64: in fp64 the printed forms cancel catastrophically for small |gamma| (reading R6).
F is evaluated at t_n + c_j dt on the mesh moved to that time (L152-154).
Auxiliary PML fields (reading R12) have Lambda = 0 and are advanced with the classic weights.
"""
from decimal import Decimal, getcontext

import numpy as np

from . import physics as _physics

RK4_C = (0.0, 0.5, 0.5, 1.0)
RK4_A = ((0.0, 0.0, 0.0, 0.0), (0.5, 0.0, 0.0, 0.0), (0.0, 0.5, 0.0, 0.0), (0.0, 0.0, 1.0, 0.0))
RK4_B = (1.0 / 6.0, 1.0 / 3.0, 1.0 / 3.0, 1.0 / 6.0)


def coefficients(gamma):
    """(a~[4][4], b~[4]) for the given gamma = -dt/tau, formulas of PAPER.md:L148; gamma = 0 -> classic RK4."""
    if gamma == 0.0:
        return [list(r) for r in RK4_A], list(RK4_B)
    getcontext().prec = 60
    g = Decimal(float(gamma))       # exact value of the fp64 gamma
    eh = (g / 2).exp()
    e = g.exp()
    a = [[Decimal(0)] * 4 for _ in range(4)]
    a[1][0] = (-1 + eh) / g
    a[2][0] = (4 + g + eh * (g - 4)) / g ** 2
    a[2][1] = (-4 - 2 * g + 4 * eh) / g ** 2
    a[3][0] = (2 + g + e * (g - 2)) / g ** 2
    a[3][1] = Decimal(0)
    a[3][2] = (-2 - 2 * g + 2 * e) / g ** 2
    b = [Decimal(0)] * 4
    b[0] = (-4 - g + e * (g ** 2 - 3 * g + 4)) / g ** 3
    b[1] = (4 + 2 * g + e * (2 * g - 4)) / g ** 3
    b[2] = b[1]
    b[3] = (-4 - 3 * g - g ** 2 + e * (4 - g)) / g ** 3
    return [[float(v) for v in row] for row in a], [float(v) for v in b]


def step_debug(problem, q, t0, dt, aux=None, verts=None):
    """One SARK4 step.  Returns (stages, aux_new): stages = [q^(1), q^(2), q^(3), q_{n+1}] (L132-134).

    verts: optional list of four (xv, vv) pairs, the vertex positions / velocities of the four stages when the
    coordinates are integrated in time (oracle/coords.py) instead of evaluated from the closed-form law."""
    dim = problem.dim
    stiff = _physics.stiff_mask(dim)                         # 1 where Lambda = 1/tau
    lam = stiff / problem.tau
    gamma = -dt / problem.tau
    a_s, b_s = coefficients(gamma)                           # stiff fields
    a_0, b_0 = [list(r) for r in RK4_A], list(RK4_B)         # Lambda = 0 fields
    nf = len(stiff)
    # per-field coefficient tables [4][4][Nf], [4][Nf]
    A = np.array([[[a_s[i][j] if stiff[k] else a_0[i][j] for k in range(nf)] for j in range(4)] for i in range(4)])
    B = np.array([[b_s[j] if stiff[k] else b_0[j] for k in range(nf)] for j in range(4)])
    has_pml = problem.sigma is not None
    if has_pml and aux is None:
        aux = np.zeros((len(problem.pml_elems), dim, nf, problem.ref.Np))

    Fs, Gs, stages = [], [], []
    qi, auxi = q, aux
    for i in range(4):
        ti = t0 + RK4_C[i] * dt
        vi = None if verts is None else verts[i]
        if has_pml:
            Fi, Gi = problem.rhs(qi, ti, aux=auxi, verts=vi)
            Gs.append(Gi)
        else:
            Fi = problem.rhs(qi, ti, verts=vi)
        Fs.append(Fi)
        if i < 3:
            ci = RK4_C[i + 1]
            qi = q * np.exp(-lam * ci * dt)[None, :, None]
            for j in range(i + 1):
                qi = qi + dt * A[i + 1][j][None, :, None] * Fs[j]
            if has_pml:
                auxi = aux
                for j in range(i + 1):
                    if RK4_A[i + 1][j] != 0.0:
                        auxi = auxi + dt * RK4_A[i + 1][j] * Gs[j]
            stages.append(qi)
    qn = q * np.exp(-lam * dt)[None, :, None]
    for j in range(4):
        qn = qn + dt * B[j][None, :, None] * Fs[j]
    stages.append(qn)
    auxn = None
    if has_pml:
        auxn = aux
        for j in range(4):
            auxn = auxn + dt * RK4_B[j] * Gs[j]
    return stages, auxn


def step(problem, q, t0, dt, nsteps, aux=None):
    """nsteps SARK4 steps from t0.  Returns q (and aux if the problem has a PML)."""
    t = t0
    for n in range(nsteps):
        stages, aux = step_debug(problem, q, t0 + n * dt, dt, aux)
        q = stages[-1]
    return (q, aux) if problem.sigma is not None else q
