"""The Galerkin-Boltzmann moment system (oracle; test infrastructure only).

PAPER.md:L34-53: second-order Hermite expansion of the BGK-Boltzmann equation; n = 6 fields in 2-D, 10 in 3-D (L39).
The 2-D coefficient matrix is blank in PAPER.md (L39-41) and the 3-D system is deferred to ref. [33] (L53), so the
matrices are *generated from the rule that defines them* (readings R1, R3): testing eq. 1 against the
orthonormal Hermite polynomials h_alpha(v/c), c = sqrt(RT), and using the three-term recurrence
    xi h_i(xi) = sqrt(i+1) h_{i+1}(xi) + sqrt(i) h_{i-1}(xi)
gives   d a_alpha/dt + c sum_d d/dx_d ( sqrt(alpha_d + 1) a_{alpha+e_d} + sqrt(alpha_d) a_{alpha-e_d} ) = collision,
truncated at |alpha| <= 2.  So (A^_d)_{alpha,beta} = sqrt(alpha_d+1) if beta = alpha+e_d, sqrt(alpha_d) if
beta = alpha-e_d, 0 otherwise.  What pins it to the paper: the printed equilibrium moments q2^2/(sqrt2 q1) (L43),
rho u = sqrt(RT) q2 (L47) and nu = tau RT (L45, Taylor-Green decay test).

Sign convention (reading R2): the physical system is  dq/dt|_xi + c sum_d A^_d dq/dx_d - v_G.grad q = N(q);
the paper's A_x (L36) is -c A^.

Field order: 2-D (00, 10, 01, 11, 20, 02) = the paper's q1..q6 (L43, L47, L51);
             3-D (000; 100, 010, 001; 110, 101, 011; 200, 020, 002) (this build's convention, R3).
"""
import numpy as np

MULTI = {
    2: [(0, 0), (1, 0), (0, 1), (1, 1), (2, 0), (0, 2)],
    3: [(0, 0, 0), (1, 0, 0), (0, 1, 0), (0, 0, 1), (1, 1, 0), (1, 0, 1), (0, 1, 1), (2, 0, 0), (0, 2, 0), (0, 0, 2)],
}


def nfields(dim):
    return len(MULTI[dim])


def stream_matrices(dim):
    """A^[d] (list of dim symmetric Nf x Nf arrays), from the Hermite recurrence."""
    idx = {a: i for i, a in enumerate(MULTI[dim])}
    nf = len(idx)
    out = []
    for d in range(dim):
        A = np.zeros((nf, nf))
        for alpha, i in idx.items():
            up = tuple(alpha[m] + (1 if m == d else 0) for m in range(dim))
            dn = tuple(alpha[m] - (1 if m == d else 0) for m in range(dim))
            if up in idx:
                A[i, idx[up]] = np.sqrt(alpha[d] + 1.0)
            if dn in idx:
                A[i, idx[dn]] = np.sqrt(float(alpha[d]))
        out.append(A)
    return out


def stiff_mask(dim):
    """Lambda = diag(0,...,0, 1/tau, ...): 1 for the second-order moments."""
    return np.array([1.0 if sum(a) == 2 else 0.0 for a in MULTI[dim]])


def second_moment_equilibrium(dim, q):
    """a^eq_alpha for |alpha| = 2 from q (array [..., Nf, ...] with the field axis = -2):
    q_i q_j / q_1 for the mixed moments, q_i^2 / (sqrt2 q_1) for the pure ones."""
    out = np.zeros_like(q)
    for i, alpha in enumerate(MULTI[dim]):
        if sum(alpha) != 2:
            continue
        nz = [d for d in range(dim) if alpha[d] > 0]
        if len(nz) == 2:
            out[..., i, :] = q[..., 1 + nz[0], :] * q[..., 1 + nz[1], :] / q[..., 0, :]
        else:
            out[..., i, :] = q[..., 1 + nz[0], :] ** 2 / (np.sqrt(2.0) * q[..., 0, :])
    return out


def N_tilde(dim, q, tau):
    """N~(q) of PAPER.md:L115 — the part of the collision term that is not -Lambda q.  q[..., Nf, Np]."""
    return second_moment_equilibrium(dim, q) / tau


def N_full(dim, q, tau):
    """N(q) of PAPER.md:L43."""
    return N_tilde(dim, q, tau) - stiff_mask(dim)[:, None] * q / tau


def normal_matrix(dim, c, nhat):
    """A_n = c sum_d n_d A^_d for nhat[..., dim] -> [..., Nf, Nf]."""
    A = stream_matrices(dim)
    out = 0.0
    for d in range(dim):
        out = out + nhat[..., d, None, None] * A[d]
    return c * out


def upwind_minus(An):
    """A_n^- = (A_n - |A_n|)/2 with |A_n| = R |Lambda| R^T from a numerical symmetric eigendecomposition
    (F_S = R Lambda R^-1; eq. 7).  The library uses a closed form instead (R7)."""
    lam, R = np.linalg.eigh(An)
    absA = np.einsum("...ik,...k,...jk->...ij", R, np.abs(lam), R)
    return 0.5 * (An - absA)


def equilibrium_state(dim, rho, u, RT):
    """q of a Maxwellian with density rho and velocity u[..., dim]: q1 = rho, q_{1+d} = rho u_d / sqrt(RT) (L47),
    second moments at equilibrium (L43; reading R16).  rho[...], returns [..., Nf]."""
    c = np.sqrt(RT)
    rho = np.asarray(rho, dtype=float)
    u = np.asarray(u, dtype=float)
    nf = nfields(dim)
    q = np.zeros(rho.shape + (nf, 1))
    q[..., 0, 0] = rho
    for d in range(dim):
        q[..., 1 + d, 0] = rho * u[..., d] / c
    q = q + second_moment_equilibrium(dim, q)
    return q[..., 0]
