"""F(q, t) = L(q) + N~(q) of the ALE Galerkin-Boltzmann semi-discretisation (oracle; test infrastructure only).

PAPER.md:L107 (eq. 9) with the time splitting of L113-117 (eq. 10-11): F excludes the stiff linear decay -Lambda q.
In the physical sign convention (reading R2) and with the collocated relaxation (reading R8):

    F = - c sum_d A^_d (d q / d x_d)  +  v_G . grad q  +  N~(q)  +  LIFT ( Fscale * ( -A_n^- [q] + max(v_n,0) [q] ) )

    d q/d x_d = sum_a (d xi_a / d x_d) D_a q                     (L103; affine metrics L88-92)
    v_G(node) = sum_v lambda_v(node) v_v                        (P1 interpolation of vertex velocities, L152, L192)
    [q] = q+ - q-,  A_n = c sum_d n_d A^_d,  A_n^- = (A_n - |A_n|)/2,  v_n = v_G . n^    (eq. 7; reading R7)

Geometry, mesh velocity, volume and surface terms are all evaluated at the same time t (L154, GCL).

Boundary states and the absorbing layer are NOT printed in the paper (boundary conditions are never stated;
L5/L371 only name the PML): the paper offers no value to compare with.  They follow DESIGN.md readings R11 and R12
and are pinned by invariants (tests/test_oracle_pins.py) and, for the layer's pieces one direction at a time, by
consistency, the weak-derivative identity and a reflection test (tests/test_oracle_pml.py):
  wall (tag 1, moves with the mesh):  q1+ = q1-,  q_m+ = 2 q1- v_G,m / c - q_m- (momentum fields),  rest q+ = q-;
  far field (tag 2):                  q+ = q_inf;
  PML (elements with sigma_d > 0):    auxiliary fields qt^d, d = 1..dim, with
        d qt^d/dt = - c A^_d dq/dx_d + LIFT( Fscale ( -1/2 n_d c A^_d [q] + 1/2 n_d^2 |A_n| [q] ) ) - sigma_d qt^d,
        and the main fields receive  - sum_d sigma_d qt^d.
"""
import numpy as np

from . import geometry as _geometry
from . import mesh as _mesh
from . import motion as _motion
from . import physics as _physics
from . import cubature as _cubature
from .operators import ReferenceElement

WALL, FARFIELD = 1, 2


class Problem:
    """Everything F(q, t) needs besides q and t.  Mirrors the arguments of the C-ABI (mesh upload, params, motion)."""

    def __init__(self, dim, N, X0, EToV, vertex_equiv=None, EToB=None, pml_sigma=None,
                 RT=1.0, tau=1.0, q_inf=None, motion_kind=0, motion_params=None, ref=None, relax="collocation"):
        self.dim, self.N = dim, N
        self.ref = ref if ref is not None else ReferenceElement(dim, N)
        self.X0 = np.ascontiguousarray(X0, dtype=float)
        self.EToV = np.ascontiguousarray(EToV, dtype=np.int64)
        self.K = self.EToV.shape[0]
        self.EToB = None if EToB is None else np.asarray(EToB, dtype=np.int64)
        self.conn = _mesh.connect(self.ref, self.EToV, vertex_equiv, self.EToB)
        self.RT, self.tau = float(RT), float(tau)
        self.c = np.sqrt(self.RT)
        self.q_inf = None if q_inf is None else np.asarray(q_inf, dtype=float)
        self.motion_kind, self.motion_params = motion_kind, motion_params
        self.Nf = _physics.nfields(dim)
        # nonlinear relaxation: collocated at the interpolation nodes (reading R8) or cubature-projected (L84-107, L197)
        if relax not in ("collocation", "cubature"):
            raise ValueError("relax must be 'collocation' or 'cubature'")
        self.relax = relax
        self.cub = _cubature.Cubature(self.ref) if relax == "cubature" else None
        self.A = _physics.stream_matrices(dim)
        if pml_sigma is not None and np.any(np.asarray(pml_sigma) > 0):
            self.sigma = np.asarray(pml_sigma, dtype=float).reshape(self.K, dim)
            self.pml_elems = np.nonzero(np.any(self.sigma > 0, axis=1))[0]
        else:
            self.sigma = None
            self.pml_elems = np.zeros(0, dtype=np.int64)

    # -- a1 + a2: vertices and geometric factors at time t
    def geometry(self, t, verts=None):
        """verts = (xv, vv) overrides the closed-form law (coordinates integrated in time, oracle/coords.py)."""
        if verts is None:
            xv, vv = _motion.vertices(self.motion_kind, self.motion_params, self.X0, t)
        else:
            xv, vv = verts
        g = _geometry.factors(self.dim, xv, self.EToV)
        g["xv"], g["vv"] = xv, vv
        return g

    def rhs(self, q, t, aux=None, want_abs=False, verts=None):
        """q[K, Nf, Np] -> F[K, Nf, Np]   (and Faux[Kpml, dim, Nf, Np] if the mesh has a PML; and Fabs if asked).

        Fabs is the same sum with every term replaced by a bound on its absolute value: the scale against which a
        different summation order may legitimately differ (R15).
        """
        ref, dim, c, K, Nf = self.ref, self.dim, self.c, self.K, self.Nf
        Np, Nfp, Nfaces = ref.Np, ref.Nfp, ref.Nfaces
        g = self.geometry(t, verts)
        Ginv = g["Ginv"]                                        # [K, a, d] = d xi_a / d x_d
        vG = np.einsum("iv,kvd->kid", ref.lam, g["vv"][self.EToV])   # [K, Np, dim]   (L152, L192)

        # ---- volume term (eq. 9, first term)
        dref = [np.einsum("ij,kfj->kfi", ref.D[a], q) for a in range(dim)]
        grad = []
        for d in range(dim):
            gd = 0.0
            for a in range(dim):
                gd = gd + Ginv[:, a, d, None, None] * dref[a]
            grad.append(gd)
        F = np.zeros_like(q)
        stream_d = []
        for d in range(dim):
            sd = -c * np.einsum("fg,kgi->kfi", self.A[d], grad[d])
            stream_d.append(sd)
            F += sd + vG[:, None, :, d] * grad[d]
        # ---- nonlinear relaxation N~ (L115): collocated (reading R8) or P N~(I q) (eq. 9 last term, L197)
        if self.cub is None:
            F += _physics.N_tilde(dim, q, self.tau)
        else:
            F += _cubature.relaxation(self.cub, dim, q, self.tau)

        if want_abs:
            aref = [np.einsum("ij,kfj->kfi", np.abs(ref.D[a]), np.abs(q)) for a in range(dim)]
            if self.cub is None:
                Fabs = np.abs(_physics.N_tilde(dim, q, self.tau))
            else:
                Fabs = _cubature.relaxation_abs(self.cub, dim, q, self.tau)
            for d in range(dim):
                gabs = 0.0
                for a in range(dim):
                    gabs = gabs + np.abs(Ginv[:, a, d, None, None]) * aref[a]
                Fabs += c * np.einsum("fg,kgi->kfi", np.abs(self.A[d]), gabs) + np.abs(vG[:, None, :, d]) * gabs

        # ---- surface term (eq. 7, eq. 9 second term)
        qflat = q.transpose(0, 2, 1).reshape(K * Np, Nf)        # [K*Np, Nf] so that vmap indexes rows
        flux = np.zeros((K, Nf, Nfaces * Nfp))
        flux_abs = np.zeros((K, Nf, Nfaces * Nfp)) if want_abs else None
        pml = self.sigma is not None
        if pml:
            flux_d = [np.zeros((K, Nf, Nfaces * Nfp)) for _ in range(dim)]
        for f in range(Nfaces):
            idM = self.conn["vmapM"][:, f, :]                   # [K, Nfp]
            idP = self.conn["vmapP"][:, f, :]
            qM = qflat[idM]                                     # [K, Nfp, Nf]
            qP = qflat[idP].copy()
            nh = g["nhat"][:, f, :]                             # [K, dim]
            vGf = vG[:, ref.fmask[f], :]                        # [K, Nfp, dim]
            if self.EToB is not None:
                wall = self.EToB[:, f] == WALL
                far = self.EToB[:, f] == FARFIELD
                if wall.any():
                    qP[wall] = qM[wall]
                    for d in range(dim):
                        qP[wall, :, 1 + d] = 2.0 * qM[wall, :, 0] * vGf[wall, :, d] / c - qM[wall, :, 1 + d]
                if far.any():
                    qP[far] = self.q_inf[None, None, :]
            dq = qP - qM                                        # [q] = q+ - q-
            vn = np.einsum("kmd,kd->km", vGf, nh)               # v_G . n^ on the own side (C0, L196)
            An = _physics.normal_matrix(dim, c, nh)             # [K, Nf, Nf]
            Am = _physics.upwind_minus(An)
            fs = g["Fscale"][:, f]
            val = -np.einsum("kfg,kmg->kfm", Am, dq) + np.maximum(vn, 0.0)[:, None, :] * dq.transpose(0, 2, 1)
            flux[:, :, f * Nfp:(f + 1) * Nfp] = fs[:, None, None] * val
            if want_abs:
                # R15: the same sum with every term replaced by its absolute value, field coupling included.
                # The jump [q] = q+ - q- is a single IEEE subtraction of inputs (bit-identical in any
                # implementation), so it is the primitive term here; bounding it by |q+| + |q-| would hide
                # flux errors of relative size |q|/|[q]| behind the tolerance.
                adq = np.abs(dq)                                # [K, Nfp, Nf]
                bound = (np.einsum("kfg,kmg->kfm", np.abs(Am), adq)
                         + np.maximum(vn, 0.0)[:, None, :] * adq.transpose(0, 2, 1))
                flux_abs[:, :, f * Nfp:(f + 1) * Nfp] = fs[:, None, None] * bound
            if pml:
                absA = An - 2.0 * Am                            # |A_n|
                for d in range(dim):
                    vd = (-0.5 * nh[:, d, None, None] * c * np.einsum("fg,kmg->kfm", self.A[d], dq)
                          + 0.5 * (nh[:, d] ** 2)[:, None, None] * np.einsum("kfg,kmg->kfm", absA, dq))
                    flux_d[d][:, :, f * Nfp:(f + 1) * Nfp] = fs[:, None, None] * vd
        F += np.einsum("im,kfm->kfi", ref.LIFT, flux)
        if want_abs:
            Fabs += np.einsum("im,kfm->kfi", np.abs(ref.LIFT), flux_abs)

        Faux = None
        if pml:
            pe = self.pml_elems
            if aux is None:
                aux = np.zeros((len(pe), dim, Nf, Np))
            Faux = np.empty_like(aux)
            for d in range(dim):
                sig = self.sigma[pe, d][:, None, None]
                Faux[:, d] = (stream_d[d][pe] + np.einsum("im,kfm->kfi", ref.LIFT, flux_d[d][pe])
                              - sig * aux[:, d])
                F[pe] -= sig * aux[:, d]
        out = (F,)
        if pml:
            out = out + (Faux,)
        if want_abs:
            out = out + (Fabs,)
        return out if len(out) > 1 else F
