"""Prescribed mesh motion evaluated at the mesh vertices (oracle; test infrastructure only).

PAPER.md:L152 — the grid velocity is prescribed at the mesh vertices and interpolated linearly inside the elements;
L202 — "the grid velocity field v_G is explicitly defined in the whole domain".  DESIGN.md reading R9: positions are
the closed-form law x_v(t) = X0_v + disp(X0_v, t) and velocities its time derivative, both at vertices only.

Laws (``kind`` and ``params`` are the contract of include/alegb.h, restated here from the paper, not imported):
  NONE          = 0  no motion.
  SINES_PRODUCT = 1  PAPER.md:L227-231 (eq. 15): every coordinate is displaced by the same scalar
                     A sin(2 pi t/T) prod_d sin(kappa_d X_d + phi_d).        params = [A, T, kappa_1..d, phi_1..d]
  SINES_CROSS   = 2  PAPER.md:L251-256 (eq. 19): x += A s(t) sin(kY+p) sin(kZ+p), y += A s(t) sin(kX+p) sin(kZ+p),
                     z += A s(t) sin(kX+p) sin(kY+p), s(t) = sin(2 pi t/T); in 2-D x += A s(t) sin(kY+p),
                     y += A s(t) sin(kX+p).                                  params = [A, T, k, p]
  PLUNGE_BLEND  = 3  PAPER.md:L284-286 (eqs. 20-21) rigid plunge h0 sin(omega t) along ``axis``, multiplied by a
                     radial blend b(rho0) = 1 (rho0 <= r1), 1 - (6u^5 - 15u^4 + 10u^3) with u = (rho0-r1)/(r2-r1),
                     0 (rho0 >= r2); rho0 = |X0 - centre| (BASELINE.json config 3; the blend is unspecified in the
                     paper).                                                 params = [h0, omega, r1, r2, axis, c_1..d]
  CARANGIFORM   = 4  PAPER.md:L339-365: x~ = clamp(X,0,1); d_eff = max(sqrt((X-x~)^2 + Y^2 + Z^2) - R_rigid, 0);
                     B = exp(-beta d_eff^2) (set to 0 below ``Bcut``); A = a0 + a1 x~ + a2 x~^2; phi = k X - omega t;
                     S(t) the cosine ramp of L357; lateral displacement h = A sin(phi) B S along ``axis``
                     (L361 prints "R" for the ramp S — reading R13), velocity = -A omega cos(phi) B S + A sin(phi) B S'.
                                                    params = [a0, a1, a2, k, omega, R_rigid, beta, T_ramp, axis, Bcut]
"""
import numpy as np

NONE, SINES_PRODUCT, SINES_CROSS, PLUNGE_BLEND, CARANGIFORM = 0, 1, 2, 3, 4


def vertices(kind, params, X0, t):
    """Returns (xv, vv): positions and velocities [Nv, dim] of the vertices at time t."""
    X0 = np.asarray(X0, dtype=float)
    nv, dim = X0.shape
    p = np.asarray(params, dtype=float) if params is not None else np.zeros(0)
    disp = np.zeros_like(X0)
    vel = np.zeros_like(X0)
    if kind == NONE:
        pass
    elif kind == SINES_PRODUCT:
        A, T = p[0], p[1]
        kappa, phi = p[2:2 + dim], p[2 + dim:2 + 2 * dim]
        shape = np.ones(nv)
        for d in range(dim):
            shape = shape * np.sin(kappa[d] * X0[:, d] + phi[d])
        om = 2.0 * np.pi / T
        for d in range(dim):
            disp[:, d] = A * np.sin(om * t) * shape
            vel[:, d] = A * om * np.cos(om * t) * shape
    elif kind == SINES_CROSS:
        A, T, k, ph = p[0], p[1], p[2], p[3]
        om = 2.0 * np.pi / T
        s = [np.sin(k * X0[:, d] + ph) for d in range(dim)]
        for d in range(dim):
            shape = np.ones(nv)
            for o in range(dim):
                if o != d:
                    shape = shape * s[o]
            disp[:, d] = A * np.sin(om * t) * shape
            vel[:, d] = A * om * np.cos(om * t) * shape
    elif kind == PLUNGE_BLEND:
        h0, om, r1, r2, axis = p[0], p[1], p[2], p[3], int(p[4])
        c = p[5:5 + dim]
        rho0 = np.sqrt(np.sum((X0 - c[None, :]) ** 2, axis=1))
        u = np.clip((rho0 - r1) / (r2 - r1), 0.0, 1.0)
        b = 1.0 - (6 * u ** 5 - 15 * u ** 4 + 10 * u ** 3)
        disp[:, axis] = h0 * np.sin(om * t) * b
        vel[:, axis] = h0 * om * np.cos(om * t) * b
    elif kind == CARANGIFORM:
        a0, a1, a2, k, om, Rr, beta, Tr, axis, Bcut = p[:10]
        axis = int(axis)
        X = X0[:, 0]
        xt = np.minimum(1.0, np.maximum(0.0, X))
        r2 = (X - xt) ** 2
        for d in range(1, dim):
            r2 = r2 + X0[:, d] ** 2
        deff = np.maximum(np.sqrt(r2) - Rr, 0.0)
        B = np.exp(-beta * deff ** 2)
        B = np.where(B < Bcut, 0.0, B)
        Amp = a0 + a1 * xt + a2 * xt ** 2
        phi = k * X - om * t
        if t < Tr:
            S = 0.5 * (1.0 - np.cos(np.pi * t / Tr))
            Sd = np.pi / (2.0 * Tr) * np.sin(np.pi * t / Tr)
        else:
            S, Sd = 1.0, 0.0
        disp[:, axis] = Amp * np.sin(phi) * B * S
        vel[:, axis] = -Amp * om * np.cos(phi) * B * S + Amp * np.sin(phi) * B * Sd
    else:
        raise ValueError("unknown motion kind %r" % (kind,))
    return X0 + disp, vel
