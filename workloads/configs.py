"""The five workload configurations of BASELINE.json as seeded synthetic inputs.

Each ``config_k(scale)`` returns a plain dict of numpy arrays and scalars — the arguments of the C-ABI calls
(mesh upload, set_params, set_motion) plus an initial state and a time step.  ``scale`` < 1 shrinks the mesh for the
tests that run the CPU oracle; scale = 1 is the BASELINE.json size.  Nothing here is the method's arithmetic:
the initial state is input data (a Maxwellian), dt is the harness's CFL choice (R14).

Motion parameter vectors follow include/alegb.h (kinds: 0 NONE, 1 SINES_PRODUCT, 2 SINES_CROSS, 3 PLUNGE_BLEND,
4 CARANGIFORM).
"""
import numpy as np

from . import meshes

SEED = 199
NP_OF = {(2, 1): 3, (2, 2): 6, (2, 3): 10, (2, 4): 15, (2, 5): 21, (3, 1): 4, (3, 2): 10, (3, 3): 20, (3, 4): 35, (3, 5): 56}
NF_OF = {2: 6, 3: 10}
FACE_VERTS = {2: [[0, 1], [1, 2], [2, 0]], 3: [[0, 1, 2], [0, 1, 3], [1, 2, 3], [0, 2, 3]]}


def maxwellian(dim, rho, u, RT):
    """Moments of an equilibrium distribution: q1 = rho, q_{1+d} = rho u_d/sqrt(RT), second moments at equilibrium.
    rho[...], u[..., dim] -> q[..., Nf]  (field order of include/alegb.h)."""
    c = np.sqrt(RT)
    rho = np.asarray(rho, float)
    m = [rho * np.asarray(u, float)[..., d] / c for d in range(dim)]
    r2 = np.sqrt(2.0)
    if dim == 2:
        fields = [rho, m[0], m[1], m[0] * m[1] / rho, m[0] ** 2 / (r2 * rho), m[1] ** 2 / (r2 * rho)]
    else:
        fields = [rho, m[0], m[1], m[2], m[0] * m[1] / rho, m[0] * m[2] / rho, m[1] * m[2] / rho,
                  m[0] ** 2 / (r2 * rho), m[1] ** 2 / (r2 * rho), m[2] ** 2 / (r2 * rho)]
    return np.stack(fields, axis=-1)


def node_coordinates(X0, EToV, lam):
    """Physical coordinates of the DG nodes at t = 0: x[K, Np, dim] = lam[Np, dim+1] . X0[EToV]."""
    return np.einsum("iv,kvd->kid", lam, X0[EToV])


def cfl_dt(dim, N, X0, EToV, RT, cfl, vmax):
    """DESIGN.md R14: dt = CFL * min_e(2 r_e) / ((N+1)^2 (sqrt3 c + max|v_G|)), r_e the inscribed radius at t = 0."""
    P = X0[EToV]
    if dim == 2:
        e1, e2 = P[:, 1] - P[:, 0], P[:, 2] - P[:, 0]
        vol = 0.5 * np.abs(e1[:, 0] * e2[:, 1] - e1[:, 1] * e2[:, 0])
        per = sum(np.linalg.norm(P[:, b] - P[:, a], axis=1) for a, b in FACE_VERTS[2])
        r = 2.0 * vol / per
    else:
        e = [P[:, i] - P[:, 0] for i in (1, 2, 3)]
        vol = np.abs(np.einsum("kd,kd->k", e[0], np.cross(e[1], e[2]))) / 6.0
        area = 0.0
        for f in FACE_VERTS[3]:
            area = area + 0.5 * np.linalg.norm(np.cross(P[:, f[1]] - P[:, f[0]], P[:, f[2]] - P[:, f[0]]), axis=1)
        r = 3.0 * vol / area
    return float(cfl * np.min(2.0 * r) / ((N + 1) ** 2 * (np.sqrt(3.0 * RT) + vmax)))


def _finish(cfg, lam):
    """Attach K, sizes and (if lam is given) the initial state evaluated at the nodes."""
    cfg["K"] = int(cfg["EToV"].shape[0])
    cfg["Np"] = NP_OF[(cfg["dim"], cfg["N"])]
    cfg["Nf"] = NF_OF[cfg["dim"]]
    if lam is not None:
        x = node_coordinates(cfg["X0"], cfg["EToV"], lam)
        cfg["q0"] = np.ascontiguousarray(np.transpose(cfg["init"](x), (0, 2, 1)))   # [K, Nf, Np]
    return cfg


def config1(lam=None, n=8):
    """2-D free-stream preservation (BASELINE.json configs[0]; eq. 15)."""
    X0, EToV, equiv = meshes.periodic_square(n, 0.0, 1.0)
    RT, tau = 1.0, 1e-3
    A, T = 0.05, 1.0
    cfg = dict(name="cfg1_freestream_2d", dim=2, N=3, X0=X0, EToV=EToV, vertex_equiv=equiv, EToB=None,
               pml_sigma=None, RT=RT, tau=tau, q_inf=None,
               motion_kind=1, motion_params=np.array([A, T, np.pi, np.pi, 0.0, 0.0]), nsteps=50)
    cfg["dt"] = cfl_dt(2, 3, X0, EToV, RT, 0.5, A * 2 * np.pi / T)
    cfg["init"] = lambda x: maxwellian(2, np.ones(x.shape[:2]), np.broadcast_to([0.1, 0.05], x.shape), RT)
    return _finish(cfg, lam)


def config2(lam=None, n=64):
    """2-D moving Taylor-Green vortex (BASELINE.json configs[1])."""
    L = 2 * np.pi
    X0, EToV, equiv = meshes.periodic_square(n, 0.0, L)
    RT, nu, U0 = 1.0, 1e-2, 0.05
    tau = nu / RT
    A, T = 0.2, 1.0
    cfg = dict(name="cfg2_tgv_2d", dim=2, N=4, X0=X0, EToV=EToV, vertex_equiv=equiv, EToB=None, pml_sigma=None,
               RT=RT, tau=tau, q_inf=None, motion_kind=1, motion_params=np.array([A, T, 0.5, 0.5, 0.0, 0.0]),
               nsteps=1000, U0=U0, nu=nu)
    cfg["dt"] = cfl_dt(2, 4, X0, EToV, RT, 0.5, A * 2 * np.pi / T)

    def init(x):
        X, Y = x[..., 0], x[..., 1]
        u = np.stack([U0 * np.sin(X) * np.cos(Y), -U0 * np.cos(X) * np.sin(Y)], axis=-1)
        rho = 1.0 + U0 ** 2 / (4 * RT) * (np.cos(2 * X) + np.cos(2 * Y))
        return maxwellian(2, rho, u, RT)
    cfg["init"] = init
    return _finish(cfg, lam)


def config3(lam=None, ntheta=300, nr=100):
    """2-D plunging NACA 0012 O-grid with PML ring (BASELINE.json configs[2])."""
    X0, EToV, EToB, sigma, centre = meshes.airfoil_ogrid(ntheta, nr)
    RT, U = 1.0, 0.1
    nu = U * 1.0 / 1000.0
    tau = nu / RT
    h0, freq = 0.25, 0.5
    om = 2 * np.pi * freq
    q_inf = maxwellian(2, np.array(1.0), np.array([U, 0.0]), RT)
    cfg = dict(name="cfg3_airfoil_2d", dim=2, N=4, X0=X0, EToV=EToV, vertex_equiv=None, EToB=EToB, pml_sigma=sigma,
               RT=RT, tau=tau, q_inf=q_inf, motion_kind=3,
               motion_params=np.array([h0, om, 2.0, 10.0, 1.0, centre[0], centre[1]]), nsteps=100)
    cfg["dt"] = cfl_dt(2, 4, X0, EToV, RT, 0.5, h0 * om)
    cfg["init"] = lambda x: np.broadcast_to(q_inf, x.shape[:2] + (6,)).copy()
    return _finish(cfg, lam)


def config4(lam=None, n=32):
    """3-D deforming periodic box, the throughput configuration (BASELINE.json configs[3])."""
    X0, EToV, equiv = meshes.periodic_cube(n, 0.0, 1.0)
    RT, tau = 1.0, 1e-4
    A, T = 0.03, 1.0
    rng = np.random.default_rng(SEED)
    nm = 8
    kvec = np.empty((4, nm, 3))
    amp = rng.uniform(-1, 1, size=(4, nm)) / 8.0
    phase = rng.uniform(0, 2 * np.pi, size=(4, nm))
    for c in range(4):
        for m in range(nm):
            while True:
                k = rng.integers(-2, 3, size=3)
                if np.any(k != 0):
                    break
            kvec[c, m] = k
    cfg = dict(name="cfg4_box_3d", dim=3, N=4, X0=X0, EToV=EToV, vertex_equiv=equiv, EToB=None, pml_sigma=None,
               RT=RT, tau=tau, q_inf=None, motion_kind=2, motion_params=np.array([A, T, 2 * np.pi, 0.0]), nsteps=200)
    cfg["dt"] = cfl_dt(3, 4, X0, EToV, RT, 0.5, A * 2 * np.pi / T)

    def init(x):
        pert = []
        for c in range(4):
            s = 0.0
            for m in range(nm):
                s = s + amp[c, m] * np.cos(2 * np.pi * (x @ kvec[c, m]) + phase[c, m])
            pert.append(1e-3 * s)
        rho = 1.0 + pert[0]
        u = np.stack(pert[1:], axis=-1) * np.sqrt(RT)
        return maxwellian(3, rho, u, RT)
    cfg["init"] = init
    return _finish(cfg, lam)


def config5(lam=None, nx=100, ny=50, nz=50):
    """3-D carangiform swimmer stand-in (BASELINE.json configs[4])."""
    X0, EToV, EToB, sigma = meshes.swimmer_box(nx, ny, nz)
    RT, U = 1.0, 0.1
    tau = U * 1.0 / 5000.0 / RT
    q_inf = maxwellian(3, np.array(1.0), np.array([U, 0.0, 0.0]), RT)
    lam_w = 0.95
    k, om = 2 * np.pi / lam_w, 2 * np.pi
    cfg = dict(name="cfg5_swimmer_3d", dim=3, N=3, X0=X0, EToV=EToV, vertex_equiv=None, EToB=EToB, pml_sigma=sigma,
               RT=RT, tau=tau, q_inf=q_inf, motion_kind=4,
               motion_params=np.array([0.02, -0.0825, 0.1625, k, om, 0.5, 10.0, 1.0, 1.0, 1e-16]), nsteps=20)
    cfg["dt"] = cfl_dt(3, 3, X0, EToV, RT, 0.5, 0.2 * om)
    cfg["init"] = lambda x: np.broadcast_to(q_inf, x.shape[:2] + (10,)).copy()
    return _finish(cfg, lam)


BY_INDEX = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}
