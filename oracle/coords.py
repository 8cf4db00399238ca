"""Mesh coordinates advanced in time with the solver's Runge-Kutta scheme (oracle; test infrastructure only).

PAPER.md:L152 (section 5): "The nodal coordinates are advanced in time using the same Runge-Kutta integration scheme
employed for the primary solver.  During each Runge-Kutta stage, we evaluate the explicit, continuous velocity field
v_G and subsequently update the spatial coordinates of the physical nodes", and L233: "The positions of the elements
are updated by solving dx/dt = v_G where v_G is found with the time derivative of Equation 15".

The scheme is the classic RK4 of Table 1 (blank in PAPER.md:L119; reading R4) applied to the VERTICES
(the elements stay affine, L152), with the prescribed vertex velocity v(X0, t) = d/dt disp(X0, t) of oracle/motion.py:

    k_1 = v(t_n)            x^(0) = x_n
    k_2 = v(t_n + dt/2)     x^(1) = x_n + dt/2 k_1
    k_3 = v(t_n + dt/2)     x^(2) = x_n + dt/2 k_2
    k_4 = v(t_n + dt)       x^(3) = x_n + dt   k_3
    x_{n+1} = x_n + dt/6 (k_1 + 2 k_2 + 2 k_3 + k_4)

Stage i of the field update sees the positions x^(i) and the velocity k_{i+1}, so that geometry, mesh velocity,
volume and surface terms belong to the same stage (L154).  This is SURVEY.md 8(f) NEXT-2; the closed-form positions
of reading R9 remain the default.

Pinned in tests/test_oracle_coords.py: 4th-order convergence of the integrated positions to the closed-form law,
exactness for a velocity that is constant in time, and free-stream preservation on the integrated mesh.
"""
import numpy as np

from . import motion as _motion
from . import sark as _sark


def velocity(problem, t):
    """Prescribed vertex velocities v(X0, t) [Nv, dim] (L152: the grid velocity is evaluated at the mesh nodes)."""
    return _motion.vertices(problem.motion_kind, problem.motion_params, problem.X0, t)[1]


def stage_vertices(problem, x_n, t0, dt, stage_velocities=None):
    """The four (positions, velocities) pairs of one step, and x_{n+1}.

    stage_velocities: optional (k_1, k_2, k_3, k_4), vertex velocities supplied by the caller for the four stages
    instead of the prescribed law (L152: "we evaluate the explicit, continuous velocity field v_G" at each stage; a
    velocity that depends on the positions, as in fluid-structure coupling (L391), has k_2 != k_3)."""
    if stage_velocities is None:
        k1 = velocity(problem, t0 + _sark.RK4_C[0] * dt)
        k2 = velocity(problem, t0 + _sark.RK4_C[1] * dt)
        k3 = velocity(problem, t0 + _sark.RK4_C[2] * dt)
        k4 = velocity(problem, t0 + _sark.RK4_C[3] * dt)
    else:
        k1, k2, k3, k4 = (np.asarray(k, dtype=float) for k in stage_velocities)
    x0 = x_n
    x1 = x_n + dt * _sark.RK4_A[1][0] * k1
    x2 = x_n + dt * _sark.RK4_A[2][1] * k2
    x3 = x_n + dt * _sark.RK4_A[3][2] * k3
    x_next = x_n + dt * (_sark.RK4_B[0] * k1 + _sark.RK4_B[1] * k2 + _sark.RK4_B[2] * k3 + _sark.RK4_B[3] * k4)
    return [(x0, k1), (x1, k2), (x2, k3), (x3, k4)], x_next


def step_debug(problem, q, x_n, t0, dt, aux=None, stage_velocities=None):
    """One SARK4 step on RK-integrated coordinates.  Returns (stages, aux_new, x_{n+1})."""
    verts, x_next = stage_vertices(problem, x_n, t0, dt, stage_velocities)
    stages, auxn = _sark.step_debug(problem, q, t0, dt, aux, verts=verts)
    return stages, auxn, x_next


def step(problem, q, x_n, t0, dt, nsteps, aux=None):
    """nsteps steps from t0.  Returns (q, x) (and aux if the problem has a PML)."""
    for n in range(nsteps):
        stages, aux, x_n = step_debug(problem, q, x_n, t0 + n * dt, dt, aux)
        q = stages[-1]
    return (q, x_n, aux) if problem.sigma is not None else (q, x_n)
