"""CPU oracle for the ALE Galerkin-Boltzmann nodal-DG + SARK4 hot path (arxiv/paper_2607_00199).

THIS PACKAGE IS TEST INFRASTRUCTURE, NOT PRODUCT.  Only ``tests/``, ``__graft_entry__.smoke()`` and the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import it.  It shares no code with the CUDA path
(``paper_2607_00199_b200/``) and imports nothing from it; the CUDA path never imports this package.

What it is: a plain, slow, fp64 numpy restatement of what the paper's method computes, following PAPER.md
step by step (citations are ``PAPER.md:Lnn`` + equation / section).  Element loops are written as numpy array
operations over the element index; a matmul / eigh / Gauss-Jacobi root finder from numpy / scipy serves as a step.
No blocking, fusion or reordering beyond what the cited passage states.

Modules
  quadrature  conical-product Gauss-Jacobi rules on the reference simplex (used to *define* M, M^f, S; L94)
  nodes       Legendre-Gauss-Lobatto points and Warp & Blend nodes (L75, ref. [34])
  operators   reference element: nodes, M, D = M^-1 S, LIFT = M^-1 M^f, barycentric interpolation (L92-103, L192)
  mesh        face connectivity and trace node maps (L75 "q-, q+", L196)
  motion      prescribed mesh-motion laws, positions and velocities at vertices (L152, L227-256, L284, L339-365)
  geometry    geometric factors of affine simplices (L88-92, L193)
  physics     Hermite-moment system matrices, collision terms, upwind matrices (L36-53, L79-84, L115)
  rhs         F(q,t) = L(q) + N~(q) of eq. 9/10 on the moved mesh (L107, L113-117)
  sark        SARK4 coefficients (L148) and the stage recurrence (L132-134)
  cubature    cubature-projected relaxation P N~(I q) of eq. 9 / kernel v (L84-107, L197)
  coords      vertex coordinates advanced by the solver's RK4 (L152, L233)
  forces      pressure / viscous force integrals on wall faces (L308, L369 with L51, L53)

Parity status: every function here (cubature.py and coords.py included) is pinned by ``tests/test_oracle_*.py`` (-m "not gpu") except the wall /
far-field boundary states and the PML terms, whose *equations* the paper never prints (PAPER.md:L5, L371 name the
PML only; boundary conditions are not stated).  Those two carry "parity unpinned by the paper" in rhs.py and
DESIGN.md: they are pinned only by invariants (uniform-state preservation, sigma=0 reduction, damping).
"""
