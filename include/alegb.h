/* alegb.h — C ABI of the B200-native ALE Galerkin-Boltzmann nodal-DG + SARK4 stage library.
 *
 * What the library computes (citations: PAPER.md line + equation of arxiv/paper_2607_00199; readings Rn are listed
 * in DESIGN.md):
 *
 *   F(q, t) = - c sum_d A^_d dq/dx_d + v_G . grad q + N~(q) + LIFT( Fscale ( -A_n^- [q] + max(v_n, 0) [q] ) )
 *
 * the ALE Galerkin-Boltzmann semi-discrete operator on the mesh moved to time t (eq. 9, L65 eq. 4,
 * L81-84 eq. 7, L115 for the split N~ / Lambda), and the semi-analytic Runge-Kutta step
 *
 *   q_ni  = q_n e^{-Lambda c_i dt} + dt sum_{j<i} a~_ij F_nj ,      q_n+1 = q_n e^{-Lambda dt} + dt sum_j b~_j F_nj
 *
 * with Lambda = diag(0,..,0,1/tau,..,1/tau) and the geometry re-evaluated at every stage time (L152-154).
 * Everything is fp64; index arrays are int32.  All arithmetic of the path runs in CUDA kernels (sm_100a); there is
 * no CPU fallback: every entry point that computes returns ALEGB_CUDA_ERROR if no device is usable.
 *
 * Conventions
 *   - every call returns 0 (ALEGB_OK) or a negative alegb_status; nothing throws or aborts across the ABI;
 *     alegb_last_error(ctx) returns a text for the last failure on that context.
 *   - "HOST" pointers are read (or written) synchronously during the call and never retained.
 *   - "DEVICE" pointers are owned by the caller (e.g. torch tensors), must be 16-byte aligned and valid on the
 *     context's device; the library never frees or retains them beyond the enqueued work.
 *   - compute calls enqueue on the given stream (a cudaStream_t passed as void*, NULL = default stream) and do NOT
 *     synchronise.  A context owns one step workspace (stage states, geometry): calls on the same context from
 *     different streams must be ordered by the caller.  alegb_mesh_upload, alegb_get_* and alegb_destroy synchronise the device.
 *   - field layout: q[K][Nf][Np] (element, field, node), node fastest.  Nf = 6 (2-D) or 10 (3-D), field order
 *     2-D (a00,a10,a01,a11,a20,a02) = the paper's q1..q6 (L43-51);
 *     3-D (a000; a100,a010,a001; a110,a101,a011; a200,a020,a002)   (reading R3).
 *     Node order: lattice order of the Warp & Blend set (L75): index of vertex 2 fastest, then vertex 3, then 4.
 *   - element order is the upload order; the library does not permute.
 */
#ifndef ALEGB_H
#define ALEGB_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct alegb_ctx alegb_ctx; /* opaque; the library owns everything inside */

typedef enum {
  ALEGB_OK = 0,
  ALEGB_INVALID_ARG = -1, /* NULL where data is required, bad dim/N/kind, misaligned device pointer */
  ALEGB_BAD_MESH = -2,    /* non-positive Jacobian at t=0, unmatched face without a tag, face shared by >2 elements,
                             periodic direction with fewer than 3 cells (reading S4) */
  ALEGB_NOT_READY = -3,   /* compute call before mesh_upload / set_params */
  ALEGB_UNSUPPORTED = -4, /* (dim, N) without a compiled kernel */
  ALEGB_CUDA_ERROR = -5   /* any CUDA runtime failure, including "no device" */
} alegb_status;

/* mesh-motion laws evaluated on the device from the t=0 vertex coordinates (reading R9:
 * closed-form positions x_v(t) = X0_v + disp(X0_v,t), velocities d/dt of it, at the VERTICES only).
 *   NONE           params: none
 *   SINES_PRODUCT  PAPER.md:L227-231 (eq. 15): every coordinate += A sin(2 pi t/T) prod_d sin(kappa_d X_d + phi_d)
 *                  params = [A, T, kappa_1..dim, phi_1..dim]
 *   SINES_CROSS    PAPER.md:L251-256 (eq. 19): x_d += A sin(2 pi t/T) prod_{o != d} sin(k X_o + p)
 *                  params = [A, T, k, p]
 *   PLUNGE_BLEND   PAPER.md:L284-286 (eqs. 20-21): x_axis += h0 sin(omega t) b(|X0 - centre|),
 *                  b = 1 (rho<=r1), 1-(6u^5-15u^4+10u^3), u=(rho-r1)/(r2-r1), 0 (rho>=r2)
 *                  params = [h0, omega, r1, r2, axis, centre_1..dim]
 *   CARANGIFORM    PAPER.md:L339-365 (reading R13): lateral displacement along `axis`
 *                  (a0+a1 x~+a2 x~^2) sin(k X - omega t) B(d_eff) S(t);
 *                  params = [a0, a1, a2, k, omega, R_rigid, beta, T_ramp, axis, Bcut]
 *   USER           positions/velocities supplied by alegb_set_motion_user (constant in time) or, per RK stage, by
 *                  alegb_set_motion_user_stages
 */
typedef enum {
  ALEGB_MOTION_NONE = 0,
  ALEGB_MOTION_SINES_PRODUCT = 1,
  ALEGB_MOTION_SINES_CROSS = 2,
  ALEGB_MOTION_PLUNGE_BLEND = 3,
  ALEGB_MOTION_CARANGIFORM = 4,
  ALEGB_MOTION_USER = 5
} alegb_motion_kind;

/* How alegb_step / alegb_step_debug obtain the vertex positions of a stage.
 *   CLOSED_FORM  x_v(t_i) = X0_v + disp(X0_v, t_i) from the law (reading R9; default)
 *   RK           the coordinates are "advanced in time using the same Runge-Kutta integration scheme employed for the
 *                primary solver" (L152; L233 dx/dt = v_G): classic RK4 on dx/dt = v(X0, t) with the law's vertex
 *                velocity; stage i sees x^(i) = x_n + dt a_{i,i-1} v(t_{i-1}) and the velocity v(t_i), and the step
 *                ends with x_{n+1} = x_n + dt sum_j b_j v(t_j).  Motion kind USER: the supplied stage velocities
 *                (alegb_set_motion_user_stages; alegb_set_motion_user: one velocity for all stages).  (SURVEY 8(f) NEXT-2.)  alegb_rhs and alegb_geometry always evaluate the closed form. */
typedef enum { ALEGB_COORDS_CLOSED_FORM = 0, ALEGB_COORDS_RK = 1 } alegb_coord_mode;

/* How the nonlinear relaxation N~(q) enters F.
 *   COLLOCATION  evaluated at the interpolation nodes (reading R8; default)
 *   CUBATURE     P N~(I q) of eq. 9 (L84-107; cubature kernel, L197): q interpolated to the N_c nodes of a
 *                conical-product Gauss-Jacobi rule exact to degree 3N, N~ evaluated there, projected back with
 *                P = M^-1 I^T diag(w).  (the rule is this build's choice, reading R20.) */
typedef enum { ALEGB_RELAX_COLLOCATION = 0, ALEGB_RELAX_CUBATURE = 1 } alegb_relax_mode;

/* Create a context for simplices of dimension dim (2 or 3) and polynomial order N (1..ALEGB_MAX_N) on CUDA device
 * `cuda_device`.  Builds the reference element on the host: Warp & Blend nodes (L75), D_r,D_s(,D_t) = M^-1 S and
 * LIFT = M^-1 M^f (L94-103).  *out is NULL on failure. */
int alegb_create(alegb_ctx** out, int dim, int N, int cuda_device);
int alegb_destroy(alegb_ctx* ctx);

/* Mesh upload (HOST pointers, copied).  Straight-sided, conforming, positively oriented simplices (L73).
 *   X0[Nverts*dim]        vertex coordinates at t = 0
 *   EToV[K*(dim+1)]       element-to-vertex table; local face numbering: 2-D f1=(v1,v2), f2=(v2,v3), f3=(v3,v1);
 *                         3-D f1=(v1,v2,v3), f2=(v1,v2,v4), f3=(v2,v3,v4), f4=(v1,v3,v4)
 *   vertex_equiv[Nverts]  periodic master id of each vertex, or NULL (no periodicity)
 *   EToB[K*(dim+1)]       0 interior, 1 moving no-slip wall, 2 far field (reading R11), or NULL (no boundary)
 *   pml_sigma[K*dim]      per-element, per-direction damping of the absorbing layer, 0 = not in the layer
 *                         (reading R12), or NULL
 * Builds EToE/EToF and the trace maps vmapM/vmapP (L75, L196) by vertex ids, uploads everything, allocates the
 * step workspace.  Synchronises. */
int alegb_mesh_upload(alegb_ctx* ctx, int64_t Nverts, const double* X0, int64_t K, const int32_t* EToV,
                      const int32_t* vertex_equiv, const int8_t* EToB, const double* pml_sigma);

/* RT (L30), tau (L30; +inf allowed: collisionless), q_inf[Nf] far-field state (HOST, or NULL if no far-field faces) */
int alegb_set_params(alegb_ctx* ctx, double RT, double tau, const double* q_inf);

/* Prescribed motion law (see alegb_motion_kind); params is a HOST array, copied. */
int alegb_set_motion(alegb_ctx* ctx, int kind, const double* params, int nparams);
/* kind USER: DEVICE arrays [Nverts*dim] of vertex positions and velocities, copied device-to-device on the
 * default stream and used for every subsequent evaluation (all four stages of every step: a velocity constant in
 * time) until the motion is set again.  Waits for the whole device first (a step still running on any stream,
 * the library's side stream included, reads the buffers this call overwrites; it also makes arrays produced on
 * another stream visible), copies on the default stream and synchronises it. */
int alegb_set_motion_user(alegb_ctx* ctx, const double* d_xv, const double* d_vv);
/* kind USER with data that change from stage to stage ("During each Runge-Kutta stage, we evaluate the
 * explicit, continuous velocity field v_G and subsequently update the spatial coordinates"; L391 fluid-structure
 * outlook): DEVICE arrays [4][Nverts*dim], entry i belongs to RK stage i of the NEXT step
 * (stage times t_n + (0, 1/2, 1/2, 1) dt); copied.  Every following alegb_step / alegb_step_debug step uses the same
 * four entries, so a caller whose velocities change in time calls this before each single step.
 *   coordinate mode CLOSED_FORM: stage i sees the positions d_xv4[i] and the velocities d_vv4[i].
 *   coordinate mode RK: d_xv4 is ignored except for entry 0 on the first call (the starting positions, see
 *     alegb_set_coordinate_mode) and may be NULL afterwards; the library integrates the positions with the classic
 *     RK4 of the solver and the caller's stage velocities k_i = d_vv4[i-1]:
 *       x^(1) = x_n + dt/2 k_1,  x^(2) = x_n + dt/2 k_2,  x^(3) = x_n + dt k_3,  x_{n+1} = x_n + dt/6 (k_1+2k_2+2k_3+k_4),
 *     stage i of the fields sees x^(i) and k_{i+1}.
 * alegb_rhs, alegb_geometry and alegb_wall_forces (one evaluation, no stage) use entry 0.
 * Synchronisation as alegb_set_motion_user: device-wide wait, copies, default stream synchronised -- calling it
 * between single steps is safe whatever stream the steps run on, at the price of draining the device.
 * Errors: INVALID_ARG (d_vv4 NULL; d_xv4 NULL before any positions were supplied), NOT_READY, CUDA_ERROR. */
int alegb_set_motion_user_stages(alegb_ctx* ctx, const double* d_xv4, const double* d_vv4);

/* Select the relaxation mode for alegb_rhs / alegb_step (every stage kernel honours it).  CUBATURE builds the rule
 * and I, P on the host, uploads them and allocates R[K][dim(dim+1)/2][Np] (part of alegb_workspace_bytes).
 * Synchronises.  Errors: INVALID_ARG, NOT_READY (no mesh), CUDA_ERROR. */
int alegb_set_relaxation(alegb_ctx* ctx, int mode);
/* The cubature rule and operators, HOST out, any pointer may be NULL: degree, Nc, rst[dim][Nc], w[Nc],
 * I[Nc][Np] (L86), P[Np][Nc] (L103).  Call with the arrays NULL first to learn Nc.  Works on host-only contexts. */
int alegb_get_cubature(alegb_ctx* ctx, int* degree, int* Nc, double* rst, double* w, double* I, double* P);

/* Pressure and viscous force on the faces tagged `tag` (1 = wall) at time t:
 *   F_p = - int p n_b dS,  F_v = int sigma . n_b dS,  p = q1 RT (L53), sigma from the second moments (L51),
 *   n_b = outward normal of the body, face integrals by the nodal face quadrature sJ (1^T M^f) (reading R22);
 * c_D = F_x / (0.5 rho u^2 c) etc. are the caller's division.  DEVICE q [K][Nf][Np]; HOST out h_Fp[dim], h_Fv[dim].
 * Geometry from the closed-form law at t.  Enqueues on `stream` and synchronises it.  Deterministic (fixed grid,
 * ordered second pass).  A mesh without tagged faces gives zeros.  Errors: INVALID_ARG, NOT_READY, CUDA_ERROR. */
int alegb_wall_forces(alegb_ctx* ctx, double t, const double* d_q, int tag, double* h_Fp, double* h_Fv, void* stream);

/* The same integrals for callers that cannot allocate device memory at the point where they need the forces.
 * Who that is: the forces are a per-time-step diagnostic (drag / lift histories, L308), so the call sits inside the
 * time loop, and alegb_wall_forces cudaMallocs its partial-sum buffer the first time it runs -- that is, in the middle
 * of the loop.  That does not work for (i) an application that, once the mesh is uploaded, gives all remaining HBM to
 * its own pool (a framework's caching allocator, a solver's arena): cudaMalloc then returns out-of-memory although the
 * pool has room; (ii) a time loop that keeps several streams busy and cannot take the device-wide stall that
 * cudaMalloc / cudaFree bring with them; (iii) a caller that wants the result to stay on the device and the stream
 * to keep running (alegb_wall_forces copies to the host and waits for the stream).
 * This entry point calls no cudaMalloc, cudaFree or allocating library routine, copies nothing to the host and does
 * not synchronise.  Its only scratch memory, the per-block partial sums of the first pass, is a fixed array inside the
 * library image: ALEGB_WALL_FORCES_STATIC_MAX_BLOCKS x 6 doubles = 48 KiB on every GPU that loads libalegb.so, held
 * until the process exits.
 *   d_q      DEVICE [K][Nf][Np], read only
 *   tag      boundary tag, 1..127
 *   nblocks  thread blocks of the first pass = partial sums kept: 0 selects 296, the grid alegb_wall_forces uses, and
 *            the result then equals that call's bit for bit; any other value 1..ALEGB_WALL_FORCES_STATIC_MAX_BLOCKS
 *            changes only the order of the final sum (round-off).  Larger values do not fit the array and are
 *            rejected with ALEGB_INVALID_ARG and a message naming the limit; nothing is launched.
 *   d_F      DEVICE out [2 dim], caller-owned: F_p[0..dim) then F_v[0..dim); valid once `stream` has reached this
 *            point.  A mesh without tagged faces gives zeros (a memset on `stream`).
 * Geometry from the closed-form law at t, exactly as alegb_wall_forces (two more launches on `stream`).
 * First call on each device: the library asks the runtime for the array's address on that device
 * (cudaGetSymbolAddress, which may load the module there) and remembers it.  Make that first call during set-up,
 * before any stream capture is begun in the process, and with no other work depending on its latency.
 * Sharing: every call on a device -- from any context, any stream, any thread -- uses the one array.  Nothing in it
 * needs to be zero beforehand (each launched block overwrites its own entry and only those entries are read), so
 * calls that follow one another on a stream, or are ordered by events, are independent of each other.  Calls whose
 * kernels may run concurrently on the same device are a data race on the partial sums: order them.
 * Errors: INVALID_ARG (NULL pointer, tag, nblocks), NOT_READY, CUDA_ERROR. */
#define ALEGB_WALL_FORCES_STATIC_MAX_BLOCKS 1024
int alegb_wall_forces_static(alegb_ctx* ctx, double t, const double* d_q, int tag, int nblocks, double* d_F,
                             void* stream);

/* Select the coordinate mode.  RK: the library's current positions x_n are set to the law's positions at t_start
 * (kind USER: to the positions last given to alegb_set_motion_user); every alegb_step then advances them, so
 * consecutive calls must continue in time where the previous one ended.  alegb_step_debug reads x_n and leaves it
 * unchanged.  Synchronises.  Errors: INVALID_ARG (mode), NOT_READY (no mesh), CUDA_ERROR. */
int alegb_set_coordinate_mode(alegb_ctx* ctx, int mode, double t_start);
/* Current vertex positions, DEVICE out [Nverts*dim]: x_n in RK mode, else the positions of the last evaluation.
 * Enqueued on `stream`, does not synchronise. */
int alegb_get_positions(alegb_ctx* ctx, double* d_x, void* stream);

/* F = L(q) + N~(q) at time t (no -Lambda q), DEVICE q, F [K][Nf][Np].  In PML elements the library's current
 * auxiliary fields enter F (term - sum_d sigma_d q~^d). */
int alegb_rhs(alegb_ctx* ctx, double t, const double* d_q, double* d_F, void* stream);
/* Same, plus the right-hand side of the auxiliary fields: d_aux, d_Faux DEVICE [Kpml][dim][Nf][Np]
 * (Kpml = alegb_pml_count; order = ascending element index).  d_aux == NULL uses the library's own state. */
int alegb_rhs_pml(alegb_ctx* ctx, double t, const double* d_q, const double* d_aux, double* d_F, double* d_Faux,
                  void* stream);

/* nsteps SARK4 steps of size dt from t0, in place on DEVICE q.  The library's PML auxiliary state advances with it. */
int alegb_step(alegb_ctx* ctx, double* d_q, double t0, double dt, int nsteps, void* stream);
/* One step, returning the four stage states q(1), q(2), q(3), q_{n+1}: d_stages DEVICE [4][K][Nf][Np].  d_q is not
 * modified; the PML auxiliary state is advanced exactly as alegb_step would. */
int alegb_step_debug(alegb_ctx* ctx, const double* d_q, double t0, double dt, double* d_stages, void* stream);

/* Geometry of the mesh moved to time t.  Any output may be NULL.  DEVICE arrays:
 *   d_vgeo[K][dim*dim+1]   (d xi_a/d x_d, a-major: r_x r_y (r_z) s_x ...; then J)
 *   d_sgeo[K][Nfaces][dim+2] (unit outward normal n_1..n_dim, sJ, Fscale = sJ/J)
 *   d_xv[Nverts][dim], d_vv[Nverts][dim] */
int alegb_geometry(alegb_ctx* ctx, double t, double* d_vgeo, double* d_sgeo, double* d_xv, double* d_vv,
                   void* stream);

/* PML auxiliary state: count of layer elements, their ids (HOST out), zeroing, device-to-device get/set. */
int64_t alegb_pml_count(const alegb_ctx* ctx);
int alegb_pml_elements(const alegb_ctx* ctx, int32_t* elems /* HOST [Kpml] */);
int alegb_pml_reset(alegb_ctx* ctx, void* stream);
int alegb_pml_get(alegb_ctx* ctx, double* d_aux, void* stream);
int alegb_pml_set(alegb_ctx* ctx, const double* d_aux, void* stream);

/* Introspection (HOST out, any pointer may be NULL): sizes, reference nodes r,s,t [Np], operators row-major
 * Dr,Ds,Dt [Np*Np], LIFT [Np*(Nfaces*Nfp)], trace maps [K*Nfaces*Nfp] (flattened node index e*Np+n), nodal
 * quadrature weights w[Np] = 1^T M, barycentric interpolation matrix lam[Np*(dim+1)] (L192). */
int alegb_get_sizes(const alegb_ctx* ctx, int* dim, int* N, int* Np, int* Nfp, int* Nfaces, int* Nfields,
                    int64_t* K, int64_t* Nverts);
int alegb_get_operators(alegb_ctx* ctx, double* r, double* s, double* t3, double* Dr, double* Ds, double* Dt,
                        double* LIFT, int32_t* vmapM, int32_t* vmapP);
int alegb_get_reference(const alegb_ctx* ctx, double* w, double* lam, int32_t* fmask);
/* SARK4 coefficients the library would use for gamma = -dt/tau (L144-148; reading R6): HOST out
 * a[6] = (a10,a20,a21,a30,a31,a32), b[4]. */
int alegb_sark_coefficients(double gamma, double* a, double* b);

int64_t alegb_workspace_bytes(const alegb_ctx* ctx);
const char* alegb_last_error(const alegb_ctx* ctx);
/* number of kernel launches the library has enqueued on this context since creation */
int64_t alegb_launch_count(const alegb_ctx* ctx);
/* Which fused stage kernel runs: 0 = automatic (the pipelined tensor-core DMMA kernel where one is compiled for
 * (dim, N), the generic kernel otherwise), 1 = generic element-blocked DFMA kernel (every (dim, N); kept as an
 * independent implementation of the same operator), 2 = pipelined DMMA kernel (producer/consumer warps; returns
 * ALEGB_UNSUPPORTED if there is none for (dim, N)).  Tests run both. */
int alegb_set_kernel(alegb_ctx* ctx, int kind);
/* Cap on the number of CTAs of the persistent kernels (stage, absorbing layer, cubature): 0 = one per SM (default).
 * A tuning / test knob: with few CTAs every CTA walks through many work units, which is the regime in which the
 * shared-memory ring of the pipelined kernel wraps many times.  Results do not depend on it. */
int alegb_set_max_ctas(alegb_ctx* ctx, int max_ctas);
/* Hand-over parameters of the pipelined stage kernel compiled for (dim, N), HOST out cfg[8] = {producer groups,
 * ring slots, work items per quad, consumer warps, warps per producer group, producer warps, elements per quad,
 * dynamic shared memory in bytes}.  ALEGB_UNSUPPORTED if there is no such kernel.  Needs no context and no device
 * (tests/test_pipe_protocol.py simulates the protocol with these numbers). */
int alegb_pipe_config(int dim, int N, int* cfg);
/* The same eight numbers for the instantiation that advances the absorbing layer inside the stage kernel (see
 * alegb_set_layer_fusion): its slots carry dim more flux tiles, so it has one producer group and as many ring slots as
 * shared memory allows, and a consumer warp releases a slot only after the directional contractions.
 * ALEGB_UNSUPPORTED if (dim, N) has no such instantiation.  Needs no context and no device. */
int alegb_pipe_config_layer(int dim, int N, int* cfg);
/* Absorbing layer (a8): where the pipelined stage kernel runs and has an instantiation for it, the auxiliary fields of
 * the layer elements are advanced INSIDE the stage kernel (their D_a q, exterior traces and metrics are already on
 * chip there): the quads outside the layer run through the plain instantiation, the quads that touch the layer
 * through a second launch that also advances their auxiliary fields.  on = 0 selects the separate layer kernel after
 * the stage kernel.  Default: on in 3-D, off in 2-D (where the layer is a thin ring and the split costs more than the
 * fusion saves; measured in profiles/r2_layer_fusion.md).  Same equations (reading R12); results agree to round-off (summation order of the LIFT
 * contraction is the same, the volume part is formed per direction in both). */
int alegb_set_layer_fusion(alegb_ctx* ctx, int on);
/* Inside a step the vertex-motion and geometric-factor kernels (a1, a2) of stage i+1 depend on time only; with the
 * overlap on (default) they run on a stream of the library's own beside the stage kernel of stage i, into a second
 * set of geometry arrays, joined by events (captured into the step graph as a parallel branch).  Same kernels, same
 * results bit for bit; off = everything in order on the caller's stream. */
int alegb_set_geometry_overlap(alegb_ctx* ctx, int on);
/* alegb_step with nsteps >= 2 replays ONE captured CUDA graph per step (clock kernel + the a1, a2, a3-a8 launches of
 * the four stages; stage times t_n + c_i dt are computed on the device with the host loop's IEEE operations, so the
 * result is bit-identical to nsteps single-step calls).  It removes the per-launch host cost that bounds the small
 * L2-resident configurations.  on = 0 switches it off (default on).  The graph is not used while
 * alegb_profile_enable is active.  SURVEY 7 step (8). */
int alegb_set_graph(alegb_ctx* ctx, int on);
/* Stage-kernel timing for roofline reports: while enabled, every launch of the fused stage kernel is bracketed by
 * CUDA events on its stream (at most 4096 launches are kept per enable).  alegb_profile_read synchronises the
 * device and returns the number of bracketed launches and the sum of their durations in milliseconds. */
int alegb_profile_enable(alegb_ctx* ctx, int on);
int alegb_profile_read(alegb_ctx* ctx, int64_t* launches, double* total_ms);
/* The fp64 ceiling of the context's device, measured: two register-resident microbenchmarks (chains of
 * mma.sync.m8n8k4.f64 = DMMA, and of DFMA; 16 warps per SM, 8 independent accumulator sets each), best of 5 timed
 * launches after a warm-up, CUDA events.  HOST out, TFLOP/s.  This is the denominator of the stage kernels' binding
 * roofline (fp64-bound at N >= 3 in 3-D); bench.py reports it beside the figure derived from unit counts
 * and the clock.  Takes about 50 ms, synchronises the device.  Errors: INVALID_ARG, CUDA_ERROR. */
int alegb_measure_fp64_peak(alegb_ctx* ctx, double* dmma_tflops, double* dfma_tflops);
/* Synchronous convenience entry for host buffers (HOST q [K][Nf][Np], updated in place): copies q to the device,
 * runs nsteps SARK4 steps, copies the result back.  Everything is enqueued on the LEGACY DEFAULT STREAM (stream 0),
 * which the call synchronises before it returns; the whole state crosses PCIe twice per call, so the cost per step
 * falls with nsteps (one step per call is bound by the two copies, not by the kernels).  Used for end-to-end timing. */
int alegb_step_host(alegb_ctx* ctx, double* h_q, double t0, double dt, int nsteps);

#define ALEGB_MAX_N 5

#ifdef __cplusplus
}
#endif
#endif /* ALEGB_H */
