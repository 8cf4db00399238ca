// C-ABI entry points (include/alegb.h): context management, mesh upload, the stage loop of the SARK4 step.
// Host logic only: every arithmetic step of the path runs in the kernels of kernels.cu / stage_pipe.cu / pml_mma.cu /
// cubature.cu.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>
#include <new>

#include "../../include/alegb.h"
#include "alegb_internal.h"

using namespace alegb;

struct alegb_ctx {
  int device = 0, num_sms = 0, max_ctas = 0;   // max_ctas: alegb_set_max_ctas (0 = one CTA per SM)
  int ctas() const { return max_ctas > 0 && max_ctas < num_sms ? max_ctas : num_sms; }
  RefElement ref;
  int Nf = 0;
  int64_t K = 0, Nverts = 0, Kpml = 0;
  bool mesh_ready = false, params_ready = false, has_boundary = false;
  double RT = 1.0, tau = 1.0, c = 1.0, invtau = 1.0;
  double q_inf[kMaxFields] = {0};
  MotionArgs motion{};
  std::vector<int32_t> vmapM_host, vmapP_host, pml_elems_host;
  // device: operators
  double *d_Dt = nullptr, *d_LIFTt = nullptr, *d_lam = nullptr, *d_Avol = nullptr, *d_AliftP = nullptr;
  int32_t* d_fmask = nullptr;
  double *d_wface = nullptr, *d_force = nullptr;   // NEXT-3: face quadrature weights; partial sums + result
  bool cub_mma_ok = false;  // a DMMA cubature kernel exists for (dim, N)
  bool pipe_ok = false;  // a pipelined DMMA stage kernel exists for (dim, N)
  bool pml_mma_ok = false;  // a DMMA kernel for the absorbing layer's auxiliary fields exists for (dim, N)
  bool pipe_layer_ok = false;  // the pipelined stage kernel has an instantiation with the absorbing layer fused in
  bool fuse_layer = true;      // alegb_set_layer_fusion
  // a8 inside the stage kernel (one launch per stage instead of two) where the pipelined kernel runs and supports it
  bool layer_fused() const { return Kpml > 0 && fuse_layer && pipe_ok && pipe_layer_ok && kernel_mode != 1; }
  int kernel_mode = 0;   // 0 auto (pipelined DMMA, else generic), 1 generic, 2 pipelined DMMA
  // device: mesh
  double *d_X0 = nullptr, *d_xv = nullptr, *d_vv = nullptr;
  // NEXT-2: coordinates integrated by RK4: current positions x_n, the user's constant velocity
  int coord_mode = ALEGB_COORDS_CLOSED_FORM;
  // NEXT-1: cubature-projected relaxation
  int relax_mode = ALEGB_RELAX_COLLOCATION;
  Cubature cub;                       // host copy (built on first use)
  int cub_EB = 0;                     // elements per CTA pass of cubature_relax_kernel
  double *d_It = nullptr, *d_Pt = nullptr, *d_R = nullptr;
  double *d_AI = nullptr, *d_AP = nullptr;   // I, P in DMMA A-fragment order (cubature_mma_kernel)
  double *d_xn = nullptr;
  double *d_user_xv = nullptr, *d_user_vv = nullptr;   // kind USER: the caller's data of the four stages, [4][Nverts*dim] each
  int32_t *d_EToV = nullptr, *d_vmapP = nullptr;
  int8_t* d_EToB = nullptr;
  double *d_vgeo = nullptr, *d_sgeo = nullptr, *d_vvel = nullptr;
  // second set of geometry arrays + side stream: a1/a2 of stage i+1 depend on time only, so inside a step they run
  // beside the stage kernel of stage i (the persistent stage kernel leaves threads and registers for them)
  double *d_vgeo1 = nullptr, *d_sgeo1 = nullptr, *d_vvel1 = nullptr;
  int geo_buf = 0;                       // which set update_geometry / fill_common use
  bool overlap_geometry = true;
  cudaStream_t geo_stream = nullptr;
  cudaEvent_t ev_fork = nullptr, ev_geo[4] = {nullptr, nullptr, nullptr, nullptr}, ev_stage[4] = {nullptr, nullptr, nullptr, nullptr};
  double* vg() const { return geo_buf ? d_vgeo1 : d_vgeo; }
  double* sg() const { return geo_buf ? d_sgeo1 : d_sgeo; }
  double* vvl() const { return geo_buf ? d_vvel1 : d_vvel; }
  int32_t *d_pml_index = nullptr, *d_pml_elems = nullptr;
  int32_t *d_quads_layer = nullptr, *d_quads_plain = nullptr;   // quads that touch the absorbing layer / the others
  int64_t nquads_layer = 0, nquads_plain = 0;
  double* d_pml_sigma = nullptr;
  // device: step workspace
  double *d_Q1 = nullptr, *d_Q2 = nullptr, *d_F0 = nullptr, *d_ACC = nullptr, *d_Qhost = nullptr;
  double *d_AUX = nullptr, *d_AUXS = nullptr, *d_AUXACC = nullptr;
  int64_t workspace_bytes = 0;
  int64_t launches = 0;
  bool profiling = false;
  std::vector<cudaEvent_t> prof_events;  // pairs (start, stop), created on demand
  size_t prof_used = 0;
  // one SARK4 step captured as a CUDA graph (alegb_step with nsteps >= 2): stage times live on the device
  bool use_graph = true;
  uint64_t config_version = 0;        // bumped by every call that changes what a step launches
  cudaStream_t capture_stream = nullptr;
  cudaGraphExec_t step_graph = nullptr;
  struct { double* d_q; double dt; uint64_t version; int64_t launches; } graph_key{nullptr, 0, 0, 0};
  double* d_clock = nullptr;          // {t0, dt, stage times[4]} of the current run of steps
  long long* d_step_counter = nullptr;
  std::string err;
};

namespace {

int fail(alegb_ctx* ctx, int code, const std::string& msg) {
  if (ctx) ctx->err = msg;
  return code;
}
int cuda_fail(alegb_ctx* ctx, cudaError_t e, const char* where) {
  return fail(ctx, ALEGB_CUDA_ERROR, std::string(where) + ": " + cudaGetErrorString(e));
}
#define CU(call)                                             \
  do {                                                       \
    cudaError_t e_ = (call);                                 \
    if (e_ != cudaSuccess) return cuda_fail(ctx, e_, #call); \
  } while (0)

template <class T>
cudaError_t dev_alloc(alegb_ctx* ctx, T** p, size_t count) {
  *p = nullptr;
  if (count == 0) return cudaSuccess;
  cudaError_t e = cudaMalloc((void**)p, count * sizeof(T));
  if (e == cudaSuccess) ctx->workspace_bytes += (int64_t)(count * sizeof(T));
  return e;
}
template <class T>
cudaError_t upload(alegb_ctx* ctx, T** p, const T* host, size_t count) {
  cudaError_t e = dev_alloc(ctx, p, count);
  if (e != cudaSuccess || count == 0) return e;
  return cudaMemcpy(*p, host, count * sizeof(T), cudaMemcpyHostToDevice);
}
template <class T>
void dev_free(T*& p) {
  if (p) cudaFree(p);
  p = nullptr;
}

void free_mesh(alegb_ctx* ctx) {
  dev_free(ctx->d_xn); dev_free(ctx->d_user_xv); dev_free(ctx->d_user_vv); ctx->coord_mode = ALEGB_COORDS_CLOSED_FORM;
  dev_free(ctx->d_R); ctx->relax_mode = ALEGB_RELAX_COLLOCATION;
  dev_free(ctx->d_X0); dev_free(ctx->d_xv); dev_free(ctx->d_vv); dev_free(ctx->d_EToV); dev_free(ctx->d_vmapP);
  dev_free(ctx->d_EToB); dev_free(ctx->d_vgeo); dev_free(ctx->d_sgeo); dev_free(ctx->d_vvel);
  dev_free(ctx->d_vgeo1); dev_free(ctx->d_sgeo1); dev_free(ctx->d_vvel1); ctx->geo_buf = 0;
  dev_free(ctx->d_pml_index); dev_free(ctx->d_pml_elems); dev_free(ctx->d_pml_sigma);
  dev_free(ctx->d_quads_layer); dev_free(ctx->d_quads_plain); ctx->nquads_layer = ctx->nquads_plain = 0;
  dev_free(ctx->d_Q1); dev_free(ctx->d_Q2); dev_free(ctx->d_F0); dev_free(ctx->d_ACC); dev_free(ctx->d_Qhost);
  dev_free(ctx->d_AUX); dev_free(ctx->d_AUXS); dev_free(ctx->d_AUXACC);
  ctx->mesh_ready = false;
  ctx->K = ctx->Nverts = ctx->Kpml = 0;
  ctx->config_version++;
}

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// a1 + a2 at time t into the context's geometry arrays
// (kind USER: no a1 launch, a2 reads the caller's positions / velocities of RK stage `stage`)
int update_geometry(alegb_ctx* ctx, double t, cudaStream_t s, const double* t_dev = nullptr, int stage = 0) {
  const int dim = ctx->ref.dim;
  const double *xv = ctx->d_xv, *vv = ctx->d_vv;
  if (ctx->motion.kind != ALEGB_MOTION_USER) {
    CU(launch_vertex_motion(dim, ctx->Nverts, ctx->d_X0, ctx->motion, t, t_dev, ctx->d_xv, ctx->d_vv, s));
    ctx->launches++;
  } else {
    const size_t n = (size_t)ctx->Nverts * dim;
    xv = ctx->d_user_xv + stage * n;
    vv = ctx->d_user_vv + stage * n;
  }
  CU(launch_geometry(dim, ctx->K, ctx->d_EToV, xv, vv, ctx->vg(), ctx->sg(), ctx->vvl(), s));
  ctx->launches++;
  return ALEGB_OK;
}

// a1 + a2 of stage `stage` of the step starting at t0 when the coordinates are integrated in time (NEXT-2);
// stage 4 = end of the step (x_n <- x_{n+1}, no geometry)
int update_geometry_rk(alegb_ctx* ctx, int stage, double t0, double dt, cudaStream_t s, const double* ts_dev) {
  const int dim = ctx->ref.dim;
  const double* uvv = ctx->motion.kind == ALEGB_MOTION_USER ? ctx->d_user_vv : nullptr;
  CU(launch_vertex_rk(dim, ctx->Nverts, ctx->d_X0, ctx->motion, uvv, stage, t0, t0 + 0.5 * dt, t0 + 1.0 * dt, dt, ts_dev,
                      ctx->d_xn, ctx->d_xv, ctx->d_vv, s));
  ctx->launches++;
  if (stage < 4) {
    CU(launch_geometry(dim, ctx->K, ctx->d_EToV, ctx->d_xv, ctx->d_vv, ctx->vg(), ctx->sg(), ctx->vvl(), s));
    ctx->launches++;
  }
  return ALEGB_OK;
}

void fill_common(const alegb_ctx* ctx, StageArgs& a) {
  std::memset(&a, 0, sizeof(a));
  a.K = ctx->K;
  a.vgeo = ctx->vg(); a.sgeo = ctx->sg(); a.vvel = ctx->vvl();
  a.vmapP = ctx->d_vmapP; a.EToB = ctx->d_EToB;
  a.pml_index = ctx->d_pml_index; a.pml_sigma = ctx->d_pml_sigma;
  a.Dt_ops = ctx->d_Dt; a.LIFTt = ctx->d_LIFTt; a.lam = ctx->d_lam; a.fmask = ctx->d_fmask;
  a.Avol = ctx->d_Avol; a.AliftP = ctx->d_AliftP;
  a.c = ctx->c; a.invtau = ctx->invtau;
  for (int k = 0; k < kMaxFields; ++k) a.q_inf[k] = ctx->q_inf[k];
}
void fill_common(const alegb_ctx* ctx, PmlArgs& a) {
  std::memset(&a, 0, sizeof(a));
  a.Kpml = ctx->Kpml; a.pml_elems = ctx->d_pml_elems; a.pml_sigma = ctx->d_pml_sigma;
  a.vgeo = ctx->vg(); a.sgeo = ctx->sg(); a.vvel = ctx->vvl();
  a.vmapP = ctx->d_vmapP; a.EToB = ctx->d_EToB;
  a.Dt_ops = ctx->d_Dt; a.LIFTt = ctx->d_LIFTt; a.lam = ctx->d_lam; a.fmask = ctx->d_fmask;
  a.Avol = ctx->d_Avol; a.AliftP = ctx->d_AliftP;
  a.c = ctx->c;
  for (int k = 0; k < kMaxFields; ++k) a.q_inf[k] = ctx->q_inf[k];
}
// the auxiliary-field part of a stage handed to the stage kernel (LAYER instantiation of stage_pipe.cu)
void layer_from(const PmlArgs& p, LayerArgs& l) {
  l.on = true;
  l.aux_n = p.aux_n; l.acc_in = p.acc_in; l.G_out = p.G_out; l.aux_out = p.aux_out; l.acc_out = p.acc_out;
  l.cx_n = p.cx_n; l.cx_acc = p.cx_acc; l.cx_g = p.cx_g; l.cy_n = p.cy_n; l.cy_acc = p.cy_acc; l.cy_g = p.cy_g;
}
// a8: the DMMA kernel unless the generic kernels were asked for (alegb_set_kernel(1)) or (dim, N) has none
cudaError_t launch_pml_any(const alegb_ctx* ctx, const PmlArgs& p, cudaStream_t s) {
  if (ctx->pml_mma_ok && ctx->kernel_mode != 1) return launch_pml_mma(ctx->ref.dim, ctx->ref.N, p, ctx->ctas(), s);
  return launch_pml(ctx->ref.dim, ctx->ref.N, p, ctx->ctas(), s);
}

int check_ready(alegb_ctx* ctx) {
  if (!ctx) return ALEGB_INVALID_ARG;
  if (ctx->device < 0) return fail(ctx, ALEGB_CUDA_ERROR, "host-only context (no CUDA device): there is no CPU fallback");
  if (!ctx->mesh_ready) return fail(ctx, ALEGB_NOT_READY, "alegb_mesh_upload has not been called");
  if (!ctx->params_ready) return fail(ctx, ALEGB_NOT_READY, "alegb_set_params has not been called");
  cudaError_t e = cudaSetDevice(ctx->device);
  if (e != cudaSuccess) return cuda_fail(ctx, e, "cudaSetDevice");
  return ALEGB_OK;
}

// the fused stage kernel, bracketed by events while profiling is enabled
int timed_stage(alegb_ctx* ctx, const StageArgs& a_in, cudaStream_t s) {
  StageArgs a = a_in;
  // profiling brackets everything the stage launches (the cubature kernel of the optional mode included)
  const bool rec = ctx->profiling && ctx->prof_used + 2 <= 8192;
  if (rec) {
    while (ctx->prof_events.size() < ctx->prof_used + 2) {
      cudaEvent_t ev;
      CU(cudaEventCreate(&ev));
      ctx->prof_events.push_back(ev);
    }
    CU(cudaEventRecord(ctx->prof_events[ctx->prof_used], s));
  }
  if (ctx->relax_mode == ALEGB_RELAX_CUBATURE) {
    // kernel v of the paper (L197): R = P N~(I q_in), read by the stage kernel in place of the collocated N~
    CubArgs cb;
    cb.K = ctx->K; cb.Np = ctx->ref.Np; cb.Nc = ctx->cub.Nc; cb.EB = ctx->cub_EB;
    cb.It = ctx->d_It; cb.Pt = ctx->d_Pt; cb.AI = ctx->d_AI; cb.AP = ctx->d_AP;
    cb.q = a.q_in; cb.R = ctx->d_R; cb.invtau = ctx->invtau;
    // kernel kind 1 (generic DFMA stage kernel) keeps the DFMA cubature kernel: two independent implementations;
    // it is also the only one for a (dim, N) without a DMMA cubature kernel (3-D N = 5)
    if (ctx->kernel_mode == 1 || !ctx->cub_mma_ok) CU(launch_cubature(ctx->ref.dim, cb, ctx->ctas(), s));
    else CU(launch_cubature_mma(ctx->ref.dim, ctx->ref.N, cb, ctx->ctas(), s));
    ctx->launches++;
    a.relax_cub = ctx->d_R;
  }
  const int mode = ctx->kernel_mode;
  if (ctx->pipe_ok && (mode == 0 || mode == 2)) {
    if (a.layer.on) {
      // the quads outside the layer through the plain instantiation (deep ring, small slots), then the quads that
      // touch it through the LAYER instantiation (a8 fused in).  An empty list is not launched: the kernel reads a
      // NULL quad_list as "every quad of the mesh", and a mesh whose every quad touches the layer has no plain list.
      if (ctx->nquads_plain > 0) {
        StageArgs b = a;
        b.layer.on = false; b.quad_list = ctx->d_quads_plain; b.nquads_list = ctx->nquads_plain;
        CU(launch_stage_pipe(ctx->ref.dim, ctx->ref.N, b, ctx->ctas(), s));
        ctx->launches++;
      }
      if (ctx->nquads_layer > 0) {
        a.quad_list = ctx->d_quads_layer; a.nquads_list = ctx->nquads_layer;
        CU(launch_stage_pipe(ctx->ref.dim, ctx->ref.N, a, ctx->ctas(), s));
        ctx->launches++;
      }
    } else {
      CU(launch_stage_pipe(ctx->ref.dim, ctx->ref.N, a, ctx->ctas(), s));
      ctx->launches++;
    }
  } else {
    CU(launch_stage(ctx->ref.dim, ctx->ref.N, a, ctx->ctas(), s));
    ctx->launches++;
  }
  if (rec) {
    CU(cudaEventRecord(ctx->prof_events[ctx->prof_used + 1], s));
    ctx->prof_used += 2;
  }
  return ALEGB_OK;
}

// One SARK4 step.  q_n: state at t0 (read only); outs[i]: where stage state i+1 is written
// (outs[3] = q_{n+1}, may alias q_n).
int sark_step(alegb_ctx* ctx, const double* q_n, double* const outs[4], double t0, double dt, cudaStream_t s,
              const double* t_dev = nullptr, bool advance_coords = true) {
  const int dim = ctx->ref.dim, N = ctx->ref.N, Nf = ctx->Nf;
  const double gamma = -dt * ctx->invtau;  // L144
  double as[6], bs[4], a0[6], b0[4];
  sark_coefficients(gamma, as, bs);
  sark_coefficients(0.0, a0, b0);
  bool stiff[kMaxFields];
  double e_half[kMaxFields], e_full[kMaxFields];
  for (int k = 0; k < Nf; ++k) {
    stiff[k] = k > dim;  // second-order moments (L115)
    const double lam = stiff[k] ? ctx->invtau : 0.0;
    e_half[k] = std::exp(-(lam * 0.5) * dt);
    e_full[k] = std::exp(-(lam * 1.0) * dt);
  }
  auto A = [&](int k, int idx) { return stiff[k] ? as[idx] : a0[idx]; };  // idx: 0 a10, 1 a20, 2 a21, 3 a30, 5 a32
  auto B = [&](int k, int j) { return stiff[k] ? bs[j] : b0[j]; };
  const double cstage[4] = {0.0, 0.5, 0.5, 1.0};
  const bool pml = ctx->Kpml > 0;
  const bool overlap = ctx->overlap_geometry;
  if (overlap && !ctx->geo_stream) {
    CU(cudaStreamCreateWithFlags(&ctx->geo_stream, cudaStreamNonBlocking));
    CU(cudaEventCreateWithFlags(&ctx->ev_fork, cudaEventDisableTiming));
    for (int i = 0; i < 4; ++i) {
      CU(cudaEventCreateWithFlags(&ctx->ev_geo[i], cudaEventDisableTiming));
      CU(cudaEventCreateWithFlags(&ctx->ev_stage[i], cudaEventDisableTiming));
    }
  }
  for (int i = 0; i < 4; ++i) {
    const double ti = t0 + cstage[i] * dt;
    // a1 + a2 of stage `j` into geometry set j & 1, on stream `gs`
    auto geometry_of = [&](int j, cudaStream_t gs) {
      ctx->geo_buf = j & 1;
      const double tj = t0 + cstage[j] * dt;
      return ctx->coord_mode == ALEGB_COORDS_RK ? update_geometry_rk(ctx, j, t0, dt, gs, t_dev)
                                                 : update_geometry(ctx, tj, gs, t_dev ? t_dev + j : nullptr, j);
    };
    (void)ti;
    int rc = ALEGB_OK;
    if (i == 0) {
      rc = geometry_of(0, s);
      if (rc == ALEGB_OK && overlap) {      // fork: the side stream starts after stage 0's geometry
        CU(cudaEventRecord(ctx->ev_fork, s));
        CU(cudaStreamWaitEvent(ctx->geo_stream, ctx->ev_fork, 0));
      }
    } else if (overlap) {
      CU(cudaStreamWaitEvent(s, ctx->ev_geo[i], 0));
    } else {
      rc = geometry_of(i, s);
    }
    if (rc != ALEGB_OK) return rc;
    if (overlap && i < 3) {
      // stage i+1's geometry beside stage i's kernels; its arrays were last read by stage i-1
      if (i >= 1) CU(cudaStreamWaitEvent(ctx->geo_stream, ctx->ev_stage[i - 1], 0));
      rc = geometry_of(i + 1, ctx->geo_stream);
      if (rc != ALEGB_OK) return rc;
      CU(cudaEventRecord(ctx->ev_geo[i + 1], ctx->geo_stream));
    }
    ctx->geo_buf = i & 1;
    StageArgs a;
    fill_common(ctx, a);
    a.q_in = i == 0 ? q_n : outs[i - 1];
    a.q_out = outs[i];
    a.aux = pml ? (i == 0 ? ctx->d_AUX : ctx->d_AUXS) : nullptr;
    StageCoef& cf = a.coef;
    if (i == 0) {
      a.q_n = q_n; a.F_out = ctx->d_F0;
      for (int k = 0; k < Nf; ++k) { cf.cq_n[k] = e_half[k]; cf.cq_f[k] = dt * A(k, 0); }
    } else if (i == 1) {
      a.q_n = q_n; a.F0_in = ctx->d_F0; a.acc_out = ctx->d_ACC;
      for (int k = 0; k < Nf; ++k) {
        cf.cq_n[k] = e_half[k]; cf.cq_f0[k] = dt * A(k, 1); cf.cq_f[k] = dt * A(k, 2);
        cf.ca_n[k] = e_full[k]; cf.ca_f0[k] = dt * B(k, 0); cf.ca_f[k] = dt * B(k, 1);
      }
    } else if (i == 2) {
      a.q_n = q_n; a.F0_in = ctx->d_F0; a.acc_in = ctx->d_ACC; a.acc_out = ctx->d_ACC;
      cf.ca_acc = 1.0;
      for (int k = 0; k < Nf; ++k) {
        cf.cq_n[k] = e_full[k]; cf.cq_f0[k] = dt * A(k, 3); cf.cq_f[k] = dt * A(k, 5);
        cf.ca_f[k] = dt * B(k, 2);
      }
    } else {
      a.acc_in = ctx->d_ACC;
      cf.cq_acc = 1.0;
      for (int k = 0; k < Nf; ++k) cf.cq_f[k] = dt * B(k, 3);
    }
    PmlArgs p;
    if (pml) {
      // auxiliary fields: Lambda = 0, classic RK4 weights (reading R12)
      fill_common(ctx, p);
      p.q_in = a.q_in;
      p.aux_in = i == 0 ? ctx->d_AUX : ctx->d_AUXS;
      if (i < 3) {
        p.aux_n = ctx->d_AUX; p.aux_out = ctx->d_AUXS; p.acc_out = ctx->d_AUXACC;
        p.cx_n = 1.0; p.cx_g = dt * (i == 2 ? 1.0 : 0.5);
        if (i == 0) { p.cy_n = 1.0; p.cy_g = dt * (1.0 / 6.0); }
        else { p.acc_in = ctx->d_AUXACC; p.cy_acc = 1.0; p.cy_g = dt * (1.0 / 3.0); }
      } else {
        p.acc_in = ctx->d_AUXACC; p.aux_out = ctx->d_AUX; p.cx_acc = 1.0; p.cx_g = dt * (1.0 / 6.0);
      }
      if (ctx->layer_fused()) layer_from(p, a.layer);   // a8 inside the stage kernel
    }
    rc = timed_stage(ctx, a, s);
    if (rc != ALEGB_OK) return rc;
    if (pml && !a.layer.on) {
      CU(launch_pml_any(ctx, p, s));
      ctx->launches++;
    }
    if (overlap) CU(cudaEventRecord(ctx->ev_stage[i], s));
  }
  ctx->geo_buf = 0;
  if (ctx->coord_mode == ALEGB_COORDS_RK && advance_coords) return update_geometry_rk(ctx, 4, t0, dt, s, t_dev);
  return ALEGB_OK;
}

void drop_step_graph(alegb_ctx* ctx) {
  if (ctx->step_graph) cudaGraphExecDestroy(ctx->step_graph);
  ctx->step_graph = nullptr;
}

// nsteps SARK4 steps as nsteps launches of ONE captured graph (clock kernel + the 12-16 launches of a step): removes
// the per-launch host cost that bounds the small, L2-resident configurations.  The graph is captured on a stream of
// the library's own (the caller's may be the legacy default stream, which cannot be captured) and launched on the
// caller's stream; it is rebuilt when the state pointer, dt or anything a step launches changes (t0 lives on the device).
int step_graph_launch(alegb_ctx* ctx, double* d_q, double* const outs[4], double t0, double dt, int nsteps, cudaStream_t s) {
  if (!ctx->capture_stream) CU(cudaStreamCreateWithFlags(&ctx->capture_stream, cudaStreamNonBlocking));
  if (!ctx->d_clock) {
    CU(dev_alloc(ctx, &ctx->d_clock, 6));
    CU(dev_alloc(ctx, &ctx->d_step_counter, 1));
  }
  auto& key = ctx->graph_key;
  if (!ctx->step_graph || key.d_q != d_q || key.dt != dt || key.version != ctx->config_version) {
    drop_step_graph(ctx);
    const int64_t before = ctx->launches;
    cudaGraph_t graph = nullptr;
    if (cudaStreamBeginCapture(ctx->capture_stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
      cudaGetLastError();
      return ALEGB_UNSUPPORTED;
    }
    int rc = ALEGB_OK;
    if (launch_step_clock(ctx->d_clock, ctx->d_step_counter, ctx->capture_stream) != cudaSuccess) rc = ALEGB_CUDA_ERROR;
    if (rc == ALEGB_OK) rc = sark_step(ctx, d_q, outs, t0, dt, ctx->capture_stream, ctx->d_clock + 2);
    cudaError_t e = cudaStreamEndCapture(ctx->capture_stream, &graph);
    key.launches = ctx->launches - before + 1;
    ctx->launches = before;
    if (rc != ALEGB_OK || e != cudaSuccess || graph == nullptr) {
      if (graph) cudaGraphDestroy(graph);
      cudaGetLastError();
      return rc != ALEGB_OK ? rc : ALEGB_UNSUPPORTED;
    }
    e = cudaGraphInstantiate(&ctx->step_graph, graph, 0);
    cudaGraphDestroy(graph);
    if (e != cudaSuccess) { ctx->step_graph = nullptr; cudaGetLastError(); return ALEGB_UNSUPPORTED; }
    key.d_q = d_q; key.dt = dt; key.version = ctx->config_version;
  }
  CU(launch_step_clock_set(ctx->d_clock, ctx->d_step_counter, t0, dt, s));
  for (int n = 0; n < nsteps; ++n) CU(cudaGraphLaunch(ctx->step_graph, s));
  ctx->launches += key.launches * nsteps + 1;
  return ALEGB_OK;
}

}  // namespace

extern "C" {

int alegb_create(alegb_ctx** out, int dim, int N, int cuda_device) {
  if (!out) return ALEGB_INVALID_ARG;
  *out = nullptr;
  if (dim != 2 && dim != 3) return ALEGB_INVALID_ARG;
  if (N < 1 || N > ALEGB_MAX_N) return ALEGB_UNSUPPORTED;
  alegb_ctx* ctx = new (std::nothrow) alegb_ctx();
  if (!ctx) return ALEGB_INVALID_ARG;
  std::string err;
  if (!build_reference(dim, N, ctx->ref, err)) { delete ctx; return ALEGB_INVALID_ARG; }
  ctx->Nf = dim == 2 ? 6 : 10;
  ctx->device = cuda_device;
  ctx->motion.kind = ALEGB_MOTION_NONE;
  if (cuda_device < 0) {  // host-only context: setup and introspection work, every compute call fails
    *out = ctx;
    return ALEGB_OK;
  }
  cudaError_t e = cudaSetDevice(cuda_device);
  cudaDeviceProp prop;
  if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, cuda_device);
  if (e == cudaSuccess) e = configure_kernels(dim, N);
  if (e != cudaSuccess) { delete ctx; return ALEGB_CUDA_ERROR; }
  ctx->num_sms = prop.multiProcessorCount;
  const RefElement& r = ctx->ref;
  const int Np = r.Np, ncol = r.Nfaces * r.Nfp;
  std::vector<double> Dt((size_t)dim * Np * Np), Lt((size_t)ncol * Np);
  for (int a = 0; a < dim; ++a)
    for (int i = 0; i < Np; ++i)
      for (int j = 0; j < Np; ++j) Dt[((size_t)a * Np + j) * Np + i] = r.D[a][i * Np + j];
  for (int i = 0; i < Np; ++i)
    for (int m = 0; m < ncol; ++m) Lt[(size_t)m * Np + i] = r.LIFT[i * ncol + m];
  std::vector<int32_t> fm(r.fmask.begin(), r.fmask.end());
  // operators in DMMA fragment order: lane l of fragment (row tile nb, k-step ks) holds A[8 nb + l/4][4 ks + l%4]
  struct { int NB, KS; } L{(Np + 7) / 8, (Np + 3) / 4};   // node blocks of 8 rows, k-steps of 4 columns
  ctx->pipe_ok = configure_stage_pipe(dim, N) == cudaSuccess;
  ctx->pml_mma_ok = configure_pml_mma(dim, N) == cudaSuccess;
  ctx->pipe_layer_ok = ctx->pipe_ok && stage_pipe_layer_supported(dim, N);
  // measured (profiles/r2_layer_fusion.md): config 5 (3-D N=3) 32.4 -> 34.3 GDOF-stage/s fused, config 3 (2-D N=4)
  // 69.5 -> 63.5: the 2-D layer is a thin ring and a second small launch costs more than the fusion saves
  ctx->fuse_layer = dim == 3;
  cudaGetLastError();
  if (ctx->pipe_ok || ctx->pml_mma_ok) {
    std::vector<double> Av((size_t)dim * L.NB * L.KS * 32, 0.0);
    for (int a = 0; a < dim; ++a)
      for (int nb = 0; nb < L.NB; ++nb)
        for (int ks = 0; ks < L.KS; ++ks)
          for (int l = 0; l < 32; ++l) {
            const int row = 8 * nb + l / 4, col = 4 * ks + l % 4;
            if (row < Np && col < Np) Av[(((size_t)a * L.NB + nb) * L.KS + ks) * 32 + l] = r.D[a][row * Np + col];
          }
    const int KFT = (ncol + 3) / 4;   // the faces' k ranges packed back to back, m = f*Nfp + mm
    std::vector<double> Alp((size_t)L.NB * KFT * 32, 0.0);
    for (int nb = 0; nb < L.NB; ++nb)
      for (int ks = 0; ks < KFT; ++ks)
        for (int l = 0; l < 32; ++l) {
          const int row = 8 * nb + l / 4, m = 4 * ks + l % 4;
          if (row < Np && m < ncol) Alp[((size_t)nb * KFT + ks) * 32 + l] = r.LIFT[row * ncol + m];
        }
    if (upload(ctx, &ctx->d_Avol, Av.data(), Av.size()) != cudaSuccess ||
        upload(ctx, &ctx->d_AliftP, Alp.data(), Alp.size()) != cudaSuccess) {
      alegb_destroy(ctx);
      return ALEGB_CUDA_ERROR;
    }
  }
  if (upload(ctx, &ctx->d_Dt, Dt.data(), Dt.size()) != cudaSuccess ||
      upload(ctx, &ctx->d_LIFTt, Lt.data(), Lt.size()) != cudaSuccess ||
      upload(ctx, &ctx->d_lam, r.lam.data(), r.lam.size()) != cudaSuccess ||
      upload(ctx, &ctx->d_fmask, fm.data(), fm.size()) != cudaSuccess ||
      upload(ctx, &ctx->d_wface, r.wface.data(), r.wface.size()) != cudaSuccess) {
    alegb_destroy(ctx);
    return ALEGB_CUDA_ERROR;
  }
  *out = ctx;
  return ALEGB_OK;
}

int alegb_destroy(alegb_ctx* ctx) {
  if (!ctx) return ALEGB_INVALID_ARG;
  if (ctx->device >= 0) {
    cudaSetDevice(ctx->device);
    cudaDeviceSynchronize();
  }
  free_mesh(ctx);
  drop_step_graph(ctx);
  if (ctx->capture_stream) cudaStreamDestroy(ctx->capture_stream);
  if (ctx->geo_stream) cudaStreamDestroy(ctx->geo_stream);
  if (ctx->ev_fork) cudaEventDestroy(ctx->ev_fork);
  for (int i = 0; i < 4; ++i) {
    if (ctx->ev_geo[i]) cudaEventDestroy(ctx->ev_geo[i]);
    if (ctx->ev_stage[i]) cudaEventDestroy(ctx->ev_stage[i]);
  }
  dev_free(ctx->d_clock); dev_free(ctx->d_step_counter);
  for (cudaEvent_t ev : ctx->prof_events) cudaEventDestroy(ev);
  dev_free(ctx->d_Dt); dev_free(ctx->d_LIFTt); dev_free(ctx->d_lam); dev_free(ctx->d_fmask);
  dev_free(ctx->d_wface); dev_free(ctx->d_force);
  dev_free(ctx->d_Avol); dev_free(ctx->d_AliftP);
  dev_free(ctx->d_It); dev_free(ctx->d_Pt); dev_free(ctx->d_AI); dev_free(ctx->d_AP);
  delete ctx;
  return ALEGB_OK;
}

int alegb_mesh_upload(alegb_ctx* ctx, int64_t Nverts, const double* X0, int64_t K, const int32_t* EToV,
                      const int32_t* vertex_equiv, const int8_t* EToB, const double* pml_sigma) {
  if (!ctx) return ALEGB_INVALID_ARG;
  if (!X0 || !EToV || Nverts <= 0 || K <= 0) return fail(ctx, ALEGB_INVALID_ARG, "X0/EToV missing or empty mesh");
  if (ctx->device >= 0) CU(cudaSetDevice(ctx->device));
  const RefElement& r = ctx->ref;
  const int dim = r.dim, nv = dim + 1, Np = r.Np, Nf = ctx->Nf;
  for (int64_t i = 0; i < K * nv; ++i)
    if (EToV[i] < 0 || EToV[i] >= Nverts) return fail(ctx, ALEGB_BAD_MESH, "EToV entry out of range");
  if (vertex_equiv)
    for (int64_t i = 0; i < Nverts; ++i)
      if (vertex_equiv[i] < 0 || vertex_equiv[i] >= Nverts) return fail(ctx, ALEGB_BAD_MESH, "vertex_equiv entry out of range");
  // positive orientation at t = 0 (L73)
  for (int64_t e = 0; e < K; ++e) {
    double G[3][3];
    for (int a = 0; a < dim; ++a)
      for (int d = 0; d < dim; ++d) G[d][a] = 0.5 * (X0[(int64_t)EToV[e * nv + a + 1] * dim + d] - X0[(int64_t)EToV[e * nv] * dim + d]);
    double J = dim == 2 ? G[0][0] * G[1][1] - G[0][1] * G[1][0]
                        : G[0][0] * (G[1][1] * G[2][2] - G[1][2] * G[2][1]) - G[0][1] * (G[1][0] * G[2][2] - G[1][2] * G[2][0]) +
                              G[0][2] * (G[1][0] * G[2][1] - G[1][1] * G[2][0]);
    if (!(J > 0.0)) return fail(ctx, ALEGB_BAD_MESH, "element " + std::to_string(e) + " has a non-positive Jacobian at t = 0");
  }
  Connectivity conn;
  std::string err;
  int rc = build_connectivity(r, K, EToV, vertex_equiv, EToB, conn, err);
  if (rc != 0) return fail(ctx, ALEGB_BAD_MESH, err);
  free_mesh(ctx);
  ctx->K = K; ctx->Nverts = Nverts;
  bool any_tag = false;
  if (EToB) for (int64_t i = 0; i < K * nv; ++i) any_tag |= EToB[i] != 0;
  ctx->has_boundary = any_tag;
  // absorbing layer: compact list of flagged elements
  std::vector<int32_t> pml_index;
  std::vector<double> sig;
  ctx->pml_elems_host.clear();
  if (pml_sigma) {
    pml_index.assign(K, -1);
    for (int64_t e = 0; e < K; ++e) {
      bool in = false;
      for (int d = 0; d < dim; ++d) {
        if (pml_sigma[e * dim + d] < 0.0) return fail(ctx, ALEGB_INVALID_ARG, "negative pml_sigma");
        in |= pml_sigma[e * dim + d] > 0.0;
      }
      if (in) {
        pml_index[e] = (int32_t)ctx->pml_elems_host.size();
        ctx->pml_elems_host.push_back((int32_t)e);
        for (int d = 0; d < dim; ++d) sig.push_back(pml_sigma[e * dim + d]);
      }
    }
  }
  ctx->Kpml = (int64_t)ctx->pml_elems_host.size();
  ctx->vmapM_host = conn.vmapM; ctx->vmapP_host = conn.vmapP;
  if (ctx->device < 0) {  // host-only context: connectivity is available for introspection, nothing else
    ctx->mesh_ready = true;
    return ALEGB_OK;
  }
  const size_t state = (size_t)K * Nf * Np;
  CU(upload(ctx, &ctx->d_X0, X0, (size_t)Nverts * dim));
  CU(dev_alloc(ctx, &ctx->d_xv, (size_t)Nverts * dim));
  CU(dev_alloc(ctx, &ctx->d_vv, (size_t)Nverts * dim));
  CU(upload(ctx, &ctx->d_EToV, EToV, (size_t)K * nv));
  CU(upload(ctx, &ctx->d_vmapP, conn.vmapP.data(), conn.vmapP.size()));
  if (any_tag) CU(upload(ctx, &ctx->d_EToB, EToB, (size_t)K * nv));
  CU(dev_alloc(ctx, &ctx->d_vgeo, (size_t)K * (dim * dim + 1)));
  CU(dev_alloc(ctx, &ctx->d_sgeo, (size_t)K * nv * (dim + 2)));
  CU(dev_alloc(ctx, &ctx->d_vvel, (size_t)K * nv * dim));
  CU(dev_alloc(ctx, &ctx->d_vgeo1, (size_t)K * (dim * dim + 1)));
  CU(dev_alloc(ctx, &ctx->d_sgeo1, (size_t)K * nv * (dim + 2)));
  CU(dev_alloc(ctx, &ctx->d_vvel1, (size_t)K * nv * dim));
  CU(dev_alloc(ctx, &ctx->d_Q1, state));
  CU(dev_alloc(ctx, &ctx->d_Q2, state));
  CU(dev_alloc(ctx, &ctx->d_F0, state));
  CU(dev_alloc(ctx, &ctx->d_ACC, state));
  if (ctx->Kpml > 0) {
    const size_t na = (size_t)ctx->Kpml * dim * Nf * Np;
    CU(upload(ctx, &ctx->d_pml_index, pml_index.data(), pml_index.size()));
    CU(upload(ctx, &ctx->d_pml_elems, ctx->pml_elems_host.data(), ctx->pml_elems_host.size()));
    CU(upload(ctx, &ctx->d_pml_sigma, sig.data(), sig.size()));
    {   // quads of 4 consecutive elements, split by whether any of them lies in the layer
      std::vector<int32_t> ql, qp;
      for (int64_t qd = 0; qd < (K + 3) / 4; ++qd) {
        bool in = false;
        for (int64_t e = 4 * qd; e < K && e < 4 * qd + 4; ++e) in |= pml_index[e] >= 0;
        (in ? ql : qp).push_back((int32_t)qd);
      }
      ctx->nquads_layer = (int64_t)ql.size(); ctx->nquads_plain = (int64_t)qp.size();
      CU(upload(ctx, &ctx->d_quads_layer, ql.data(), ql.size()));
      CU(upload(ctx, &ctx->d_quads_plain, qp.data(), qp.size()));
    }
    CU(dev_alloc(ctx, &ctx->d_AUX, na));
    CU(dev_alloc(ctx, &ctx->d_AUXS, na));
    CU(dev_alloc(ctx, &ctx->d_AUXACC, na));
    CU(cudaMemset(ctx->d_AUX, 0, na * sizeof(double)));
  }
  CU(cudaMemcpy(ctx->d_xv, ctx->d_X0, (size_t)Nverts * dim * sizeof(double), cudaMemcpyDeviceToDevice));
  CU(cudaMemset(ctx->d_vv, 0, (size_t)Nverts * dim * sizeof(double)));
  CU(cudaDeviceSynchronize());
  ctx->mesh_ready = true;
  return ALEGB_OK;
}

int alegb_set_params(alegb_ctx* ctx, double RT, double tau, const double* q_inf) {
  if (!ctx) return ALEGB_INVALID_ARG;
  if (!(RT > 0.0) || !(tau > 0.0)) return fail(ctx, ALEGB_INVALID_ARG, "RT and tau must be positive");
  ctx->RT = RT; ctx->tau = tau; ctx->c = std::sqrt(RT);
  ctx->invtau = std::isinf(tau) ? 0.0 : 1.0 / tau;
  for (int k = 0; k < kMaxFields; ++k) ctx->q_inf[k] = 0.0;
  if (q_inf) for (int k = 0; k < ctx->Nf; ++k) ctx->q_inf[k] = q_inf[k];
  ctx->params_ready = true;
  ctx->config_version++;
  return ALEGB_OK;
}

int alegb_set_motion(alegb_ctx* ctx, int kind, const double* params, int nparams) {
  if (!ctx) return ALEGB_INVALID_ARG;
  const int dim = ctx->ref.dim;
  int need = 0;
  switch (kind) {
    case ALEGB_MOTION_NONE: need = 0; break;
    case ALEGB_MOTION_SINES_PRODUCT: need = 2 + 2 * dim; break;
    case ALEGB_MOTION_SINES_CROSS: need = 4; break;
    case ALEGB_MOTION_PLUNGE_BLEND: need = 5 + dim; break;
    case ALEGB_MOTION_CARANGIFORM: need = 10; break;
    default: return fail(ctx, ALEGB_INVALID_ARG, "unknown motion kind (USER is set by alegb_set_motion_user)");
  }
  if (nparams < need || (need > 0 && !params)) return fail(ctx, ALEGB_INVALID_ARG, "too few motion parameters");
  if (kind == ALEGB_MOTION_PLUNGE_BLEND || kind == ALEGB_MOTION_CARANGIFORM) {
    int axis = (int)params[kind == ALEGB_MOTION_PLUNGE_BLEND ? 4 : 8];
    if (axis < 0 || axis >= dim) return fail(ctx, ALEGB_INVALID_ARG, "motion axis out of range");
  }
  ctx->motion.kind = kind; ctx->motion.nparams = need;
  for (int i = 0; i < 16; ++i) ctx->motion.p[i] = i < need ? params[i] : 0.0;
  ctx->config_version++;
  return ALEGB_OK;
}

// kind USER: stage data [4][Nverts*dim]; `stride` = 0 replicates one array over the four stages
static int set_user_motion(alegb_ctx* ctx, const double* d_xv, const double* d_vv, size_t stride) {
  if (!ctx) return ALEGB_INVALID_ARG;
  if (ctx->device < 0) return fail(ctx, ALEGB_CUDA_ERROR, "host-only context (no CUDA device)");
  if (!ctx->mesh_ready) return fail(ctx, ALEGB_NOT_READY, "alegb_mesh_upload has not been called");
  if (!d_vv) return fail(ctx, ALEGB_INVALID_ARG, "NULL device array");
  if (!d_xv && !ctx->d_user_xv) return fail(ctx, ALEGB_INVALID_ARG, "positions are required the first time");
  CU(cudaSetDevice(ctx->device));
  const size_t n = (size_t)ctx->Nverts * ctx->ref.dim, bytes = n * sizeof(double);
  if (!ctx->d_user_xv) CU(dev_alloc(ctx, &ctx->d_user_xv, 4 * n));
  if (!ctx->d_user_vv) CU(dev_alloc(ctx, &ctx->d_user_vv, 4 * n));
  // The buffers about to be overwritten are read by every a1 / a2 launch of a step, on the caller's stepping stream
  // and on the library's side stream (the step graph keeps their addresses): wait for whatever is still in flight on
  // ANY stream, non-blocking ones included, before the copies below go out on the default stream.  The same wait
  // makes the caller's arrays visible if a kernel on another stream produced them.
  CU(cudaDeviceSynchronize());
  for (int i = 0; i < 4; ++i) {
    if (d_xv) CU(cudaMemcpyAsync(ctx->d_user_xv + i * n, d_xv + i * stride, bytes, cudaMemcpyDeviceToDevice, 0));
    CU(cudaMemcpyAsync(ctx->d_user_vv + i * n, d_vv + i * stride, bytes, cudaMemcpyDeviceToDevice, 0));
  }
  // the library's "current" vertices (alegb_geometry / alegb_get_positions outputs): the first stage
  CU(cudaMemcpyAsync(ctx->d_xv, ctx->d_user_xv, bytes, cudaMemcpyDeviceToDevice, 0));
  CU(cudaMemcpyAsync(ctx->d_vv, ctx->d_user_vv, bytes, cudaMemcpyDeviceToDevice, 0));
  CU(cudaStreamSynchronize(0));
  if (ctx->motion.kind != ALEGB_MOTION_USER) ctx->config_version++;   // the step graph reads the library's own buffers
  ctx->motion.kind = ALEGB_MOTION_USER;
  return ALEGB_OK;
}

int alegb_set_motion_user(alegb_ctx* ctx, const double* d_xv, const double* d_vv) {
  if (ctx && !d_xv) return fail(ctx, ALEGB_INVALID_ARG, "NULL device array");
  return set_user_motion(ctx, d_xv, d_vv, 0);
}

int alegb_set_motion_user_stages(alegb_ctx* ctx, const double* d_xv4, const double* d_vv4) {
  if (!ctx) return ALEGB_INVALID_ARG;
  return set_user_motion(ctx, d_xv4, d_vv4, (size_t)ctx->Nverts * ctx->ref.dim);
}

static int ensure_cubature(alegb_ctx* ctx) {
  if (ctx->cub.Nc > 0) return ALEGB_OK;
  std::string err;
  if (!build_cubature(ctx->ref, 3 * ctx->ref.N, ctx->cub, err)) return fail(ctx, ALEGB_INVALID_ARG, err);
  return ALEGB_OK;
}

int alegb_set_relaxation(alegb_ctx* ctx, int mode) {
  if (!ctx) return ALEGB_INVALID_ARG;
  if (mode != ALEGB_RELAX_COLLOCATION && mode != ALEGB_RELAX_CUBATURE) return fail(ctx, ALEGB_INVALID_ARG, "unknown relaxation mode");
  if (mode == ALEGB_RELAX_CUBATURE) {
    if (ctx->device < 0) return fail(ctx, ALEGB_CUDA_ERROR, "host-only context (no CUDA device)");
    if (!ctx->mesh_ready) return fail(ctx, ALEGB_NOT_READY, "alegb_mesh_upload has not been called");
    int rc = ensure_cubature(ctx);
    if (rc != ALEGB_OK) return rc;
    CU(cudaSetDevice(ctx->device));
    const int dim = ctx->ref.dim, Np = ctx->ref.Np, Nc = ctx->cub.Nc, NS = dim * (dim + 1) / 2;
    if (!ctx->d_It) {
      std::vector<double> It((size_t)Np * Nc), Pt((size_t)Nc * Np);
      for (int c = 0; c < Nc; ++c) for (int j = 0; j < Np; ++j) {
        It[(size_t)j * Nc + c] = ctx->cub.I[(size_t)c * Np + j];
        Pt[(size_t)c * Np + j] = ctx->cub.P[(size_t)j * Nc + c];
      }
      CU(dev_alloc(ctx, &ctx->d_It, It.size()));
      CU(dev_alloc(ctx, &ctx->d_Pt, Pt.size()));
      CU(cudaMemcpy(ctx->d_It, It.data(), It.size() * sizeof(double), cudaMemcpyHostToDevice));
      CU(cudaMemcpy(ctx->d_Pt, Pt.data(), Pt.size() * sizeof(double), cudaMemcpyHostToDevice));
      ctx->cub_mma_ok = cubature_mma_available(dim, ctx->ref.N);
      if (ctx->cub_mma_ok) {   // A-fragment order: lane l of fragment (row tile, k-step) holds A[8 tile + l/4][4 k + l%4], zero outside
        int NRT, KS, NB;
        cubature_mma_layout(dim, ctx->ref.N, NRT, KS, NB);
        std::vector<double> AI((size_t)NRT * KS * 32, 0.0), AP((size_t)NB * 2 * NRT * 32, 0.0);
        for (int rt = 0; rt < NRT; ++rt) for (int ks = 0; ks < KS; ++ks) for (int l = 0; l < 32; ++l) {
          const int row = 8 * rt + l / 4, col = 4 * ks + l % 4;
          if (row < Nc && col < Np) AI[((size_t)rt * KS + ks) * 32 + l] = ctx->cub.I[(size_t)row * Np + col];
        }
        for (int r = 0; r < NB; ++r) for (int k = 0; k < 2 * NRT; ++k) for (int l = 0; l < 32; ++l) {
          const int row = 8 * r + l / 4, col = 4 * k + l % 4;
          if (row < Np && col < Nc) AP[((size_t)r * 2 * NRT + k) * 32 + l] = ctx->cub.P[(size_t)row * Nc + col];
        }
        CU(dev_alloc(ctx, &ctx->d_AI, AI.size()));
        CU(dev_alloc(ctx, &ctx->d_AP, AP.size()));
        CU(cudaMemcpy(ctx->d_AI, AI.data(), AI.size() * sizeof(double), cudaMemcpyHostToDevice));
        CU(cudaMemcpy(ctx->d_AP, AP.data(), AP.size() * sizeof(double), cudaMemcpyHostToDevice));
      }
      int EB = 256 / Np;
      while (EB > 1 && cubature_smem_bytes(dim, Np, Nc, EB) > 200 * 1024) --EB;
      ctx->cub_EB = EB;
      CU(configure_cubature(dim, cubature_smem_bytes(dim, Np, Nc, EB)));
    }
    if (!ctx->d_R) CU(dev_alloc(ctx, &ctx->d_R, (size_t)ctx->K * NS * Np));
  }
  ctx->relax_mode = mode;
  ctx->config_version++;
  return ALEGB_OK;
}

int alegb_get_cubature(alegb_ctx* ctx, int* degree, int* Nc, double* rst, double* w, double* I, double* P) {
  if (!ctx) return ALEGB_INVALID_ARG;
  int rc = ensure_cubature(ctx);
  if (rc != ALEGB_OK) return rc;
  const Cubature& c = ctx->cub;
  if (degree) *degree = c.degree;
  if (Nc) *Nc = c.Nc;
  if (rst) std::memcpy(rst, c.rst.data(), c.rst.size() * sizeof(double));
  if (w) std::memcpy(w, c.w.data(), c.w.size() * sizeof(double));
  if (I) std::memcpy(I, c.I.data(), c.I.size() * sizeof(double));
  if (P) std::memcpy(P, c.P.data(), c.P.size() * sizeof(double));
  return ALEGB_OK;
}

int alegb_wall_forces(alegb_ctx* ctx, double t, const double* d_q, int tag, double* h_Fp, double* h_Fv, void* stream) {
  int rc = check_ready(ctx);
  if (rc != ALEGB_OK) return rc;
  if (!d_q || !h_Fp || !h_Fv) return fail(ctx, ALEGB_INVALID_ARG, "NULL pointer");
  if (tag < 1 || tag > 127) return fail(ctx, ALEGB_INVALID_ARG, "tag must be a boundary tag (1..127)");
  const int dim = ctx->ref.dim;
  for (int d = 0; d < dim; ++d) h_Fp[d] = h_Fv[d] = 0.0;
  if (!ctx->d_EToB) return ALEGB_OK;                    // no tagged faces at all
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  constexpr int kBlocks = 296;
  if (!ctx->d_force) CU(dev_alloc(ctx, &ctx->d_force, (size_t)(kBlocks + 1) * 6));
  rc = update_geometry(ctx, t, s);
  if (rc != ALEGB_OK) return rc;
  CU(launch_wall_force(dim, ctx->K, ctx->d_EToB, tag, d_q, ctx->d_sgeo, ctx->d_fmask, ctx->d_wface, ctx->ref.Np,
                       ctx->ref.Nfp, ctx->RT, ctx->d_force, kBlocks, ctx->d_force + (size_t)kBlocks * 6, s));
  ctx->launches += 2;
  double out[6];
  CU(cudaMemcpyAsync(out, ctx->d_force + (size_t)kBlocks * 6, 2 * dim * sizeof(double), cudaMemcpyDeviceToHost, s));
  CU(cudaStreamSynchronize(s));
  for (int d = 0; d < dim; ++d) { h_Fp[d] = out[d]; h_Fv[d] = out[dim + d]; }
  return ALEGB_OK;
}

// The no-allocation form of alegb_wall_forces (include/alegb.h): partial sums in the library's static device array
// (kernels.cu), result left on the device, nothing allocated, nothing synchronised.
int alegb_wall_forces_static(alegb_ctx* ctx, double t, const double* d_q, int tag, int nblocks, double* d_F,
                             void* stream) {
  int rc = check_ready(ctx);
  if (rc != ALEGB_OK) return rc;
  if (!d_q || !d_F) return fail(ctx, ALEGB_INVALID_ARG, "NULL pointer");
  if (tag < 1 || tag > 127) return fail(ctx, ALEGB_INVALID_ARG, "tag must be a boundary tag (1..127)");
  if (nblocks == 0) nblocks = 296;                      // the grid of alegb_wall_forces
  if (nblocks < 0) return fail(ctx, ALEGB_INVALID_ARG, "nblocks must be 0 (default) or positive");
  if (nblocks > ALEGB_WALL_FORCES_STATIC_MAX_BLOCKS)
    return fail(ctx, ALEGB_INVALID_ARG,
                "nblocks = " + std::to_string(nblocks) + " does not fit the static partial-sum array: the limit is "
                "ALEGB_WALL_FORCES_STATIC_MAX_BLOCKS = " + std::to_string(ALEGB_WALL_FORCES_STATIC_MAX_BLOCKS));
  const int dim = ctx->ref.dim;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  if (!ctx->d_EToB) {                                   // no tagged faces at all
    CU(cudaMemsetAsync(d_F, 0, 2 * dim * sizeof(double), s));
    return ALEGB_OK;
  }
  rc = update_geometry(ctx, t, s);
  if (rc != ALEGB_OK) return rc;
  CU(launch_wall_force_static(dim, ctx->K, ctx->d_EToB, tag, d_q, ctx->sg(), ctx->d_fmask, ctx->d_wface, ctx->ref.Np,
                              ctx->ref.Nfp, ctx->RT, nblocks, d_F, s));
  ctx->launches += 2;
  return ALEGB_OK;
}

int alegb_set_coordinate_mode(alegb_ctx* ctx, int mode, double t_start) {
  if (!ctx) return ALEGB_INVALID_ARG;
  if (mode != ALEGB_COORDS_CLOSED_FORM && mode != ALEGB_COORDS_RK) return fail(ctx, ALEGB_INVALID_ARG, "unknown coordinate mode");
  if (mode == ALEGB_COORDS_RK) {
    if (ctx->device < 0) return fail(ctx, ALEGB_CUDA_ERROR, "host-only context (no CUDA device)");
    if (!ctx->mesh_ready) return fail(ctx, ALEGB_NOT_READY, "alegb_mesh_upload has not been called");
    CU(cudaSetDevice(ctx->device));
    const int dim = ctx->ref.dim;
    if (!ctx->d_xn) CU(dev_alloc(ctx, &ctx->d_xn, (size_t)ctx->Nverts * dim));
    // x_n = the law's own position at t_start (USER: the positions last supplied)
    if (ctx->motion.kind != ALEGB_MOTION_USER)
      CU(launch_vertex_motion(dim, ctx->Nverts, ctx->d_X0, ctx->motion, t_start, nullptr, ctx->d_xv, ctx->d_vv, 0));
    CU(cudaMemcpyAsync(ctx->d_xn, ctx->d_xv, (size_t)ctx->Nverts * dim * sizeof(double), cudaMemcpyDeviceToDevice, 0));
    CU(cudaStreamSynchronize(0));
  }
  ctx->coord_mode = mode;
  ctx->config_version++;
  return ALEGB_OK;
}

int alegb_get_positions(alegb_ctx* ctx, double* d_x, void* stream) {
  if (!ctx) return ALEGB_INVALID_ARG;
  if (ctx->device < 0) return fail(ctx, ALEGB_CUDA_ERROR, "host-only context (no CUDA device)");
  if (!ctx->mesh_ready) return fail(ctx, ALEGB_NOT_READY, "alegb_mesh_upload has not been called");
  if (!d_x) return fail(ctx, ALEGB_INVALID_ARG, "NULL device array");
  CU(cudaSetDevice(ctx->device));
  const double* src = ctx->coord_mode == ALEGB_COORDS_RK ? ctx->d_xn : ctx->d_xv;
  CU(cudaMemcpyAsync(d_x, src, (size_t)ctx->Nverts * ctx->ref.dim * sizeof(double), cudaMemcpyDeviceToDevice,
                     static_cast<cudaStream_t>(stream)));
  return ALEGB_OK;
}

int alegb_rhs_pml(alegb_ctx* ctx, double t, const double* d_q, const double* d_aux, double* d_F, double* d_Faux,
                  void* stream) {
  int rc = check_ready(ctx);
  if (rc != ALEGB_OK) return rc;
  if (!d_q || !d_F) return fail(ctx, ALEGB_INVALID_ARG, "NULL field pointer");
  if (!aligned16(d_q) || !aligned16(d_F)) return fail(ctx, ALEGB_INVALID_ARG, "field pointers must be 16-byte aligned");
  cudaStream_t s = (cudaStream_t)stream;
  rc = update_geometry(ctx, t, s);
  if (rc != ALEGB_OK) return rc;
  StageArgs a;
  fill_common(ctx, a);
  a.q_in = d_q; a.F_out = d_F;
  a.aux = ctx->Kpml > 0 ? (d_aux ? d_aux : ctx->d_AUX) : nullptr;
  PmlArgs p;
  if (d_Faux && ctx->Kpml > 0) {
    fill_common(ctx, p);
    p.q_in = d_q; p.aux_in = a.aux; p.G_out = d_Faux;
    if (ctx->layer_fused()) layer_from(p, a.layer);
  }
  rc = timed_stage(ctx, a, s);
  if (rc != ALEGB_OK) return rc;
  if (d_Faux && ctx->Kpml > 0 && !a.layer.on) {
    CU(launch_pml_any(ctx, p, s));
    ctx->launches++;
  }
  return ALEGB_OK;
}

int alegb_rhs(alegb_ctx* ctx, double t, const double* d_q, double* d_F, void* stream) {
  return alegb_rhs_pml(ctx, t, d_q, nullptr, d_F, nullptr, stream);
}

int alegb_step(alegb_ctx* ctx, double* d_q, double t0, double dt, int nsteps, void* stream) {
  int rc = check_ready(ctx);
  if (rc != ALEGB_OK) return rc;
  if (!d_q || nsteps < 0) return fail(ctx, ALEGB_INVALID_ARG, "NULL field pointer or negative step count");
  if (!aligned16(d_q)) return fail(ctx, ALEGB_INVALID_ARG, "field pointers must be 16-byte aligned");
  cudaStream_t s = (cudaStream_t)stream;
  double* outs[4] = {ctx->d_Q1, ctx->d_Q2, ctx->d_Q1, d_q};
  if (ctx->use_graph && !ctx->profiling && nsteps >= 2) {
    rc = step_graph_launch(ctx, d_q, outs, t0, dt, nsteps, s);
    if (rc != ALEGB_UNSUPPORTED) return rc;   // UNSUPPORTED: capture not possible here, launch directly instead
  }
  for (int n = 0; n < nsteps; ++n) {
    rc = sark_step(ctx, d_q, outs, t0 + n * dt, dt, s);
    if (rc != ALEGB_OK) return rc;
  }
  return ALEGB_OK;
}

int alegb_step_debug(alegb_ctx* ctx, const double* d_q, double t0, double dt, double* d_stages, void* stream) {
  int rc = check_ready(ctx);
  if (rc != ALEGB_OK) return rc;
  if (!d_q || !d_stages) return fail(ctx, ALEGB_INVALID_ARG, "NULL field pointer");
  if (!aligned16(d_q) || !aligned16(d_stages)) return fail(ctx, ALEGB_INVALID_ARG, "field pointers must be 16-byte aligned");
  const size_t state = (size_t)ctx->K * ctx->Nf * ctx->ref.Np;
  double* outs[4] = {d_stages, d_stages + state, d_stages + 2 * state, d_stages + 3 * state};
  return sark_step(ctx, d_q, outs, t0, dt, (cudaStream_t)stream, nullptr, /*advance_coords=*/false);
}

int alegb_step_host(alegb_ctx* ctx, double* h_q, double t0, double dt, int nsteps) {
  int rc = check_ready(ctx);
  if (rc != ALEGB_OK) return rc;
  if (!h_q) return fail(ctx, ALEGB_INVALID_ARG, "NULL host pointer");
  const size_t state = (size_t)ctx->K * ctx->Nf * ctx->ref.Np;
  if (!ctx->d_Qhost) CU(dev_alloc(ctx, &ctx->d_Qhost, state));
  CU(cudaMemcpyAsync(ctx->d_Qhost, h_q, state * sizeof(double), cudaMemcpyHostToDevice, 0));
  rc = alegb_step(ctx, ctx->d_Qhost, t0, dt, nsteps, nullptr);
  if (rc != ALEGB_OK) return rc;
  CU(cudaMemcpyAsync(h_q, ctx->d_Qhost, state * sizeof(double), cudaMemcpyDeviceToHost, 0));
  CU(cudaStreamSynchronize(0));
  return ALEGB_OK;
}

int alegb_geometry(alegb_ctx* ctx, double t, double* d_vgeo, double* d_sgeo, double* d_xv, double* d_vv, void* stream) {
  if (!ctx) return ALEGB_INVALID_ARG;
  if (ctx->device < 0) return fail(ctx, ALEGB_CUDA_ERROR, "host-only context (no CUDA device)");
  if (!ctx->mesh_ready) return fail(ctx, ALEGB_NOT_READY, "alegb_mesh_upload has not been called");
  CU(cudaSetDevice(ctx->device));
  cudaStream_t s = (cudaStream_t)stream;
  int rc = update_geometry(ctx, t, s);
  if (rc != ALEGB_OK) return rc;
  const int dim = ctx->ref.dim;
  const size_t K = (size_t)ctx->K, nvb = (size_t)ctx->Nverts * dim * sizeof(double);
  if (d_vgeo) CU(cudaMemcpyAsync(d_vgeo, ctx->d_vgeo, K * (dim * dim + 1) * sizeof(double), cudaMemcpyDeviceToDevice, s));
  if (d_sgeo) CU(cudaMemcpyAsync(d_sgeo, ctx->d_sgeo, K * (dim + 1) * (dim + 2) * sizeof(double), cudaMemcpyDeviceToDevice, s));
  if (d_xv) CU(cudaMemcpyAsync(d_xv, ctx->d_xv, nvb, cudaMemcpyDeviceToDevice, s));
  if (d_vv) CU(cudaMemcpyAsync(d_vv, ctx->d_vv, nvb, cudaMemcpyDeviceToDevice, s));
  return ALEGB_OK;
}

int64_t alegb_pml_count(const alegb_ctx* ctx) { return ctx ? ctx->Kpml : 0; }

int alegb_pml_elements(const alegb_ctx* ctx, int32_t* elems) {
  if (!ctx || !elems) return ALEGB_INVALID_ARG;
  for (size_t i = 0; i < ctx->pml_elems_host.size(); ++i) elems[i] = ctx->pml_elems_host[i];
  return ALEGB_OK;
}

int alegb_pml_reset(alegb_ctx* ctx, void* stream) {
  if (!ctx) return ALEGB_INVALID_ARG;
  if (ctx->Kpml == 0) return ALEGB_OK;
  if (ctx->device < 0) return fail(ctx, ALEGB_CUDA_ERROR, "host-only context (no CUDA device)");
  CU(cudaSetDevice(ctx->device));
  const size_t na = (size_t)ctx->Kpml * ctx->ref.dim * ctx->Nf * ctx->ref.Np;
  CU(cudaMemsetAsync(ctx->d_AUX, 0, na * sizeof(double), (cudaStream_t)stream));
  return ALEGB_OK;
}

int alegb_pml_get(alegb_ctx* ctx, double* d_aux, void* stream) {
  if (!ctx || !d_aux) return ALEGB_INVALID_ARG;
  if (ctx->Kpml == 0) return ALEGB_OK;
  if (ctx->device < 0) return fail(ctx, ALEGB_CUDA_ERROR, "host-only context (no CUDA device)");
  CU(cudaSetDevice(ctx->device));
  const size_t na = (size_t)ctx->Kpml * ctx->ref.dim * ctx->Nf * ctx->ref.Np;
  CU(cudaMemcpyAsync(d_aux, ctx->d_AUX, na * sizeof(double), cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
  return ALEGB_OK;
}

int alegb_pml_set(alegb_ctx* ctx, const double* d_aux, void* stream) {
  if (!ctx || !d_aux) return ALEGB_INVALID_ARG;
  if (ctx->Kpml == 0) return ALEGB_OK;
  if (ctx->device < 0) return fail(ctx, ALEGB_CUDA_ERROR, "host-only context (no CUDA device)");
  CU(cudaSetDevice(ctx->device));
  const size_t na = (size_t)ctx->Kpml * ctx->ref.dim * ctx->Nf * ctx->ref.Np;
  CU(cudaMemcpyAsync(ctx->d_AUX, d_aux, na * sizeof(double), cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
  return ALEGB_OK;
}

int alegb_get_sizes(const alegb_ctx* ctx, int* dim, int* N, int* Np, int* Nfp, int* Nfaces, int* Nfields, int64_t* K,
                    int64_t* Nverts) {
  if (!ctx) return ALEGB_INVALID_ARG;
  if (dim) *dim = ctx->ref.dim;
  if (N) *N = ctx->ref.N;
  if (Np) *Np = ctx->ref.Np;
  if (Nfp) *Nfp = ctx->ref.Nfp;
  if (Nfaces) *Nfaces = ctx->ref.Nfaces;
  if (Nfields) *Nfields = ctx->Nf;
  if (K) *K = ctx->K;
  if (Nverts) *Nverts = ctx->Nverts;
  return ALEGB_OK;
}

int alegb_get_operators(alegb_ctx* ctx, double* r, double* s, double* t3, double* Dr, double* Ds, double* Dt,
                        double* LIFT, int32_t* vmapM, int32_t* vmapP) {
  if (!ctx) return ALEGB_INVALID_ARG;
  const RefElement& R = ctx->ref;
  const int Np = R.Np;
  auto cp = [](double* dst, const double* src, size_t n) { if (dst) std::memcpy(dst, src, n * sizeof(double)); };
  cp(r, R.rst.data(), Np);
  cp(s, R.rst.data() + Np, Np);
  if (R.dim == 3) cp(t3, R.rst.data() + 2 * Np, Np);
  cp(Dr, R.D[0].data(), (size_t)Np * Np);
  cp(Ds, R.D[1].data(), (size_t)Np * Np);
  if (R.dim == 3) cp(Dt, R.D[2].data(), (size_t)Np * Np);
  cp(LIFT, R.LIFT.data(), R.LIFT.size());
  if (vmapM || vmapP) {
    if (!ctx->mesh_ready) return fail(ctx, ALEGB_NOT_READY, "alegb_mesh_upload has not been called");
    if (vmapM) std::memcpy(vmapM, ctx->vmapM_host.data(), ctx->vmapM_host.size() * sizeof(int32_t));
    if (vmapP) std::memcpy(vmapP, ctx->vmapP_host.data(), ctx->vmapP_host.size() * sizeof(int32_t));
  }
  return ALEGB_OK;
}

int alegb_get_reference(const alegb_ctx* ctx, double* w, double* lam, int32_t* fmask) {
  if (!ctx) return ALEGB_INVALID_ARG;
  const RefElement& R = ctx->ref;
  if (w) std::memcpy(w, R.w.data(), R.w.size() * sizeof(double));
  if (lam) std::memcpy(lam, R.lam.data(), R.lam.size() * sizeof(double));
  if (fmask) for (size_t i = 0; i < R.fmask.size(); ++i) fmask[i] = R.fmask[i];
  return ALEGB_OK;
}

int alegb_sark_coefficients(double gamma, double* a, double* b) {
  if (!a || !b) return ALEGB_INVALID_ARG;
  sark_coefficients(gamma, a, b);
  return ALEGB_OK;
}

int alegb_set_kernel(alegb_ctx* ctx, int kind) {
  if (!ctx) return ALEGB_INVALID_ARG;
  if (kind < 0 || kind > 2) return fail(ctx, ALEGB_INVALID_ARG, "kernel kind must be 0 (auto), 1 (generic) or 2 (pipelined DMMA)");
  if (kind == 2 && !ctx->pipe_ok) return fail(ctx, ALEGB_UNSUPPORTED, "no pipelined DMMA stage kernel for this (dim, N)");
  ctx->kernel_mode = kind;
  ctx->config_version++;
  return ALEGB_OK;
}

int alegb_set_max_ctas(alegb_ctx* ctx, int max_ctas) {
  if (!ctx) return ALEGB_INVALID_ARG;
  if (max_ctas < 0) return fail(ctx, ALEGB_INVALID_ARG, "max_ctas must be >= 0 (0 = one CTA per SM)");
  ctx->max_ctas = max_ctas;
  ctx->config_version++;
  return ALEGB_OK;
}

int alegb_pipe_config(int dim, int N, int* cfg) {
  if (!cfg) return ALEGB_INVALID_ARG;
  PipeConfig c{};
  if (!stage_pipe_config(dim, N, c)) return ALEGB_UNSUPPORTED;
  cfg[0] = c.producer_groups; cfg[1] = c.slots; cfg[2] = c.items_per_quad; cfg[3] = c.consumer_warps;
  cfg[4] = c.warps_per_group; cfg[5] = c.producer_warps; cfg[6] = c.elements_per_quad; cfg[7] = c.smem_bytes;
  return ALEGB_OK;
}

int alegb_pipe_config_layer(int dim, int N, int* cfg) {
  if (!cfg) return ALEGB_INVALID_ARG;
  PipeConfig c{};
  if (!stage_pipe_config(dim, N, c, true)) return ALEGB_UNSUPPORTED;
  cfg[0] = c.producer_groups; cfg[1] = c.slots; cfg[2] = c.items_per_quad; cfg[3] = c.consumer_warps;
  cfg[4] = c.warps_per_group; cfg[5] = c.producer_warps; cfg[6] = c.elements_per_quad; cfg[7] = c.smem_bytes;
  return ALEGB_OK;
}

int alegb_set_layer_fusion(alegb_ctx* ctx, int on) {
  if (!ctx) return ALEGB_INVALID_ARG;
  ctx->fuse_layer = on != 0;
  ctx->config_version++;
  return ALEGB_OK;
}

int alegb_set_geometry_overlap(alegb_ctx* ctx, int on) {
  if (!ctx) return ALEGB_INVALID_ARG;
  ctx->overlap_geometry = on != 0;
  ctx->config_version++;
  return ALEGB_OK;
}

int alegb_set_graph(alegb_ctx* ctx, int on) {
  if (!ctx) return ALEGB_INVALID_ARG;
  ctx->use_graph = on != 0;
  return ALEGB_OK;
}

int alegb_profile_enable(alegb_ctx* ctx, int on) {
  if (!ctx) return ALEGB_INVALID_ARG;
  ctx->profiling = on != 0;
  ctx->prof_used = 0;
  return ALEGB_OK;
}

int alegb_profile_read(alegb_ctx* ctx, int64_t* launches, double* total_ms) {
  if (!ctx || !launches || !total_ms) return ALEGB_INVALID_ARG;
  if (ctx->device < 0) return fail(ctx, ALEGB_CUDA_ERROR, "host-only context (no CUDA device)");
  CU(cudaSetDevice(ctx->device));
  CU(cudaDeviceSynchronize());
  double sum = 0.0;
  for (size_t i = 0; i + 1 < ctx->prof_used; i += 2) {
    float ms = 0.f;
    CU(cudaEventElapsedTime(&ms, ctx->prof_events[i], ctx->prof_events[i + 1]));
    sum += ms;
  }
  *launches = (int64_t)(ctx->prof_used / 2);
  *total_ms = sum;
  return ALEGB_OK;
}

int alegb_measure_fp64_peak(alegb_ctx* ctx, double* dmma_tflops, double* dfma_tflops) {
  if (!ctx || !dmma_tflops || !dfma_tflops) return ALEGB_INVALID_ARG;
  if (ctx->device < 0) return fail(ctx, ALEGB_CUDA_ERROR, "host-only context (no CUDA device)");
  CU(cudaSetDevice(ctx->device));
  CU(cudaDeviceSynchronize());
  CU(measure_fp64_peak(ctx->num_sms, 5, dmma_tflops, dfma_tflops, 0));
  ctx->launches += 12;
  return ALEGB_OK;
}

int64_t alegb_workspace_bytes(const alegb_ctx* ctx) { return ctx ? ctx->workspace_bytes : 0; }
const char* alegb_last_error(const alegb_ctx* ctx) { return ctx ? ctx->err.c_str() : "null context"; }
int64_t alegb_launch_count(const alegb_ctx* ctx) { return ctx ? ctx->launches : 0; }

}  // extern "C"
