// Internal declarations shared by the library's translation units (not part of the ABI).
#pragma once
#include <cuda_runtime.h>

#include <cstdint>
#include <string>
#include <vector>

#include "host_ref.h"

namespace alegb {

constexpr int kMaxFields = 10;

// Per-field coefficients of one fused stage (PAPER.md:L132-134 written as two linear combinations):
//   q_out   = cq_n  q_n + cq_f0 F0 + cq_acc acc_in + cq_f F
//   acc_out = ca_n  q_n + ca_f0 F0 + ca_acc acc_in + ca_f F
// The per-field values depend on the field k only through k <= dim (lambda = 0) or k > dim (lambda = 1/tau, L115):
// stage_pipe.cu reads entries [0] and [dim + 1] only.
// F is the operator of eq. 9 evaluated on q_in at the stage time.  A NULL output pointer skips that output; inputs
// whose coefficients are all zero are not read.
struct StageCoef {
  double cq_n[kMaxFields], cq_f0[kMaxFields], cq_f[kMaxFields];
  double ca_n[kMaxFields], ca_f0[kMaxFields], ca_f[kMaxFields];
  double cq_acc, ca_acc;
};

// a8 fused into the pipelined stage kernel (stage_pipe.cu, LAYER instantiation): the auxiliary fields of the absorbing
// layer [Kpml][dim][Nf][Np] (reading R12).  G = right-hand side of the auxiliary equation evaluated on StageArgs::aux;
//   aux_out = cx_n aux_n + cx_acc acc_in + cx_g G ;  acc_out = cy_n aux_n + cy_acc acc_in + cy_g G
struct LayerArgs {
  bool on;                 // run the fused path (false: the stage kernel only subtracts sigma_d q~^d from F)
  const double* aux_n; const double* acc_in;
  double* G_out; double* aux_out; double* acc_out;
  double cx_n, cx_acc, cx_g, cy_n, cy_acc, cy_g;
};

struct StageArgs {
  // mesh / geometry at the stage time
  int64_t K;
  const double* vgeo;    // [K][dim*dim+1]
  const double* sgeo;    // [K][Nfaces][dim+2]
  const double* vvel;    // [K][dim+1][dim] vertex velocities of each element
  const int32_t* vmapP;  // [K][Nfaces*Nfp]
  const int8_t* EToB;    // [K][Nfaces] or NULL
  const int32_t* pml_index;  // [K] index into the auxiliary arrays, -1 outside the layer; or NULL
  const double* pml_sigma;   // [Kpml][dim]
  const double* aux;         // [Kpml][dim][Nf][Np] auxiliary state entering F, or NULL
  // operators (device, transposed for coalesced staging)
  const double* Dt_ops;  // [dim][Np(j)][Np(i)] : D_a[i][j]
  const double* LIFTt;   // [Nfaces*Nfp(m)][Np(i)] : LIFT[i][m]
  const double* lam;     // [Np][dim+1]
  const int32_t* fmask;  // [Nfaces*Nfp]
  const double* Avol;    // DMMA path: D_a in fragment order [dim][NB][KS][32]
  const double* AliftP;  // DMMA path: LIFT in fragment order, faces packed along k: [NB][ceil(Nfaces*Nfp/4)][32]
  // physics
  double c, invtau;
  const double* relax_cub;   // R = P N~(I q) [K][Ns][Np] replacing the collocated N~(q), or NULL (reading R8)
  double q_inf[kMaxFields];
  // fields
  const double* q_in;
  const double* q_n;
  const double* F0_in;
  const double* acc_in;
  double* F_out;    // plain F (stage 0 writes F0 here; rhs mode writes the result here)
  double* q_out;
  double* acc_out;
  StageCoef coef;
  LayerArgs layer;
  const int32_t* quad_list;   // pipelined kernel: the quads (groups of 4 consecutive elements) of this launch, or NULL = all
  int64_t nquads_list;
};

// cubature-projected relaxation (cubature.cu): R[K][Ns][Np] = P N~(I q), Ns = dim (dim+1)/2 stiff fields
struct CubArgs {
  int64_t K;
  int Np, Nc, EB;        // nodes, cubature nodes, elements per CTA pass
  const double* It;      // [Np][Nc]  I transposed
  const double* Pt;      // [Nc][Np]  P transposed
  const double* AI;      // DMMA path: I in A-fragment order [NRT][KS][32]
  const double* AP;      // DMMA path: P in A-fragment order [NB][2 NRT][32]
  const double* q;       // [K][Nf][Np]
  double* R;
  double invtau;
};

struct PmlArgs {
  int64_t Kpml;
  const int32_t* pml_elems;  // [Kpml]
  const double* pml_sigma;   // [Kpml][dim]
  const double* vgeo; const double* sgeo; const double* vvel;
  const int32_t* vmapP; const int8_t* EToB;
  const double* Dt_ops; const double* LIFTt; const double* lam; const int32_t* fmask;
  const double* Avol; const double* AliftP;   // DMMA path (pml_mma.cu): operator fragments as in StageArgs
  double c;
  double q_inf[kMaxFields];
  const double* q_in;
  // auxiliary fields [Kpml][dim][Nf][Np]:  G = rhs of the auxiliary equation (reading R12)
  //   aux_out = cx_n aux_n + cx_acc acc_in + cx_g G ;  acc_out = cy_n aux_n + cy_acc acc_in + cy_g G
  const double* aux_in;   // state G is evaluated on
  const double* aux_n; const double* acc_in;
  double* G_out; double* aux_out; double* acc_out;
  double cx_n, cx_acc, cx_g, cy_n, cy_acc, cy_g;
};

struct MotionArgs {
  int kind; int nparams;
  double p[16];
};

// kernel launchers (kernels.cu); return cudaGetLastError()
// t_dev != NULL: the stage time is read from the device (graph-captured steps) and t is ignored
cudaError_t launch_vertex_motion(int dim, int64_t Nverts, const double* X0, const MotionArgs& m, double t,
                                 const double* t_dev, double* xv, double* vv, cudaStream_t s);
// coordinates integrated by RK4 (NEXT-2): stage 0..3 writes xv, vv of that stage; stage 4 advances x_n to x_{n+1}
cudaError_t launch_vertex_rk(int dim, int64_t Nverts, const double* X0, const MotionArgs& m, const double* user_vv,
                             int stage, double t_n, double t_h, double t_e, double dt, const double* ts_dev, double* x_n,
                             double* xv, double* vv, cudaStream_t s);
// NEXT-3: wall-force integrals; partial[nblocks][2 dim] scratch, out[2 dim] = (F_p, F_v) on the device
cudaError_t launch_wall_force(int dim, int64_t K, const int8_t* EToB, int tag, const double* q, const double* sgeo,
                              const int32_t* fmask, const double* wface, int Np, int Nfp, double RT, double* partial,
                              int nblocks, double* out, cudaStream_t s);
// the same with the partial sums in the library's static device array (no allocation; alegb_wall_forces_static);
// the caller's device must be current; cudaErrorInvalidValue if nblocks is outside 1..ALEGB_WALL_FORCES_STATIC_MAX_BLOCKS
cudaError_t launch_wall_force_static(int dim, int64_t K, const int8_t* EToB, int tag, const double* q,
                                     const double* sgeo, const int32_t* fmask, const double* wface, int Np, int Nfp,
                                     double RT, int nblocks, double* out, cudaStream_t s);
// clock = {t0, dt, stage times[4]} on the device; _set starts a run of steps, the other advances to the next step
cudaError_t launch_step_clock(double* clock, long long* counter, cudaStream_t s);
cudaError_t launch_step_clock_set(double* clock, long long* counter, double t0, double dt, cudaStream_t s);
cudaError_t launch_geometry(int dim, int64_t K, const int32_t* EToV, const double* xv, const double* vv, double* vgeo,
                            double* sgeo, double* vvel, cudaStream_t s);
// returns cudaErrorInvalidValue if (dim, N) has no compiled kernel
cudaError_t launch_stage(int dim, int N, const StageArgs& a, int num_sms, cudaStream_t s);
cudaError_t launch_pml(int dim, int N, const PmlArgs& a, int num_sms, cudaStream_t s);
cudaError_t configure_kernels(int dim, int N);

// cubature-projected relaxation, cubature.cu
size_t cubature_smem_bytes(int dim, int Np, int Nc, int EB);
cudaError_t configure_cubature(int dim, size_t smem);
cudaError_t launch_cubature(int dim, const CubArgs& a, int num_sms, cudaStream_t s);
void cubature_mma_layout(int dim, int N, int& NRT, int& KS, int& NB);   // fragment-array extents
bool cubature_mma_available(int dim, int N);
cudaError_t launch_cubature_mma(int dim, int N, const CubArgs& a, int num_sms, cudaStream_t s);   // InvalidValue: none for (dim, N)

// tensor-core kernel of the absorbing layer's auxiliary fields, pml_mma.cu
cudaError_t configure_pml_mma(int dim, int N);        // cudaErrorInvalidValue if (dim, N) has no such kernel
cudaError_t launch_pml_mma(int dim, int N, const PmlArgs& a, int num_sms, cudaStream_t s);

// pipelined tensor-core stage kernel (producer / consumer warps), stage_pipe.cu; same operator fragments
cudaError_t configure_stage_pipe(int dim, int N);     // cudaErrorInvalidValue if (dim, N) has no such kernel
cudaError_t launch_stage_pipe(int dim, int N, const StageArgs& a, int num_sms, cudaStream_t s);
struct PipeConfig { int producer_groups, slots, items_per_quad, consumer_warps, warps_per_group, producer_warps, elements_per_quad, smem_bytes; };
bool stage_pipe_config(int dim, int N, PipeConfig& c, bool layer = false);   // false if (dim, N) has no such kernel; layer: the LAYER instantiation
bool stage_pipe_layer_supported(int dim, int N);          // the instantiation with the absorbing layer fused in exists

// fp64 ceiling of the current device measured with register-resident DMMA / DFMA chains (fp64_peak.cu)
cudaError_t measure_fp64_peak(int num_sms, int reps, double* dmma_tflops, double* dfma_tflops, cudaStream_t s);

}  // namespace alegb
