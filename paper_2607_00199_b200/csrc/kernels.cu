// CUDA kernels of the ALE Galerkin-Boltzmann stage (sm_100a), generic element-blocked path for every (dim, N).
//
//   a1  vertex_motion_kernel   positions / velocities of the vertices from the prescribed law
//   a2  geometry_kernel        geometric factors of the moved affine simplices (L88-92, L193)
//   a3-a6 stage_kernel         volume + collocated relaxation + surface + SARK stage update, fused (L107, L132-134)
//   a8  pml_kernel             auxiliary fields of the absorbing layer (reading R12)
//
// The tensor-core (DMMA) stage kernel lives in stage_pipe.cu.
#include <cstdio>
#include <mutex>

#include "../../include/alegb.h"
#include "alegb_internal.h"
#include "device_common.cuh"

namespace alegb {

// ------------------------------------------------------------------------------------------------------------------
// The prescribed motion laws at one vertex: displacement and velocity at time t from the t = 0 coordinate X
// (include/alegb.h lists the parameters).
template <int DIM>
__device__ __forceinline__ void motion_law(const MotionArgs& m, const double* X, double t, double* disp, double* vel) {
#pragma unroll
  for (int d = 0; d < DIM; ++d) { disp[d] = 0.0; vel[d] = 0.0; }
  const double* p = m.p;
  if (m.kind == 1) {  // SINES_PRODUCT: eq. 15
    double A = p[0], om = 2.0 * M_PI / p[1], shape = 1.0;
#pragma unroll
    for (int d = 0; d < DIM; ++d) shape *= sin(p[2 + d] * X[d] + p[2 + DIM + d]);
    double s = A * sin(om * t) * shape, ds = A * om * cos(om * t) * shape;
#pragma unroll
    for (int d = 0; d < DIM; ++d) { disp[d] = s; vel[d] = ds; }
  } else if (m.kind == 2) {  // SINES_CROSS: eq. 19
    double A = p[0], om = 2.0 * M_PI / p[1], k = p[2], ph = p[3];
    double sn[DIM];
#pragma unroll
    for (int d = 0; d < DIM; ++d) sn[d] = sin(k * X[d] + ph);
#pragma unroll
    for (int d = 0; d < DIM; ++d) {
      double shape = 1.0;
#pragma unroll
      for (int o = 0; o < DIM; ++o) if (o != d) shape *= sn[o];
      disp[d] = A * sin(om * t) * shape;
      vel[d] = A * om * cos(om * t) * shape;
    }
  } else if (m.kind == 3) {  // PLUNGE_BLEND: eqs. 20-21 times a radial quintic blend
    double h0 = p[0], om = p[1], r1 = p[2], r2 = p[3];
    int axis = (int)p[4];
    double rho2 = 0.0;
#pragma unroll
    for (int d = 0; d < DIM; ++d) rho2 += (X[d] - p[5 + d]) * (X[d] - p[5 + d]);
    double u = (sqrt(rho2) - r1) / (r2 - r1);
    u = fmin(fmax(u, 0.0), 1.0);
    double b = 1.0 - (6.0 * u * u * u * u * u - 15.0 * u * u * u * u + 10.0 * u * u * u);
#pragma unroll
    for (int d = 0; d < DIM; ++d)
      if (d == axis) { disp[d] = h0 * sin(om * t) * b; vel[d] = h0 * om * cos(om * t) * b; }
  } else if (m.kind == 4) {  // CARANGIFORM: L339-365
    double a0 = p[0], a1 = p[1], a2 = p[2], k = p[3], om = p[4], Rr = p[5], beta = p[6], Tr = p[7];
    int axis = (int)p[8];
    double Bcut = p[9];
    double xt = fmin(1.0, fmax(0.0, X[0]));
    double r2 = (X[0] - xt) * (X[0] - xt);
#pragma unroll
    for (int d = 1; d < DIM; ++d) r2 += X[d] * X[d];
    double deff = fmax(sqrt(r2) - Rr, 0.0);
    double B = exp(-beta * deff * deff);
    if (B < Bcut) B = 0.0;
    double Amp = a0 + a1 * xt + a2 * xt * xt;
    double phi = k * X[0] - om * t;
    double S = 1.0, Sd = 0.0;
    if (t < Tr) { S = 0.5 * (1.0 - cos(M_PI * t / Tr)); Sd = M_PI / (2.0 * Tr) * sin(M_PI * t / Tr); }
#pragma unroll
    for (int d = 0; d < DIM; ++d)
      if (d == axis) {
        disp[d] = Amp * sin(phi) * B * S;
        vel[d] = -Amp * om * cos(phi) * B * S + Amp * sin(phi) * B * Sd;
      }
  }
}

// a1: vertex motion.  One thread per vertex.
template <int DIM>
__global__ void vertex_motion_kernel(int64_t Nverts, const double* __restrict__ X0, MotionArgs m, double t,
                                     const double* __restrict__ t_dev, double* __restrict__ xv,
                                     double* __restrict__ vv) {
  int64_t v = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (v >= Nverts) return;
  if (t_dev != nullptr) t = *t_dev;   // stage time kept on the device (graph-captured steps)
  double X[DIM], disp[DIM], vel[DIM];
#pragma unroll
  for (int d = 0; d < DIM; ++d) X[d] = X0[v * DIM + d];
  motion_law<DIM>(m, X, t, disp, vel);
#pragma unroll
  for (int d = 0; d < DIM; ++d) { xv[v * DIM + d] = X[d] + disp[d]; vv[v * DIM + d] = vel[d]; }
}

// a1, coordinates integrated in time ("the nodal coordinates are advanced in time using the same
// Runge-Kutta integration scheme", L233 dx/dt = v_G).  Classic RK4 on dx/dt = v(X0, t):
//   stage 0: x_n, v(t_n)   1: x_n + dt/2 v(t_n), v(t_h)   2: x_n + dt/2 v(t_h), v(t_h)   3: x_n + dt v(t_h), v(t_n+dt)
//   stage 4 (end of the step): x_n <- x_n + dt/6 (v(t_n) + 2 v(t_h) + 2 v(t_h) + v(t_n+dt))
// The velocities are re-evaluated from the law (a few sincos per vertex) instead of being kept between launches;
// user_vv != NULL: a velocity that is constant in time (motion kind USER).
// ts = {t_n, t_h, t_h, t_n + dt}; ts_dev (graph-captured steps) points at the same four times on the device, with dt
// one double before them (the step clock).
template <int DIM>
__global__ void vertex_rk_kernel(int64_t Nverts, const double* __restrict__ X0, MotionArgs m,
                                 const double* __restrict__ user_vv, int stage, double t_n, double t_h, double t_e,
                                 double dt, const double* __restrict__ ts_dev, double* __restrict__ x_n,
                                 double* __restrict__ xv, double* __restrict__ vv) {
  int64_t v = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (v >= Nverts) return;
  if (ts_dev != nullptr) { t_n = ts_dev[0]; t_h = ts_dev[1]; t_e = ts_dev[3]; dt = ts_dev[-1]; }
  double X[DIM], xn[DIM], disp[DIM], k1[DIM], k2[DIM], k3[DIM], k4[DIM];
#pragma unroll
  for (int d = 0; d < DIM; ++d) { X[d] = X0[v * DIM + d]; xn[d] = x_n[v * DIM + d]; }
  if (user_vv != nullptr) {   // kind USER: the caller's vertex velocities of the four stages, [4][Nverts][DIM]
    const int64_t n = Nverts * DIM;
#pragma unroll
    for (int d = 0; d < DIM; ++d) {
      k1[d] = user_vv[v * DIM + d];
      k2[d] = user_vv[n + v * DIM + d];
      k3[d] = user_vv[2 * n + v * DIM + d];
      k4[d] = user_vv[3 * n + v * DIM + d];
    }
  } else {                    // a law v(X0, t): the two middle stages see the same velocity
    motion_law<DIM>(m, X, t_n, disp, k1);
    motion_law<DIM>(m, X, t_h, disp, k2);
    motion_law<DIM>(m, X, t_e, disp, k4);
#pragma unroll
    for (int d = 0; d < DIM; ++d) k3[d] = k2[d];
  }
#pragma unroll
  for (int d = 0; d < DIM; ++d) {
    double x, w;
    if (stage == 0) { x = xn[d]; w = k1[d]; }
    else if (stage == 1) { x = fma(0.5 * dt, k1[d], xn[d]); w = k2[d]; }
    else if (stage == 2) { x = fma(0.5 * dt, k2[d], xn[d]); w = k3[d]; }
    else if (stage == 3) { x = fma(dt, k3[d], xn[d]); w = k4[d]; }
    else {
      x_n[v * DIM + d] = xn[d] + dt * ((1.0 / 6.0) * k1[d] + (1.0 / 3.0) * k2[d] + (1.0 / 3.0) * k3[d] + (1.0 / 6.0) * k4[d]);
      continue;
    }
    xv[v * DIM + d] = x;
    vv[v * DIM + d] = w;
  }
}

cudaError_t launch_vertex_rk(int dim, int64_t Nverts, const double* X0, const MotionArgs& m, const double* user_vv,
                             int stage, double t_n, double t_h, double t_e, double dt, const double* ts_dev, double* x_n,
                             double* xv, double* vv, cudaStream_t s) {
  if (Nverts == 0) return cudaSuccess;
  int nb = (int)((Nverts + 255) / 256);
  if (dim == 2) vertex_rk_kernel<2><<<nb, 256, 0, s>>>(Nverts, X0, m, user_vv, stage, t_n, t_h, t_e, dt, ts_dev, x_n, xv, vv);
  else vertex_rk_kernel<3><<<nb, 256, 0, s>>>(Nverts, X0, m, user_vv, stage, t_n, t_h, t_e, dt, ts_dev, x_n, xv, vv);
  return cudaGetLastError();
}

cudaError_t launch_vertex_motion(int dim, int64_t Nverts, const double* X0, const MotionArgs& m, double t,
                                 const double* t_dev, double* xv, double* vv, cudaStream_t s) {
  if (Nverts == 0) return cudaSuccess;
  int nb = (int)((Nverts + 255) / 256);
  if (dim == 2) vertex_motion_kernel<2><<<nb, 256, 0, s>>>(Nverts, X0, m, t, t_dev, xv, vv);
  else vertex_motion_kernel<3><<<nb, 256, 0, s>>>(Nverts, X0, m, t, t_dev, xv, vv);
  return cudaGetLastError();
}

// Stage times of the next step on the device, for graph-captured steps.  clock = {t0, dt, times[4]}:
// n = *counter, t_n = t0 + n dt, times[i] = t_n + c_i dt (c = 0, 1/2, 1/2, 1; L126), then *counter = n + 1.  Plain IEEE
// multiply and add in the same order as the host loop of alegb_step, so both paths see bit-identical stage times.
__global__ void step_clock_kernel(double* clock, long long* counter) {
  const long long n = *counter;
  const double t0 = clock[0], dt = clock[1];
  const double tn = __dadd_rn(t0, __dmul_rn((double)n, dt));
  const double cst[4] = {0.0, 0.5, 0.5, 1.0};
  for (int i = 0; i < 4; ++i) clock[2 + i] = __dadd_rn(tn, __dmul_rn(cst[i], dt));
  *counter = n + 1;
}
__global__ void step_clock_set_kernel(double* clock, long long* counter, double t0, double dt) {
  clock[0] = t0;
  clock[1] = dt;
  *counter = 0;
}
cudaError_t launch_step_clock(double* clock, long long* counter, cudaStream_t s) {
  step_clock_kernel<<<1, 1, 0, s>>>(clock, counter);
  return cudaGetLastError();
}
cudaError_t launch_step_clock_set(double* clock, long long* counter, double t0, double dt, cudaStream_t s) {
  step_clock_set_kernel<<<1, 1, 0, s>>>(clock, counter, t0, dt);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------------
// NEXT-3: pressure and viscous force on the faces tagged `tag` (p = rho RT L53, sigma L51):
//   F_p = - int p n_b dS,  F_v = int sigma . n_b dS,  n_b = -n^ (outward normal of the body),
// face integral by the nodal face quadrature sJ sum_m (1^T M^f)_m g_m (reading R22).  One thread per element face,
// fixed grid and an ordered second pass: the result is deterministic.
template <int DIM>
__global__ void wall_force_kernel(int64_t K, const int8_t* __restrict__ EToB, int tag, const double* __restrict__ q,
                                  const double* __restrict__ sgeo, const int32_t* __restrict__ fmask,
                                  const double* __restrict__ wface, int Np, int Nfp, double RT,
                                  double* __restrict__ partial) {
  constexpr int Nf = DIM == 2 ? 6 : 10, Nfaces = DIM + 1, NO = 2 * DIM;
  double acc[NO];
#pragma unroll
  for (int x = 0; x < NO; ++x) acc[x] = 0.0;
  const int64_t total = K * Nfaces;
  for (int64_t ef = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; ef < total; ef += (int64_t)gridDim.x * blockDim.x) {
    if (EToB[ef] != tag) continue;
    const int64_t e = ef / Nfaces;
    const int f = (int)(ef - e * Nfaces);
    const double* sg = sgeo + ef * (DIM + 2);
    double nb[DIM];
#pragma unroll
    for (int d = 0; d < DIM; ++d) nb[d] = -sg[d];
    const double sJ = sg[DIM];
    const double* qe = q + e * Nf * Np;
    for (int m = 0; m < Nfp; ++m) {
      const int n = fmask[f * Nfp + m];
      const double w = sJ * wface[f * Nfp + m];
      double v[Nf];
#pragma unroll
      for (int k = 0; k < Nf; ++k) v[k] = qe[k * Np + n];
      const double p = RT * v[0], ir = 1.0 / v[0];
      double sig[DIM][DIM];
      if constexpr (DIM == 2) {
        sig[0][1] = sig[1][0] = -RT * (v[3] - v[1] * v[2] * ir);
        sig[0][0] = -RT * (ALEGB_SQRT2 * v[4] - v[1] * v[1] * ir);
        sig[1][1] = -RT * (ALEGB_SQRT2 * v[5] - v[2] * v[2] * ir);
      } else {
        sig[0][1] = sig[1][0] = -RT * (v[4] - v[1] * v[2] * ir);
        sig[0][2] = sig[2][0] = -RT * (v[5] - v[1] * v[3] * ir);
        sig[1][2] = sig[2][1] = -RT * (v[6] - v[2] * v[3] * ir);
        sig[0][0] = -RT * (ALEGB_SQRT2 * v[7] - v[1] * v[1] * ir);
        sig[1][1] = -RT * (ALEGB_SQRT2 * v[8] - v[2] * v[2] * ir);
        sig[2][2] = -RT * (ALEGB_SQRT2 * v[9] - v[3] * v[3] * ir);
      }
#pragma unroll
      for (int i = 0; i < DIM; ++i) {
        acc[i] -= w * p * nb[i];
        double s = 0.0;
#pragma unroll
        for (int j = 0; j < DIM; ++j) s = fma(sig[i][j], nb[j], s);
        acc[DIM + i] = fma(w, s, acc[DIM + i]);
      }
    }
  }
  __shared__ double red[256][NO];
#pragma unroll
  for (int x = 0; x < NO; ++x) red[threadIdx.x][x] = acc[x];
  __syncthreads();
  for (int s = blockDim.x / 2; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s) {
#pragma unroll
      for (int x = 0; x < NO; ++x) red[threadIdx.x][x] += red[threadIdx.x + s][x];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
#pragma unroll
    for (int x = 0; x < NO; ++x) partial[blockIdx.x * NO + x] = red[0][x];
  }
}

__global__ void wall_force_reduce_kernel(const double* __restrict__ partial, int nblocks, int NO, double* __restrict__ out) {
  const int x = threadIdx.x;
  if (x >= NO) return;
  double s = 0.0;
  for (int b = 0; b < nblocks; ++b) s += partial[b * NO + x];
  out[x] = s;
}

cudaError_t launch_wall_force(int dim, int64_t K, const int8_t* EToB, int tag, const double* q, const double* sgeo,
                              const int32_t* fmask, const double* wface, int Np, int Nfp, double RT, double* partial,
                              int nblocks, double* out, cudaStream_t s) {
  if (dim == 2) wall_force_kernel<2><<<nblocks, 256, 0, s>>>(K, EToB, tag, q, sgeo, fmask, wface, Np, Nfp, RT, partial);
  else wall_force_kernel<3><<<nblocks, 256, 0, s>>>(K, EToB, tag, q, sgeo, fmask, wface, Np, Nfp, RT, partial);
  wall_force_reduce_kernel<<<1, 32, 0, s>>>(partial, nblocks, 2 * dim, out);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------------
// The same two passes for callers that must not allocate (alegb_wall_forces_static, include/alegb.h).  The per-block
// partial sums of the first pass live in an array that is part of the library image instead of in a cudaMalloc'd
// buffer: kWallForceStaticBlocks x 6 doubles = 48 KiB, resident on every GPU that loads libalegb.so until the process
// exits, whether or not the entry point is ever called.
//
// g_wall_force_partial is a DEVICE symbol.  In host code its name is only a handle for the runtime's symbol calls;
// its value is not an address a kernel can use.  The address on the current device comes from cudaGetSymbolAddress,
// and it differs from device to device, so it is looked up once per device and kept in a small host table.
//
// Nothing in the array has to start at zero: the first pass overwrites partial[b][0..2 dim) for every block b it
// launches, including blocks that found no tagged face, and the second pass reads exactly those entries.  What a
// previous call left behind is never read.  All calls on one device share the array, so two calls whose kernels can
// run at the same time (different streams, no ordering between them) overwrite each other's partial sums.
constexpr int kWallForceStaticBlocks = ALEGB_WALL_FORCES_STATIC_MAX_BLOCKS;
constexpr int kWallForceStaticDevices = 64;
static __device__ __align__(256) double g_wall_force_partial[kWallForceStaticBlocks * 6];
static double* g_wall_force_partial_addr[kWallForceStaticDevices] = {};
static std::mutex g_wall_force_partial_mutex;

// Device address of g_wall_force_partial on the CURRENT device (the caller has made its device current).
static cudaError_t wall_force_static_scratch(double** addr) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kWallForceStaticDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_wall_force_partial_mutex);
  if (!g_wall_force_partial_addr[dev]) {
    double* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_wall_force_partial);   // loads the module on this device if need be
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_wall_force_partial_addr[dev] = p;
  }
  *addr = g_wall_force_partial_addr[dev];
  return cudaSuccess;
}

cudaError_t launch_wall_force_static(int dim, int64_t K, const int8_t* EToB, int tag, const double* q,
                                     const double* sgeo, const int32_t* fmask, const double* wface, int Np, int Nfp,
                                     double RT, int nblocks, double* out, cudaStream_t s) {
  if (nblocks < 1 || nblocks > kWallForceStaticBlocks) return cudaErrorInvalidValue;   // the ABI call checks first
  double* partial = nullptr;
  cudaError_t e = wall_force_static_scratch(&partial);
  if (e != cudaSuccess) return e;
  return launch_wall_force(dim, K, EToB, tag, q, sgeo, fmask, wface, Np, Nfp, RT, partial, nblocks, out, s);
}

// ------------------------------------------------------------------------------------------------------------------
// a2: geometric factors.  One thread per element, registers only (as PAPER.md:L193).
template <int DIM>
__global__ void geometry_kernel(int64_t K, const int32_t* __restrict__ EToV, const double* __restrict__ xv,
                                const double* __restrict__ vv, double* __restrict__ vgeo, double* __restrict__ sgeo,
                                double* __restrict__ vvel) {
  int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (e >= K) return;
  double X[DIM + 1][DIM];
#pragma unroll
  for (int v = 0; v <= DIM; ++v) {
    int64_t id = EToV[e * (DIM + 1) + v];
#pragma unroll
    for (int d = 0; d < DIM; ++d) {
      X[v][d] = xv[id * DIM + d];
      if (vvel) vvel[(e * (DIM + 1) + v) * DIM + d] = vv[id * DIM + d];
    }
  }
  double vg[DIM * DIM + 1], sg[(DIM + 1) * (DIM + 2)];
  element_geometry<DIM>(X, vg, sg);
  if (vgeo)
#pragma unroll
    for (int i = 0; i < DIM * DIM + 1; ++i) vgeo[e * (DIM * DIM + 1) + i] = vg[i];
  if (sgeo)
#pragma unroll
    for (int i = 0; i < (DIM + 1) * (DIM + 2); ++i) sgeo[e * (DIM + 1) * (DIM + 2) + i] = sg[i];
}

cudaError_t launch_geometry(int dim, int64_t K, const int32_t* EToV, const double* xv, const double* vv, double* vgeo,
                            double* sgeo, double* vvel, cudaStream_t s) {
  if (K == 0) return cudaSuccess;
  int nb = (int)((K + 127) / 128);
  if (dim == 2) geometry_kernel<2><<<nb, 128, 0, s>>>(K, EToV, xv, vv, vgeo, sgeo, vvel);
  else geometry_kernel<3><<<nb, 128, 0, s>>>(K, EToV, xv, vv, vgeo, sgeo, vvel);
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------------
// a3-a6: fused stage, generic path.  A persistent CTA stages the operator matrices in shared memory once and loops
// over batches of EB consecutive elements; thread = (element in batch, node).
template <int DIM, int N>
struct StageCfg {
  static constexpr int Np = DIM == 2 ? (N + 1) * (N + 2) / 2 : (N + 1) * (N + 2) * (N + 3) / 6;
  static constexpr int Nfp = DIM == 2 ? N + 1 : (N + 1) * (N + 2) / 2;
  static constexpr int Nfaces = DIM + 1;
  static constexpr int NFN = Nfaces * Nfp;
  static constexpr int Nf = DIM == 2 ? 6 : 10;
  static constexpr int EB = (256 / Np) > 0 ? (256 / Np) : 1;
  static constexpr int Threads = EB * Np;
  static constexpr size_t smem_doubles = (size_t)DIM * Np * Np + (size_t)NFN * Np + (size_t)EB * Nf * Np +
                                         (size_t)EB * Nf * NFN + (size_t)Np * (DIM + 1);
  static constexpr size_t smem_bytes = smem_doubles * 8 + (size_t)NFN * 4;
};

// trace state q+ on a face node, including the boundary states of reading R11
template <int DIM>
__device__ __forceinline__ void exterior_state(int tag, const double* qM, const double* vG, double c,
                                               const double* q_inf, double* qP) {
  constexpr int Nf = DIM == 2 ? 6 : 10;
  if (tag == 1) {  // wall moving with the mesh
#pragma unroll
    for (int k = 0; k < Nf; ++k) qP[k] = qM[k];
#pragma unroll
    for (int d = 0; d < DIM; ++d) qP[1 + d] = 2.0 * qM[0] * vG[d] / c - qM[1 + d];
  } else {  // far field
#pragma unroll
    for (int k = 0; k < Nf; ++k) qP[k] = q_inf[k];
  }
}

template <int DIM, int N>
__global__ void __launch_bounds__(StageCfg<DIM, N>::Threads) stage_kernel(StageArgs a) {
  using C = StageCfg<DIM, N>;
  constexpr int Np = C::Np, Nfp = C::Nfp, Nfaces = C::Nfaces, NFN = C::NFN, Nf = C::Nf, EB = C::EB;
  extern __shared__ double smem[];
  double* sD = smem;                     // [DIM][Np j][Np i]
  double* sL = sD + DIM * Np * Np;       // [NFN m][Np i]
  double* sq = sL + NFN * Np;            // [EB][Nf][Np]
  double* sflux = sq + EB * Nf * Np;     // [EB][Nf][NFN]
  double* slam = sflux + EB * Nf * NFN;  // [Np][DIM+1]
  int* sfmask = reinterpret_cast<int*>(slam + Np * (DIM + 1));
  const int tid = threadIdx.x;
  for (int x = tid; x < DIM * Np * Np; x += C::Threads) sD[x] = a.Dt_ops[x];
  for (int x = tid; x < NFN * Np; x += C::Threads) sL[x] = a.LIFTt[x];
  for (int x = tid; x < Np * (DIM + 1); x += C::Threads) slam[x] = a.lam[x];
  for (int x = tid; x < NFN; x += C::Threads) sfmask[x] = a.fmask[x];
  const int el = tid / Np, i = tid - el * Np;
  const double c = a.c;
  const int64_t nbatch = (a.K + EB - 1) / EB;
  for (int64_t batch = blockIdx.x; batch < nbatch; batch += gridDim.x) {
    const int64_t e0 = batch * EB;
    const int64_t e = e0 + el;
    const bool active = e < a.K;
    __syncthreads();
    {
      const int64_t nel = (a.K - e0) < EB ? (a.K - e0) : EB;
      const int nload = (int)nel * Nf * Np;
      const double* src = a.q_in + e0 * Nf * Np;
      for (int x = tid; x < nload; x += C::Threads) sq[x] = src[x];
    }
    __syncthreads();
    double rhs[Nf];
    if (active) {
      // ---- a3: reference derivatives, dense Np x Np mat-vecs (L103, L195)
      double dr[DIM][Nf];
#pragma unroll
      for (int d = 0; d < DIM; ++d)
#pragma unroll
        for (int k = 0; k < Nf; ++k) dr[d][k] = 0.0;
      for (int j = 0; j < Np; ++j) {
        double dm[DIM];
#pragma unroll
        for (int d = 0; d < DIM; ++d) dm[d] = sD[(d * Np + j) * Np + i];
#pragma unroll
        for (int k = 0; k < Nf; ++k) {
          double qv = sq[(el * Nf + k) * Np + j];
#pragma unroll
          for (int d = 0; d < DIM; ++d) dr[d][k] = fma(dm[d], qv, dr[d][k]);
        }
      }
      const double* vg = a.vgeo + e * (DIM * DIM + 1);
      double G[DIM][DIM];
#pragma unroll
      for (int r = 0; r < DIM; ++r)
#pragma unroll
        for (int d = 0; d < DIM; ++d) G[r][d] = vg[r * DIM + d];
      double vG[DIM];
      node_velocity<DIM>(slam + i * (DIM + 1), a.vvel + e * (DIM + 1) * DIM, vG);
      double gr[DIM][Nf];
#pragma unroll
      for (int d = 0; d < DIM; ++d)
#pragma unroll
        for (int k = 0; k < Nf; ++k) {
          double s = 0.0;
#pragma unroll
          for (int r = 0; r < DIM; ++r) s = fma(G[r][d], dr[r][k], s);
          gr[d][k] = s;
        }
      double st[Nf];
      hermite_apply<DIM>([&](int d, int j) { return gr[d][j]; }, st);
      double qn[Nf];
#pragma unroll
      for (int k = 0; k < Nf; ++k) qn[k] = sq[(el * Nf + k) * Np + i];
      double nt[Nf];
      relaxation_term<DIM>(a, qn, e, i, Np, nt);  // a4 (L115; reading R8, or cubature-projected)
#pragma unroll
      for (int k = 0; k < Nf; ++k) {
        double v = -c * st[k];
#pragma unroll
        for (int d = 0; d < DIM; ++d) v = fma(vG[d], gr[d][k], v);
        rhs[k] = v + nt[k];
      }
      if (a.pml_index != nullptr && a.aux != nullptr) {
        int p = a.pml_index[e];
        if (p >= 0) {
#pragma unroll
          for (int d = 0; d < DIM; ++d) {
            double sig = a.pml_sigma[(int64_t)p * DIM + d];
#pragma unroll
            for (int k = 0; k < Nf; ++k) rhs[k] -= sig * a.aux[(((int64_t)p * DIM + d) * Nf + k) * Np + i];
          }
        }
      }
    }
    // ---- a5: surface flux at the face nodes of the batch (eq. 7; reading R7)
    for (int x = tid; x < EB * NFN; x += C::Threads) {
      const int fe = x / NFN, m = x - fe * NFN;
      const int64_t ee = e0 + fe;
      if (ee >= a.K) break;
      const int f = m / Nfp, n = sfmask[m];
      double qM[Nf], qP[Nf];
#pragma unroll
      for (int k = 0; k < Nf; ++k) qM[k] = sq[(fe * Nf + k) * Np + n];
      const double* sg = a.sgeo + (ee * Nfaces + f) * (DIM + 2);
      double nh[DIM], vG[DIM];
#pragma unroll
      for (int d = 0; d < DIM; ++d) nh[d] = sg[d];
      const double Fscale = sg[DIM + 1];
      node_velocity<DIM>(slam + n * (DIM + 1), a.vvel + ee * (DIM + 1) * DIM, vG);
      const int tag = a.EToB ? a.EToB[ee * Nfaces + f] : 0;
      if (tag == 0) {
        const int idP = a.vmapP[ee * NFN + m];
        const int eP = idP / Np, nP = idP - eP * Np;
        const double* qp = a.q_in + (int64_t)eP * Nf * Np + nP;
#pragma unroll
        for (int k = 0; k < Nf; ++k) qP[k] = qp[k * Np];
      } else {
        exterior_state<DIM>(tag, qM, vG, c, a.q_inf, qP);
      }
      double vn = 0.0;
#pragma unroll
      for (int d = 0; d < DIM; ++d) vn = fma(vG[d], nh[d], vn);
      double fl[Nf];
      upwind_flux<DIM>(qM, qP, nh, c, vn, Fscale, fl);
#pragma unroll
      for (int k = 0; k < Nf; ++k) sflux[(fe * Nf + k) * NFN + m] = fl[k];
    }
    __syncthreads();
    if (active) {
      // ---- LIFT (L103, L196)
      for (int m = 0; m < NFN; ++m) {
        double l = sL[m * Np + i];
#pragma unroll
        for (int k = 0; k < Nf; ++k) rhs[k] = fma(l, sflux[(el * Nf + k) * NFN + m], rhs[k]);
      }
      // ---- a6: SARK stage update (L132-134)
#pragma unroll
      for (int k = 0; k < Nf; ++k) {
        const int64_t idx = (e * Nf + k) * Np + i;
        stage_update(a, k, idx, rhs[k]);
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------------------------
// a8: auxiliary fields of the absorbing layer (reading R12), elements of the layer only.
template <int DIM, int N>
__global__ void __launch_bounds__(StageCfg<DIM, N>::Threads) pml_kernel(PmlArgs a) {
  using C = StageCfg<DIM, N>;
  constexpr int Np = C::Np, Nfp = C::Nfp, Nfaces = C::Nfaces, NFN = C::NFN, Nf = C::Nf, EB = C::EB;
  extern __shared__ double smem[];
  double* sD = smem;
  double* sL = sD + DIM * Np * Np;
  double* sq = sL + NFN * Np;
  double* sflux = sq + EB * Nf * Np;
  double* slam = sflux + EB * Nf * NFN;
  int* sfmask = reinterpret_cast<int*>(slam + Np * (DIM + 1));
  const int tid = threadIdx.x;
  for (int x = tid; x < DIM * Np * Np; x += C::Threads) sD[x] = a.Dt_ops[x];
  for (int x = tid; x < NFN * Np; x += C::Threads) sL[x] = a.LIFTt[x];
  for (int x = tid; x < Np * (DIM + 1); x += C::Threads) slam[x] = a.lam[x];
  for (int x = tid; x < NFN; x += C::Threads) sfmask[x] = a.fmask[x];
  const int el = tid / Np, i = tid - el * Np;
  const double c = a.c;
  const int64_t nbatch = (a.Kpml + EB - 1) / EB;
  for (int64_t batch = blockIdx.x; batch < nbatch; batch += gridDim.x) {
    const int64_t p0 = batch * EB;
    const int64_t p = p0 + el;
    const bool active = p < a.Kpml;
    const int64_t e = active ? a.pml_elems[p] : 0;
    __syncthreads();
    if (active)
      for (int k = 0; k < Nf; ++k) sq[(el * Nf + k) * Np + i] = a.q_in[(e * Nf + k) * Np + i];
    __syncthreads();
    double gr[DIM][Nf];
    if (active) {
      double dr[DIM][Nf];
#pragma unroll
      for (int d = 0; d < DIM; ++d)
#pragma unroll
        for (int k = 0; k < Nf; ++k) dr[d][k] = 0.0;
      for (int j = 0; j < Np; ++j) {
        double dm[DIM];
#pragma unroll
        for (int d = 0; d < DIM; ++d) dm[d] = sD[(d * Np + j) * Np + i];
#pragma unroll
        for (int k = 0; k < Nf; ++k) {
          double qv = sq[(el * Nf + k) * Np + j];
#pragma unroll
          for (int d = 0; d < DIM; ++d) dr[d][k] = fma(dm[d], qv, dr[d][k]);
        }
      }
      const double* vg = a.vgeo + e * (DIM * DIM + 1);
#pragma unroll
      for (int d = 0; d < DIM; ++d)
#pragma unroll
        for (int k = 0; k < Nf; ++k) {
          double s = 0.0;
#pragma unroll
          for (int r = 0; r < DIM; ++r) s = fma(vg[r * DIM + d], dr[r][k], s);
          gr[d][k] = s;
        }
    }
#pragma unroll
    for (int dd = 0; dd < DIM; ++dd) {
      __syncthreads();
      for (int x = tid; x < EB * NFN; x += C::Threads) {
        const int fe = x / NFN, m = x - fe * NFN;
        if (p0 + fe >= a.Kpml) break;
        const int64_t ee = a.pml_elems[p0 + fe];
        const int f = m / Nfp, n = sfmask[m];
        double qM[Nf], qP[Nf];
#pragma unroll
        for (int k = 0; k < Nf; ++k) qM[k] = sq[(fe * Nf + k) * Np + n];
        const double* sg = a.sgeo + (ee * Nfaces + f) * (DIM + 2);
        double nh[DIM];
#pragma unroll
        for (int d = 0; d < DIM; ++d) nh[d] = sg[d];
        const double Fscale = sg[DIM + 1];
        const int tag = a.EToB ? a.EToB[ee * Nfaces + f] : 0;
        if (tag == 0) {
          const int idP = a.vmapP[ee * NFN + m];
          const int eP = idP / Np, nP = idP - eP * Np;
          const double* qp = a.q_in + (int64_t)eP * Nf * Np + nP;
#pragma unroll
          for (int k = 0; k < Nf; ++k) qP[k] = qp[k * Np];
        } else {
          double vG[DIM];
          node_velocity<DIM>(slam + n * (DIM + 1), a.vvel + ee * (DIM + 1) * DIM, vG);
          exterior_state<DIM>(tag, qM, vG, c, a.q_inf, qP);
        }
        double fl[Nf];
        directional_flux<DIM>(dd, qM, qP, nh, c, Fscale, fl);
#pragma unroll
        for (int k = 0; k < Nf; ++k) sflux[(fe * Nf + k) * NFN + m] = fl[k];
      }
      __syncthreads();
      if (active) {
        double G[Nf];
        hermite_apply<DIM>([&](int d, int j) { return d == dd ? gr[dd][j] : 0.0; }, G);
#pragma unroll
        for (int k = 0; k < Nf; ++k) G[k] = -c * G[k];
        for (int m = 0; m < NFN; ++m) {
          double l = sL[m * Np + i];
#pragma unroll
          for (int k = 0; k < Nf; ++k) G[k] = fma(l, sflux[(el * Nf + k) * NFN + m], G[k]);
        }
        const double sig = a.pml_sigma[p * DIM + dd];
#pragma unroll
        for (int k = 0; k < Nf; ++k) {
          const int64_t idx = ((p * DIM + dd) * Nf + k) * Np + i;
          const double g = G[k] - sig * a.aux_in[idx];
          if (a.G_out) a.G_out[idx] = g;
          const double xn = a.aux_n ? a.aux_n[idx] : 0.0;
          const double ac = a.acc_in ? a.acc_in[idx] : 0.0;
          if (a.aux_out) a.aux_out[idx] = fma(a.cx_g, g, fma(a.cx_acc, ac, a.cx_n * xn));
          if (a.acc_out) a.acc_out[idx] = fma(a.cy_g, g, fma(a.cy_acc, ac, a.cy_n * xn));
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------------------------
template <int DIM, int N>
static cudaError_t configure_one() {
  using C = StageCfg<DIM, N>;
  cudaError_t err = cudaFuncSetAttribute(stage_kernel<DIM, N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem_bytes);
  if (err != cudaSuccess) return err;
  return cudaFuncSetAttribute(pml_kernel<DIM, N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem_bytes);
}

template <int DIM, int N>
static cudaError_t launch_stage_one(const StageArgs& a, int num_sms, cudaStream_t s) {
  using C = StageCfg<DIM, N>;
  int64_t nbatch = (a.K + C::EB - 1) / C::EB;
  if (nbatch == 0) return cudaSuccess;
  int per_sm = (int)(200 * 1024 / C::smem_bytes);
  if (per_sm < 1) per_sm = 1;
  if (per_sm > 2048 / C::Threads) per_sm = 2048 / C::Threads;
  int64_t grid = (int64_t)num_sms * per_sm;
  if (grid > nbatch) grid = nbatch;
  stage_kernel<DIM, N><<<(int)grid, C::Threads, C::smem_bytes, s>>>(a);
  return cudaGetLastError();
}

template <int DIM, int N>
static cudaError_t launch_pml_one(const PmlArgs& a, int num_sms, cudaStream_t s) {
  using C = StageCfg<DIM, N>;
  int64_t nbatch = (a.Kpml + C::EB - 1) / C::EB;
  if (nbatch == 0) return cudaSuccess;
  int per_sm = (int)(200 * 1024 / C::smem_bytes);
  if (per_sm < 1) per_sm = 1;
  if (per_sm > 2048 / C::Threads) per_sm = 2048 / C::Threads;
  int64_t grid = (int64_t)num_sms * per_sm;
  if (grid > nbatch) grid = nbatch;
  pml_kernel<DIM, N><<<(int)grid, C::Threads, C::smem_bytes, s>>>(a);
  return cudaGetLastError();
}

#define ALEGB_DISPATCH(FN, ...)                                          \
  switch (dim * 10 + N) {                                                \
    case 21: return FN<2, 1>(__VA_ARGS__);                               \
    case 22: return FN<2, 2>(__VA_ARGS__);                               \
    case 23: return FN<2, 3>(__VA_ARGS__);                               \
    case 24: return FN<2, 4>(__VA_ARGS__);                               \
    case 25: return FN<2, 5>(__VA_ARGS__);                               \
    case 31: return FN<3, 1>(__VA_ARGS__);                               \
    case 32: return FN<3, 2>(__VA_ARGS__);                               \
    case 33: return FN<3, 3>(__VA_ARGS__);                               \
    case 34: return FN<3, 4>(__VA_ARGS__);                               \
    case 35: return FN<3, 5>(__VA_ARGS__);                               \
    default: return cudaErrorInvalidValue;                               \
  }

cudaError_t configure_kernels(int dim, int N) { ALEGB_DISPATCH(configure_one) }
cudaError_t launch_stage(int dim, int N, const StageArgs& a, int num_sms, cudaStream_t s) {
  ALEGB_DISPATCH(launch_stage_one, a, num_sms, s)
}
cudaError_t launch_pml(int dim, int N, const PmlArgs& a, int num_sms, cudaStream_t s) {
  ALEGB_DISPATCH(launch_pml_one, a, num_sms, s)
}

}  // namespace alegb
