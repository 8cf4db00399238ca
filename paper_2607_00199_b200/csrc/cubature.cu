// Cubature-projected nonlinear relaxation  R = P N~(I q)  (eq. 9 last term; kernel v of L197;
// SURVEY 8(f) NEXT-1).  R replaces the collocated N~(q) of reading R8 inside the stage kernels when
// alegb_set_relaxation(ALEGB_RELAX_CUBATURE) is active.
//
// Kept from the paper's kernel (L197): fields copied to shared memory, interpolated to the N_c cubature nodes with I,
// nonlinear term evaluated there and kept in shared memory, projected back with P.  Changed: a CTA handles EB =
// 256 / Np elements at once so that both phases fill the block (the paper's block per element leaves N_c - Np
// threads idle in the projection), I and P are read transposed (coalesced, served by L1/L2 for all elements of the
// CTA), and only what N~ needs moves: 1 + dim input fields, the dim (dim + 1) / 2 stiff output fields.
//
// First version on the DFMA path: per element 2 Nc Np (1 + dim + Ns) flop, 240 kflop at 3-D N = 4 (Nc = 343) --
// twice the rest of the stage.  The DMMA version (rows = cubature nodes / nodes, columns = element x field pairs as
// in stage_pipe.cu) is the next step; see DESIGN.md.
#include "alegb_internal.h"
#include "device_common.cuh"

namespace alegb {

template <int DIM>
__global__ void __launch_bounds__(256) cubature_relax_kernel(CubArgs a) {
  constexpr int NI = 4;                       // input fields per node, padded (q1 .. q_{1+DIM})
  constexpr int NS = DIM * (DIM + 1) / 2;     // stiff fields
  constexpr int Nf = DIM == 2 ? 6 : 10;
  extern __shared__ double sm[];
  const int Np = a.Np, Nc = a.Nc, EB = a.EB;
  double* qs = sm;                            // [EB][Np][NI]
  double* nc = sm + (size_t)EB * Np * NI;     // [EB][Nc][NS]
  const int tid = threadIdx.x;
  for (int64_t e0 = (int64_t)blockIdx.x * EB; e0 < a.K; e0 += (int64_t)gridDim.x * EB) {
    const int nel = (a.K - e0) < EB ? (int)(a.K - e0) : EB;
    __syncthreads();
    for (int x = tid; x < nel * Np * NI; x += blockDim.x) {
      const int f = x % NI, j = (x / NI) % Np, e = x / (NI * Np);
      qs[x] = f <= DIM ? a.q[((e0 + e) * Nf + f) * Np + j] : 0.0;
    }
    __syncthreads();
    // ---- interpolate to the cubature nodes (L86), nonlinear term there (L115)
    for (int x = tid; x < nel * Nc; x += blockDim.x) {
      const int c = x % Nc, e = x / Nc;
      double v[NI];
#pragma unroll
      for (int f = 0; f < NI; ++f) v[f] = 0.0;
      const double* qe = qs + (size_t)e * Np * NI;
      for (int j = 0; j < Np; ++j) {
        const double w = __ldg(a.It + (size_t)j * Nc + c);
        const double2 q01 = *reinterpret_cast<const double2*>(qe + j * NI);
        const double2 q23 = *reinterpret_cast<const double2*>(qe + j * NI + 2);
        v[0] = fma(w, q01.x, v[0]); v[1] = fma(w, q01.y, v[1]);
        v[2] = fma(w, q23.x, v[2]); v[3] = fma(w, q23.y, v[3]);
      }
      double qq[Nf], nt[Nf];
#pragma unroll
      for (int f = 0; f < Nf; ++f) qq[f] = f <= DIM ? v[f] : 0.0;
      relaxation<DIM>(qq, a.invtau, nt);
      double* dst = nc + ((size_t)e * Nc + c) * NS;
#pragma unroll
      for (int s = 0; s < NS; ++s) dst[s] = nt[DIM + 1 + s];
    }
    __syncthreads();
    // ---- project back to the interpolation nodes (L103)
    for (int x = tid; x < nel * Np; x += blockDim.x) {
      const int i = x % Np, e = x / Np;
      double r[NS];
#pragma unroll
      for (int s = 0; s < NS; ++s) r[s] = 0.0;
      const double* ne = nc + (size_t)e * Nc * NS;
      for (int c = 0; c < Nc; ++c) {
        const double w = __ldg(a.Pt + (size_t)c * Np + i);
#pragma unroll
        for (int s = 0; s < NS; ++s) r[s] = fma(w, ne[c * NS + s], r[s]);
      }
#pragma unroll
      for (int s = 0; s < NS; ++s) a.R[((e0 + e) * NS + s) * Np + i] = r[s];
    }
  }
}

size_t cubature_smem_bytes(int dim, int Np, int Nc, int EB) {
  const int NS = dim * (dim + 1) / 2;
  return ((size_t)EB * Np * 4 + (size_t)EB * Nc * NS) * sizeof(double);
}

cudaError_t configure_cubature(int dim, size_t smem) {
  if (dim == 2) return cudaFuncSetAttribute(cubature_relax_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  return cudaFuncSetAttribute(cubature_relax_kernel<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
}

cudaError_t launch_cubature(int dim, const CubArgs& a, int num_sms, cudaStream_t s) {
  if (a.K == 0) return cudaSuccess;
  const size_t smem = cubature_smem_bytes(dim, a.Np, a.Nc, a.EB);
  const int64_t groups = (a.K + a.EB - 1) / a.EB;
  const int per_sm = smem > 110 * 1024 ? 1 : (smem > 70 * 1024 ? 2 : 4);
  int64_t grid = groups < (int64_t)num_sms * per_sm ? groups : (int64_t)num_sms * per_sm;
  if (dim == 2) cubature_relax_kernel<2><<<(int)grid, 256, smem, s>>>(a);
  else cubature_relax_kernel<3><<<(int)grid, 256, smem, s>>>(a);
  return cudaGetLastError();
}

}  // namespace alegb
