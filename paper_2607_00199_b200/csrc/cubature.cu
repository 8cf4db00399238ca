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

// ------------------------------------------------------------------------------------------------------------------
#ifndef ALEGB_CUB_MINB
#define ALEGB_CUB_MINB 1
#endif
#ifndef ALEGB_CUB_WARPS
#define ALEGB_CUB_WARPS 12   // 3 per SM sub-partition (up to 168 registers); 8: 20.1, 16: 22.4, 12: 22.9 GDOF-stage/s on config 4
#endif
// Tensor-core version (DMMA, mma.sync.m8n8k4.f64).  One warp owns a quad of 4 consecutive elements from start to end;
// no shared-memory operand tiles, no block-level synchronisation:
//   * I and P are stored in A-fragment order (lane l of fragment (row tile, k-step) holds A[8 tile + l/4][4 k + l%4]),
//     so an operand is one coalesced 256-byte load; both matrices (99 + 110 kB at 3-D N = 4) are shared by every warp
//     of the SM and live in L1 (the kernel uses < 13 kB of shared memory);
//   * the quad's input fields are the B operand of the interpolation and stay in registers for all row tiles:
//     column g <-> (element g/2, field 2t + g%2) as in stage_pipe.cu, so after the contraction lane (g, c) holds
//     q1 .. q_{1+dim} of element c at cubature node 8 rt + g and evaluates N~ there (L115);
//   * the projection is a K-accumulation over the cubature nodes, so it is fused block by block: the 8 nodes of a row
//     tile are 2 k-steps of P N~; N~ goes through a 2 kB warp-private staging tile to become a B fragment;
//   * the result leaves the accumulators in the layout of the stage kernels (lane = node, element).
template <int DIM, int N>
struct CubCfg {
  static constexpr int Np = DIM == 2 ? (N + 1) * (N + 2) / 2 : (N + 1) * (N + 2) * (N + 3) / 6;
  static constexpr int NQ = 3 * N / 2 + 1;                       // Gauss-Jacobi points per direction, degree 3N
  static constexpr int Nc = DIM == 2 ? NQ * NQ : NQ * NQ * NQ;
  static constexpr int NRT = (Nc + 7) / 8;                       // row tiles of the interpolation = blocks of 8 nodes
  static constexpr int KS = (Np + 3) / 4;                        // k-steps of the interpolation
  static constexpr int NB = (Np + 7) / 8;                        // row tiles of the projection
  static constexpr int NS = DIM * (DIM + 1) / 2;                 // stiff fields
  static constexpr int NT2 = (NS + 1) / 2;                       // column tiles of the projection (field pairs)
  static constexpr int NSP = 2 * NT2;
  static constexpr int ST = 10;                                  // staging row stride (doubles)
  static constexpr int Warps = ALEGB_CUB_WARPS;
  static constexpr int stage_doubles = 4 * NSP * ST;
  static constexpr size_t smem_bytes = (size_t)Warps * stage_doubles * 8;
};

__device__ __forceinline__ void cub_dmma(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

template <int DIM, int N>
__global__ void __launch_bounds__(CubCfg<DIM, N>::Warps * 32, ALEGB_CUB_MINB) cubature_mma_kernel(CubArgs a) {
  using C = CubCfg<DIM, N>;
  constexpr int Np = C::Np, Nc = C::Nc, NRT = C::NRT, KS = C::KS, NB = C::NB, NS = C::NS, NT2 = C::NT2, NSP = C::NSP;
  constexpr int ST = C::ST, Nf = DIM == 2 ? 6 : 10;
  extern __shared__ double sm[];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, g = lane >> 2, c = lane & 3;
  double* sN = sm + warp * C::stage_doubles;              // [4 elements x NSP fields][ST]: N~ at the 8 nodes of a block
  for (int x = lane; x < C::stage_doubles; x += 32) sN[x] = 0.0;
  __syncwarp();
  const int64_t nquads = (a.K + 3) / 4;
  for (int64_t quad = (int64_t)blockIdx.x * C::Warps + warp; quad < nquads; quad += (int64_t)gridDim.x * C::Warps) {
    const int64_t e0 = quad * 4;
    const int nel = (a.K - e0) < 4 ? (int)(a.K - e0) : 4;
    // B operand of the interpolation, two column tiles: tile t, column g <-> (element g/2, field 2t + g%2); k = c
    double bq[KS][2];
    {
      const int eb = (g >> 1) < nel ? (g >> 1) : 0;
#pragma unroll
      for (int t = 0; t < 2; ++t) {
        const int f = 2 * t + (g & 1);
        const double* src = a.q + ((e0 + eb) * Nf + (f <= DIM ? f : 0)) * Np;
#pragma unroll
        for (int ks = 0; ks < KS; ++ks) {
          const int j = 4 * ks + c;
          bq[ks][t] = (f <= DIM && j < Np) ? __ldg(src + j) : 0.0;
        }
      }
    }
    double acc2[NB][NT2][2];
#pragma unroll
    for (int r = 0; r < NB; ++r)
#pragma unroll
      for (int t = 0; t < NT2; ++t) acc2[r][t][0] = acc2[r][t][1] = 0.0;
#pragma unroll 1
    for (int rt = 0; rt < NRT; ++rt) {
      // ---- interpolation to the 8 cubature nodes of this block (L86): lane (g, c) <- node 8 rt + g, element c
      double i0[2] = {0.0, 0.0}, i1[2] = {0.0, 0.0};
      const double* ai = a.AI + ((size_t)rt * KS) * 32 + lane;
#pragma unroll
      for (int ks = 0; ks < KS; ++ks) {
        const double af = __ldg(ai + ks * 32);
        cub_dmma(i0[0], i0[1], af, bq[ks][0]);
        cub_dmma(i1[0], i1[1], af, bq[ks][1]);
      }
      // ---- N~ at the node (L115)
      double qq[Nf], nt[Nf];
#pragma unroll
      for (int f = 0; f < Nf; ++f) qq[f] = 0.0;
      qq[0] = i0[0]; qq[1] = i0[1]; qq[2] = i1[0];
      if constexpr (DIM == 3) qq[3] = i1[1];
      const bool pvalid = 8 * rt + g < Nc;
      if (!pvalid) qq[0] = 1.0;                           // padding node: any finite value, its P column is zero
      relaxation<DIM>(qq, a.invtau, nt);
      __syncwarp();
#pragma unroll
      for (int s = 0; s < NS; ++s) sN[(c * NSP + s) * ST + g] = pvalid ? nt[DIM + 1 + s] : 0.0;
      __syncwarp();
      // ---- projection, K-accumulated over this block's 2 k-steps (L103)
#pragma unroll
      for (int k2 = 0; k2 < 2; ++k2) {
        double bf[NT2];
#pragma unroll
        for (int t = 0; t < NT2; ++t) bf[t] = sN[((g >> 1) * NSP + 2 * t + (g & 1)) * ST + 4 * k2 + c];
        const double* ap = a.AP + ((size_t)(2 * rt + k2)) * 32 + lane;
#pragma unroll
        for (int r = 0; r < NB; ++r) {
          const double af = __ldg(ap + (size_t)r * (2 * NRT) * 32);
#pragma unroll
          for (int t = 0; t < NT2; ++t) cub_dmma(acc2[r][t][0], acc2[r][t][1], af, bf[t]);
        }
      }
    }
    // ---- store: lane (g, c) holds node 8 r + g of element c, fields 2t, 2t+1
    if (c < nel) {
#pragma unroll
      for (int r = 0; r < NB; ++r) {
        const int i = 8 * r + g;
        if (i < Np) {
#pragma unroll
          for (int t = 0; t < NT2; ++t)
#pragma unroll
            for (int h = 0; h < 2; ++h)
              if (2 * t + h < NS) a.R[((e0 + c) * NS + 2 * t + h) * Np + i] = acc2[r][t][h];
        }
      }
    }
  }
}

template <int DIM, int N>
static cudaError_t launch_cub_mma_one(const CubArgs& a, int num_sms, cudaStream_t s) {
  using C = CubCfg<DIM, N>;
  const int64_t nquads = (a.K + 3) / 4;
  if (nquads == 0) return cudaSuccess;
  const int64_t want = (nquads + C::Warps - 1) / C::Warps;
  const int64_t cap = (int64_t)num_sms * ALEGB_CUB_MINB;
  cubature_mma_kernel<DIM, N><<<(int)(want < cap ? want : cap), C::Warps * 32, C::smem_bytes, s>>>(a);
  return cudaGetLastError();
}

void cubature_mma_layout(int dim, int N, int& NRT, int& KS, int& NB) {
  const int Np = dim == 2 ? (N + 1) * (N + 2) / 2 : (N + 1) * (N + 2) * (N + 3) / 6;
  const int NQ = 3 * N / 2 + 1, Nc = dim == 2 ? NQ * NQ : NQ * NQ * NQ;
  NRT = (Nc + 7) / 8; KS = (Np + 3) / 4; NB = (Np + 7) / 8;
}

bool cubature_mma_available(int dim, int N) {   // the (dim, N) pairs launch_cubature_mma dispatches
  return (dim == 2 && N >= 1 && N <= 5) || (dim == 3 && N >= 1 && N <= 4);
}

cudaError_t launch_cubature_mma(int dim, int N, const CubArgs& a, int num_sms, cudaStream_t s) {
  switch (dim * 10 + N) {
    case 21: return launch_cub_mma_one<2, 1>(a, num_sms, s);
    case 22: return launch_cub_mma_one<2, 2>(a, num_sms, s);
    case 23: return launch_cub_mma_one<2, 3>(a, num_sms, s);
    case 24: return launch_cub_mma_one<2, 4>(a, num_sms, s);
    case 25: return launch_cub_mma_one<2, 5>(a, num_sms, s);
    case 31: return launch_cub_mma_one<3, 1>(a, num_sms, s);
    case 32: return launch_cub_mma_one<3, 2>(a, num_sms, s);
    case 33: return launch_cub_mma_one<3, 3>(a, num_sms, s);
    case 34: return launch_cub_mma_one<3, 4>(a, num_sms, s);
    default: return cudaErrorInvalidValue;
  }
}

}  // namespace alegb
