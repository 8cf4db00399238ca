// Fused stage kernel on the fp64 tensor-core path (DMMA, mma.sync.m8n8k4.f64) for sm_100a.
//
// Why DMMA: the 3-D N=4 stage needs ~380 flop per degree of freedom against ~38 B of HBM traffic, i.e. it is bound by
// the SM's fp64 pipe, not by HBM.  On B200 DFMA and DMMA run on the same pipe at the same peak (measured, see
// profiles/fp64_peak_r1.md), but DMMA takes its operands as register fragments: 256 FMA per instruction for two
// 8-byte shared-memory loads, where the DFMA form needs ~0.4 shared-memory wavefronts per warp-DFMA and stalls there.
//
// Work decomposition: a warp owns a group of 4 consecutive elements from load to store; warps of a CTA share only
// the operator fragments in shared memory.  Both contractions of the stage are written as C[node, col] += A * B with
//     rows    = nodes, in blocks of 8 (NB blocks),
//     columns = 8 per tile: (element c = 0..3) x (field pair member h = 0,1) of field pair t (NT = Nf/2 tiles),
//     K       = nodes j (volume, D_a) or face nodes m of one face (surface, LIFT).
// In the m8n8k4 accumulator layout lane (g = lane/4, c = lane%4) then holds, for node 8*nb+g of element c, the
// derivatives d/dr, d/ds, d/dt of ALL fields -- exactly the operands of the point-wise volume term (metrics, moment
// system matrices, mesh-velocity advection, relaxation), which therefore runs on the accumulator registers with no
// shared-memory round trip; the LIFT contraction accumulates into the same registers and the SARK update and the
// global stores are issued from them.
#include "alegb_internal.h"
#include "device_common.cuh"

namespace alegb {

__host__ __device__ constexpr int stride_pad(int x) {
  // smallest s >= x with s = 4 (mod 16): the 8 columns x 4 k-values of a B fragment then fall on 16 distinct
  // 8-byte bank pairs twice each, i.e. the 2 wavefronts a 256-byte warp load needs at minimum
  int s = x;
  while (s % 16 != 4) ++s;
  return s;
}

template <int DIM, int N>
struct MmaCfg {
  static constexpr int Np = DIM == 2 ? (N + 1) * (N + 2) / 2 : (N + 1) * (N + 2) * (N + 3) / 6;
  static constexpr int Nfp = DIM == 2 ? N + 1 : (N + 1) * (N + 2) / 2;
  static constexpr int Nfaces = DIM + 1;
  static constexpr int NFN = Nfaces * Nfp;
  static constexpr int Nf = DIM == 2 ? 6 : 10;
  static constexpr int NT = Nf / 2;            // column tiles (field pairs)
  static constexpr int NB = (Np + 7) / 8;      // node blocks (row tiles)
  static constexpr int KS = (Np + 3) / 4;      // k-steps of the volume contraction
  static constexpr int KF = (Nfp + 3) / 4;     // k-steps of the surface contraction, per face
  static constexpr int S = stride_pad(4 * KS);   // node stride of a q-tile row
  static constexpr int SG = stride_pad(4 * KF);  // face-node stride of a flux-tile row
  static constexpr int EG = 4;                 // elements per warp group
  static constexpr int WARPS = 8;
  static constexpr int Threads = WARPS * 32;
  static constexpr int avol_doubles = DIM * NB * KS * 32;
  static constexpr int alift_doubles = Nfaces * NB * KF * 32;
  static constexpr int lam_doubles = NB * 8 * (DIM + 1);
  static constexpr int qtile_doubles = EG * Nf * S;
  static constexpr int gtile_doubles = EG * Nf * SG;
  static constexpr size_t smem_bytes =
      (size_t)(avol_doubles + alift_doubles + lam_doubles + WARPS * (qtile_doubles + gtile_doubles)) * 8 + (size_t)NFN * 4;
  static constexpr bool supported = (NB * Nf <= 50) && smem_bytes <= 227 * 1024;
};

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

template <int DIM, int N>
__global__ void __launch_bounds__(MmaCfg<DIM, N>::Threads, 1) stage_mma_kernel(StageArgs a) {
  using C = MmaCfg<DIM, N>;
  constexpr int Np = C::Np, Nfp = C::Nfp, Nfaces = C::Nfaces, NFN = C::NFN, Nf = C::Nf, NT = C::NT, NB = C::NB;
  constexpr int KS = C::KS, KF = C::KF, S = C::S, SG = C::SG, EG = C::EG;
  extern __shared__ double smem[];
  double* sAvol = smem;                              // [DIM][NB][KS][32] fragment order
  double* sAlift = sAvol + C::avol_doubles;          // [Nfaces][NB][KF][32]
  double* slam = sAlift + C::alift_doubles;          // [NB*8][DIM+1], rows >= Np repeat the last node
  double* stiles = slam + C::lam_doubles;
  int* sfmask = reinterpret_cast<int*>(stiles + C::WARPS * (C::qtile_doubles + C::gtile_doubles));
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = lane >> 2, c = lane & 3;
  double* qt = stiles + warp * (C::qtile_doubles + C::gtile_doubles);   // [EG*Nf][S]
  double* gt = qt + C::qtile_doubles;                                   // [EG*Nf][SG]

  for (int x = tid; x < C::avol_doubles; x += C::Threads) sAvol[x] = a.Avol[x];
  for (int x = tid; x < C::alift_doubles; x += C::Threads) sAlift[x] = a.Alift[x];
  for (int x = tid; x < NB * 8; x += C::Threads) {
    const int n = x < Np ? x : Np - 1;
#pragma unroll
    for (int v = 0; v <= DIM; ++v) slam[x * (DIM + 1) + v] = a.lam[n * (DIM + 1) + v];
  }
  for (int x = tid; x < NFN; x += C::Threads) sfmask[x] = a.fmask[x];
  // zero both tiles once: the k-padding (j >= Np, m >= Nfp) is never written again and must multiply as 0
  for (int x = lane; x < C::qtile_doubles + C::gtile_doubles; x += 32) qt[x] = 0.0;
  __syncthreads();

  const double cs = a.c;
  const int64_t ngroups = (a.K + EG - 1) / EG;
  // B-fragment column of this lane: column j = g  <->  element g/2, field 2t + (g&1); k index = c
  const int bcol = (g >> 1) * Nf + (g & 1);
  for (int64_t grp = (int64_t)blockIdx.x * C::WARPS + warp; grp < ngroups; grp += (int64_t)gridDim.x * C::WARPS) {
    const int64_t e0 = grp * EG;
    const int nel = (a.K - e0) < EG ? (int)(a.K - e0) : EG;
    // ---- q tile of the group: [element][field][node] with node stride S
    {
      const double* src = a.q_in + e0 * Nf * Np;
      const int total = nel * Nf * Np;
      for (int x = lane; x < total; x += 32) {
        const int row = x / Np, j = x - row * Np;
        qt[row * S + j] = __ldg(src + x);
      }
    }
    __syncwarp();
    const bool evalid = c < nel;
    const int64_t e = e0 + (evalid ? c : 0);      // element of this lane in the accumulator layout
    // geometry of element e (constant per element: affine, L88-92)
    double G[DIM][DIM], vv[DIM + 1][DIM];
    {
      const double* vg = a.vgeo + e * (DIM * DIM + 1);
#pragma unroll
      for (int r = 0; r < DIM; ++r)
#pragma unroll
        for (int d = 0; d < DIM; ++d) G[r][d] = vg[r * DIM + d];
      const double* ve = a.vvel + e * (DIM + 1) * DIM;
#pragma unroll
      for (int v = 0; v <= DIM; ++v)
#pragma unroll
        for (int d = 0; d < DIM; ++d) vv[v][d] = ve[v * DIM + d];
    }
    int pml = -1;
    if (a.pml_index != nullptr && a.aux != nullptr) pml = a.pml_index[e];

    double V[NB][NT][2];   // F at (node 8nb+g, element c, field 2t+h), accumulator layout
    // ---- a3 + a4: volume contraction and point-wise terms, one node block at a time
#pragma unroll
    for (int nb = 0; nb < NB; ++nb) {
      double acc[DIM][NT][2];
#pragma unroll
      for (int d = 0; d < DIM; ++d)
#pragma unroll
        for (int t = 0; t < NT; ++t) acc[d][t][0] = acc[d][t][1] = 0.0;
#pragma unroll
      for (int ks = 0; ks < KS; ++ks) {
        double bf[NT], af[DIM];
#pragma unroll
        for (int t = 0; t < NT; ++t) bf[t] = qt[(bcol + 2 * t) * S + 4 * ks + c];
#pragma unroll
        for (int d = 0; d < DIM; ++d) af[d] = sAvol[((d * NB + nb) * KS + ks) * 32 + lane];
#pragma unroll
        for (int d = 0; d < DIM; ++d)
#pragma unroll
          for (int t = 0; t < NT; ++t) dmma(acc[d][t][0], acc[d][t][1], af[d], bf[t]);
      }
      // point-wise: node n of element c
      const int n = 8 * nb + g;
      const int nn = n < Np ? n : Np - 1;
      double vG[DIM];
#pragma unroll
      for (int d = 0; d < DIM; ++d) {
        double s = 0.0;
#pragma unroll
        for (int v = 0; v <= DIM; ++v) s = fma(slam[n * (DIM + 1) + v], vv[v][d], s);
        vG[d] = s;
      }
      double gr[DIM][Nf];
#pragma unroll
      for (int d = 0; d < DIM; ++d)
#pragma unroll
        for (int k = 0; k < Nf; ++k) {
          double s = 0.0;
#pragma unroll
          for (int r = 0; r < DIM; ++r) s = fma(G[r][d], acc[r][k >> 1][k & 1], s);
          gr[d][k] = s;
        }
      double st[Nf], qn[Nf], nt[Nf];
      hermite_apply<DIM>([&](int d, int j) { return gr[d][j]; }, st);
#pragma unroll
      for (int k = 0; k < Nf; ++k) qn[k] = qt[(c * Nf + k) * S + nn];
      relaxation_term<DIM>(a, qn, e, nn, Np, nt);
#pragma unroll
      for (int k = 0; k < Nf; ++k) {
        double v = -cs * st[k];
#pragma unroll
        for (int d = 0; d < DIM; ++d) v = fma(vG[d], gr[d][k], v);
        V[nb][k >> 1][k & 1] = v + nt[k];
      }
      if (pml >= 0) {
#pragma unroll
        for (int d = 0; d < DIM; ++d) {
          const double sig = a.pml_sigma[(int64_t)pml * DIM + d];
#pragma unroll
          for (int k = 0; k < Nf; ++k)
            V[nb][k >> 1][k & 1] -= sig * a.aux[(((int64_t)pml * DIM + d) * Nf + k) * Np + nn];
        }
      }
    }

    // ---- a5: surface flux and LIFT contraction, one face at a time
#pragma unroll 1
    for (int f = 0; f < Nfaces; ++f) {
      for (int task = lane; task < EG * Nfp; task += 32) {
        const int fe = task / Nfp, m = task - fe * Nfp;
        double fl[Nf];
        if (fe < nel) {
          const int64_t ee = e0 + fe;
          const int n = sfmask[f * Nfp + m];
          double qM[Nf], qP[Nf];
#pragma unroll
          for (int k = 0; k < Nf; ++k) qM[k] = qt[(fe * Nf + k) * S + n];
          const double* sg = a.sgeo + (ee * Nfaces + f) * (DIM + 2);
          double nh[DIM], vG[DIM];
#pragma unroll
          for (int d = 0; d < DIM; ++d) nh[d] = sg[d];
          const double Fscale = sg[DIM + 1];
          node_velocity<DIM>(slam + n * (DIM + 1), a.vvel + ee * (DIM + 1) * DIM, vG);
          const int tag = a.EToB ? a.EToB[ee * Nfaces + f] : 0;
          if (tag == 0) {
            const int idP = a.vmapP[ee * NFN + f * Nfp + m];
            const int eP = idP / Np, nP = idP - eP * Np;
            const double* qp = a.q_in + (int64_t)eP * Nf * Np + nP;
#pragma unroll
            for (int k = 0; k < Nf; ++k) qP[k] = __ldg(qp + k * Np);
          } else if (tag == 1) {
#pragma unroll
            for (int k = 0; k < Nf; ++k) qP[k] = qM[k];
#pragma unroll
            for (int d = 0; d < DIM; ++d) qP[1 + d] = 2.0 * qM[0] * vG[d] / cs - qM[1 + d];
          } else {
#pragma unroll
            for (int k = 0; k < Nf; ++k) qP[k] = a.q_inf[k];
          }
          double vn = 0.0;
#pragma unroll
          for (int d = 0; d < DIM; ++d) vn = fma(vG[d], nh[d], vn);
          upwind_flux<DIM>(qM, qP, nh, cs, vn, Fscale, fl);
        } else {
#pragma unroll
          for (int k = 0; k < Nf; ++k) fl[k] = 0.0;
        }
#pragma unroll
        for (int k = 0; k < Nf; ++k) gt[(fe * Nf + k) * SG + m] = fl[k];
      }
      __syncwarp();
#pragma unroll
      for (int ks = 0; ks < KF; ++ks) {
        double bf[NT];
#pragma unroll
        for (int t = 0; t < NT; ++t) bf[t] = gt[(bcol + 2 * t) * SG + 4 * ks + c];
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) {
          const double af = sAlift[((f * NB + nb) * KF + ks) * 32 + lane];
#pragma unroll
          for (int t = 0; t < NT; ++t) dmma(V[nb][t][0], V[nb][t][1], af, bf[t]);
        }
      }
      __syncwarp();
    }

    // ---- a6: SARK stage update, straight from the accumulator registers
    if (evalid) {
      const bool qn_in_tile = a.q_n == a.q_in;
#pragma unroll
      for (int nb = 0; nb < NB; ++nb) {
        const int n = 8 * nb + g;
        if (n < Np) {
#pragma unroll
          for (int k = 0; k < Nf; ++k) {
            const int64_t idx = (e * Nf + k) * Np + n;
            const double F = V[nb][k >> 1][k & 1];
            if (a.F_out) a.F_out[idx] = F;
            if (a.q_out != nullptr || a.acc_out != nullptr) {
              const double qn = a.q_n ? (qn_in_tile ? qt[(c * Nf + k) * S + n] : a.q_n[idx]) : 0.0;
              const double f0 = a.F0_in ? a.F0_in[idx] : 0.0;
              const double ac = a.acc_in ? a.acc_in[idx] : 0.0;
              if (a.q_out) {
                double v = a.coef.cq_n[k] * qn;
                v = fma(a.coef.cq_f0[k], f0, v);
                v = fma(a.coef.cq_acc, ac, v);
                a.q_out[idx] = fma(a.coef.cq_f[k], F, v);
              }
              if (a.acc_out) {
                double v = a.coef.ca_n[k] * qn;
                v = fma(a.coef.ca_f0[k], f0, v);
                v = fma(a.coef.ca_acc, ac, v);
                a.acc_out[idx] = fma(a.coef.ca_f[k], F, v);
              }
            }
          }
        }
      }
    }
    __syncwarp();   // the q tile is reused by the next group
  }
}

// ------------------------------------------------------------------------------------------------------------------
template <int DIM, int N>
static cudaError_t launch_mma_one(const StageArgs& a, int num_sms, cudaStream_t s, bool configure_only) {
  using C = MmaCfg<DIM, N>;
  if constexpr (!C::supported) {
    return cudaErrorInvalidValue;
  } else {
    if (configure_only)
      return cudaFuncSetAttribute(stage_mma_kernel<DIM, N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem_bytes);
    const int64_t ngroups = (a.K + C::EG - 1) / C::EG;
    if (ngroups == 0) return cudaSuccess;
    int64_t grid = (ngroups + C::WARPS - 1) / C::WARPS;
    if (grid > num_sms) grid = num_sms;
    stage_mma_kernel<DIM, N><<<(int)grid, C::Threads, C::smem_bytes, s>>>(a);
    return cudaGetLastError();
  }
}

#define ALEGB_MMA_DISPATCH(...)                                  \
  switch (dim * 10 + N) {                                        \
    case 21: return launch_mma_one<2, 1>(__VA_ARGS__);           \
    case 22: return launch_mma_one<2, 2>(__VA_ARGS__);           \
    case 23: return launch_mma_one<2, 3>(__VA_ARGS__);           \
    case 24: return launch_mma_one<2, 4>(__VA_ARGS__);           \
    case 25: return launch_mma_one<2, 5>(__VA_ARGS__);           \
    case 31: return launch_mma_one<3, 1>(__VA_ARGS__);           \
    case 32: return launch_mma_one<3, 2>(__VA_ARGS__);           \
    case 33: return launch_mma_one<3, 3>(__VA_ARGS__);           \
    case 34: return launch_mma_one<3, 4>(__VA_ARGS__);           \
    default: return cudaErrorInvalidValue;                       \
  }

cudaError_t launch_stage_mma(int dim, int N, const StageArgs& a, int num_sms, cudaStream_t s) {
  ALEGB_MMA_DISPATCH(a, num_sms, s, false)
}
cudaError_t configure_stage_mma(int dim, int N) {
  StageArgs a{};
  ALEGB_MMA_DISPATCH(a, 0, nullptr, true)
}

bool mma_layout(int dim, int N, MmaLayout& L) {
  auto fill = [&](auto cfg) {
    using C = decltype(cfg);
    L.NB = C::NB; L.KS = C::KS; L.KF = C::KF;
    return C::supported;
  };
  switch (dim * 10 + N) {
    case 21: return fill(MmaCfg<2, 1>{});
    case 22: return fill(MmaCfg<2, 2>{});
    case 23: return fill(MmaCfg<2, 3>{});
    case 24: return fill(MmaCfg<2, 4>{});
    case 25: return fill(MmaCfg<2, 5>{});
    case 31: return fill(MmaCfg<3, 1>{});
    case 32: return fill(MmaCfg<3, 2>{});
    case 33: return fill(MmaCfg<3, 3>{});
    case 34: return fill(MmaCfg<3, 4>{});
    default: return false;
  }
}

}  // namespace alegb
