// a8 on the fp64 tensor-core path: auxiliary fields of the absorbing layer (reading R12) for the flagged elements,
//   d/dt q~^d = -c A^_d d_d q + LIFT( Fscale ( -1/2 n_d c A^_d [q] + 1/2 n_d^2 |A_n| [q] ) ) - sigma_d q~^d ,  d = 1..DIM.
//
// Why: the generic pml_kernel (kernels.cu) spends its time in DIM dense LIFT mat-vecs per element on the DFMA path
// and re-gathers the exterior traces once per direction; on config 5 (36 % of the elements in the layer) it took
// 15.3 ms per stage, three times the fused stage kernel (profiles/r1_pml_kernel.md).  Here a team of two warps owns a
// "quad" of 4 layer elements: the q tile and the DIM directional flux tiles (one gather of q+, |A_n|[q] shared by the
// directions) live in shared memory, D_r,D_s,D_t q is one DMMA contraction per 8-node block (operands and lane layout
// as in stage_pipe.cu), each direction's volume term is formed on the accumulator registers and its LIFT contraction
// accumulates into them, and the RK combination of the auxiliary state is stored from the registers.
#include "alegb_internal.h"
#include "device_common.cuh"

namespace alegb {

namespace pmlmma {

__host__ __device__ constexpr int stride_pad(int x) {
  int s = x;   // s = 4 (mod 8): conflict-free B-fragment loads (see stage_pipe.cu)
  while (s % 8 != 4) ++s;
  return s;
}

template <int DIM, int N>
struct Cfg {
  static constexpr int Np = DIM == 2 ? (N + 1) * (N + 2) / 2 : (N + 1) * (N + 2) * (N + 3) / 6;
  static constexpr int Nfp = DIM == 2 ? N + 1 : (N + 1) * (N + 2) / 2;
  static constexpr int Nfaces = DIM + 1;
  static constexpr int NFN = Nfaces * Nfp;
  static constexpr int Nf = DIM == 2 ? 6 : 10;
  static constexpr int NT = Nf / 2;
  static constexpr int NB = (Np + 7) / 8;
  static constexpr int KS = (Np + 3) / 4;
  static constexpr int KFT = (NFN + 3) / 4;
  static constexpr int S = stride_pad(4 * KS);
  static constexpr int SG = stride_pad(4 * KFT);
  static constexpr int EG = 4;                   // elements per quad
  static constexpr int TW = 2;                   // warps per team (one team per quad)
  static constexpr int TT = TW * 32;             // threads per team
  static constexpr int avol_doubles = DIM * NB * KS * 32;
  static constexpr int alift_doubles = NB * KFT * 32;
  static constexpr int lam_doubles = NB * 8 * (DIM + 1);
  static constexpr int qtile_doubles = EG * Nf * S;
  static constexpr int gtile_doubles = EG * Nf * SG;             // one per direction
  static constexpr int team_doubles = qtile_doubles + DIM * gtile_doubles;
  static constexpr size_t fixed_bytes = (size_t)(avol_doubles + alift_doubles + lam_doubles) * 8 + (size_t)NFN * 4 + 16;
  static constexpr int teams_fit = (int)((216 * 1024 - fixed_bytes) / ((size_t)team_doubles * 8));
  static constexpr int TEAMS = teams_fit > 4 ? 4 : teams_fit;    // teams per CTA
  static constexpr int Threads = (TEAMS > 0 ? TEAMS : 1) * TT;
  static constexpr size_t smem_bytes = fixed_bytes + (size_t)(TEAMS > 0 ? TEAMS : 1) * team_doubles * 8;
  static constexpr bool supported = TEAMS >= 1;
};

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}
__device__ __forceinline__ void prefetch_l2(const void* p, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_async8(double* dst, const double* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
__device__ __forceinline__ void team_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

}  // namespace pmlmma

template <int DIM, int N>
__global__ void __launch_bounds__(pmlmma::Cfg<DIM, N>::Threads, 1) pml_mma_kernel(PmlArgs a) {
  using namespace pmlmma;
  using C = Cfg<DIM, N>;
  constexpr int Np = C::Np, Nfp = C::Nfp, Nfaces = C::Nfaces, NFN = C::NFN, Nf = C::Nf, NT = C::NT, NB = C::NB;
  constexpr int KS = C::KS, KFT = C::KFT, S = C::S, SG = C::SG, EG = C::EG, TW = C::TW, TT = C::TT;
  extern __shared__ double smem[];
  double* sAvol = smem;                              // [DIM][NB][KS][32] fragment order
  double* sAlift = sAvol + C::avol_doubles;          // [NB][KFT][32], faces packed along k
  double* slam = sAlift + C::alift_doubles;          // [NB*8][DIM+1]
  double* steam = slam + C::lam_doubles;             // [TEAMS][team_doubles]
  int* sfmask = reinterpret_cast<int*>(steam + C::TEAMS * C::team_doubles);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  for (int x = tid; x < C::avol_doubles; x += C::Threads) sAvol[x] = a.Avol[x];
  for (int x = tid; x < C::alift_doubles; x += C::Threads) sAlift[x] = a.AliftP[x];
  for (int x = tid; x < NB * 8; x += C::Threads) {
    const int n = x < Np ? x : Np - 1;
#pragma unroll
    for (int v = 0; v <= DIM; ++v) slam[x * (DIM + 1) + v] = a.lam[n * (DIM + 1) + v];
  }
  for (int x = tid; x < NFN; x += C::Threads) sfmask[x] = a.fmask[x];
  // zero the tiles once: their k-padding (j >= Np, m >= NFN) is never written and multiplies as 0
  for (int x = tid; x < C::TEAMS * C::team_doubles; x += C::Threads) steam[x] = 0.0;
  __syncthreads();

  const int team = warp / TW, h = warp - team * TW, tl = tid - team * TT;
  double* qt = steam + team * C::team_doubles;       // [EG*Nf][S]
  double* gt = qt + C::qtile_doubles;                // [DIM][EG*Nf][SG]
  const int g = lane >> 2, c = lane & 3;
  const int bcol = (g >> 1) * Nf + (g & 1);          // B-fragment column of this lane (element g/2, field 2t + g%2)
  const double cs = a.c, hc = 0.5 * a.c;
  const int64_t nquads = (a.Kpml + EG - 1) / EG;

  for (int64_t qd = (int64_t)blockIdx.x * C::TEAMS + team; qd < nquads; qd += (int64_t)gridDim.x * C::TEAMS) {
    const int64_t p0 = qd * EG;
    const int nel = (a.Kpml - p0) < EG ? (int)(a.Kpml - p0) : EG;
    team_sync(1 + team, TT);   // the previous quad's tiles are no longer read
    {   // pull the next quad of this team towards L2 while this one is processed: q rows and auxiliary rows
      const int64_t pn = (qd + (int64_t)gridDim.x * C::TEAMS) * EG;
      if (pn < a.Kpml) {
        const int nn_el = (a.Kpml - pn) < EG ? (int)(a.Kpml - pn) : EG;
        for (int x = tl; x < nn_el * (1 + DIM); x += TT) {
          const int el = x / (1 + DIM), w = x - el * (1 + DIM);
          const int64_t pp = pn + el;
          const uint32_t bytes = (uint32_t)(Nf * Np * 8);
          if (w == 0) {
            prefetch_l2(a.q_in + (int64_t)a.pml_elems[pp] * Nf * Np, bytes);
          } else {
            const int64_t off = (pp * DIM + (w - 1)) * Nf * Np;
            prefetch_l2(a.aux_in + off, bytes);
            if (a.aux_n && a.aux_n != a.aux_in) prefetch_l2(a.aux_n + off, bytes);
            if (a.acc_in) prefetch_l2(a.acc_in + off, bytes);
          }
        }
      }
    }
    // ---- element ids of the quad (one load per element, shared by everything below)
    int eid[EG];
#pragma unroll
    for (int el = 0; el < EG; ++el) eid[el] = a.pml_elems[p0 + (el < nel ? el : 0)];
    // ---- q tile of the quad's elements, rows (element, field), node stride S, asynchronously (rows of missing
    //      elements keep the previous quad's finite values; nothing of them is stored)
    for (int x = tl; x < nel * Nf * Np; x += TT) {
      const int row = x / Np, j = x - row * Np;
      const int el = row / Nf, k = row - el * Nf;
      int e = eid[0];
#pragma unroll
      for (int u = 1; u < EG; ++u) if (el == u) e = eid[u];
      cp_async8(qt + row * S + j, a.q_in + ((int64_t)e * Nf + k) * Np + j);
    }
    // ---- indices of my face nodes (boundary tag, exterior node), requested together before the tile is waited for
    constexpr int FR = (EG * NFN + TT - 1) / TT;
    int f_tag[FR], f_idP[FR], f_e[FR];
#pragma unroll
    for (int r = 0; r < FR; ++r) {
      const int x = tl + r * TT;
      f_tag[r] = 0; f_idP[r] = 0; f_e[r] = eid[0];
      if (x < nel * NFN) {
        const int fe = x / NFN, m = x - fe * NFN;
        int e = eid[0];
#pragma unroll
        for (int u = 1; u < EG; ++u) if (fe == u) e = eid[u];
        f_e[r] = e;
        if (a.EToB) f_tag[r] = a.EToB[(int64_t)e * Nfaces + m / Nfp];
        f_idP[r] = a.vmapP[(int64_t)e * NFN + m];
      }
    }
    cp_async_wait_all();
    team_sync(1 + team, TT);
    // ---- directional flux tiles: one gather of q+, one |A_n|[q], DIM directional pieces per face node
#pragma unroll
    for (int r = 0; r < FR; ++r) {
      const int x = tl + r * TT;
      if (x >= nel * NFN) continue;
      const int fe = x / NFN, m = x - fe * NFN;
      const int64_t ee = f_e[r];
      const int f = m / Nfp, n = sfmask[m];
      double qM[Nf], qP[Nf];
#pragma unroll
      for (int k = 0; k < Nf; ++k) qM[k] = qt[(fe * Nf + k) * S + n];
      const double* sg = a.sgeo + (ee * Nfaces + f) * (DIM + 2);
      double nh[DIM];
#pragma unroll
      for (int d = 0; d < DIM; ++d) nh[d] = sg[d];
      const double Fscale = sg[DIM + 1];
      const int tag = f_tag[r];
      if (tag == 0) {
        const int idP = f_idP[r];
        const int eP = idP / Np, nP = idP - eP * Np;
        const double* qp = a.q_in + (int64_t)eP * Nf * Np + nP;
#pragma unroll
        for (int k = 0; k < Nf; ++k) qP[k] = qp[k * Np];
      } else if (tag == 1) {   // wall moving with the mesh (reading R11)
        double vG[DIM];
        node_velocity<DIM>(slam + n * (DIM + 1), a.vvel + ee * (DIM + 1) * DIM, vG);
#pragma unroll
        for (int k = 0; k < Nf; ++k) qP[k] = qM[k];
#pragma unroll
        for (int d = 0; d < DIM; ++d) qP[1 + d] = 2.0 * qM[0] * vG[d] / cs - qM[1 + d];
      } else {                 // far field
#pragma unroll
        for (int k = 0; k < Nf; ++k) qP[k] = a.q_inf[k];
      }
      double dq[Nf], y1[Nf], absA[Nf];
#pragma unroll
      for (int k = 0; k < Nf; ++k) dq[k] = qP[k] - qM[k];
      abs_normal_apply<DIM>(nh, dq, y1, absA);
#pragma unroll
      for (int dd = 0; dd < DIM; ++dd) {
        double ad[Nf];
        hermite_apply<DIM>([&](int d, int j) { return d == dd ? dq[j] : 0.0; }, ad);
        const double nd = nh[dd];
#pragma unroll
        for (int k = 0; k < Nf; ++k)
          gt[dd * C::gtile_doubles + (fe * Nf + k) * SG + m] = Fscale * hc * (nd * nd * absA[k] - nd * ad[k]);
      }
    }
    team_sync(1 + team, TT);
    // ---- per 8-node block: D_a q (DMMA), then per direction the volume term, its LIFT contraction and the update
    //      The two warps of the team alternate over the blocks; an odd last block is shared by directions.
    for (int nb = 0; nb < NB; ++nb) {
      int dd_lo = 0, dd_hi = DIM;
      if ((NB & 1) && nb == NB - 1) {
        if (h == 0) dd_hi = DIM / 2; else dd_lo = DIM / 2;
      } else if ((nb & 1) != h) {
        continue;
      }
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
      const int n = 8 * nb + g;
      const int nn = n < Np ? n : Np - 1;
      const bool evalid = c < nel && n < Np;
      const int64_t p = p0 + (c < nel ? c : 0);
      int64_t e = eid[0];
#pragma unroll
      for (int u = 1; u < EG; ++u) if (c == u && c < nel) e = eid[u];
      double G[DIM * DIM];
      {
        const double* vg = a.vgeo + e * (DIM * DIM + 1);
#pragma unroll
        for (int x = 0; x < DIM * DIM; ++x) G[x] = vg[x];
      }
#pragma unroll
      for (int dd = 0; dd < DIM; ++dd) {
        if (dd < dd_lo || dd >= dd_hi) continue;
        // volume part -c A^_dd d_dd q on the accumulator registers
        double st[Nf], V[NT][2];
        hermite_apply<DIM>(
            [&](int d, int j) {
              if (d != dd) return 0.0;
              double s = 0.0;
#pragma unroll
              for (int r = 0; r < DIM; ++r) s = fma(G[r * DIM + dd], acc[r][j >> 1][j & 1], s);
              return s;   // d q_j / d x_dd
            },
            st);
#pragma unroll
        for (int k = 0; k < Nf; ++k) V[k >> 1][k & 1] = -cs * st[k];
        // RK inputs of this direction, requested before the LIFT contraction so that their latency hides behind it
        const double sig = evalid ? a.pml_sigma[p * DIM + dd] : 0.0;
        const int64_t base = ((p * DIM + dd) * Nf) * Np + nn;
        // (p and nn are clamped, so the addresses are valid for every lane: straight-line loads behind one uniform
        //  branch per array -- per-lane predicates made the compiler wait for each load before issuing the next,
        //  53 % of the kernel's stall samples, profiles/r1_pml_kernel.md)
        double xi[Nf], xn[Nf], xa[Nf];
        {
          const double* pi = a.aux_in + base;
#pragma unroll
          for (int k = 0; k < Nf; ++k) xi[k] = pi[k * Np];
        }
#pragma unroll
        for (int k = 0; k < Nf; ++k) { xn[k] = 0.0; xa[k] = 0.0; }
        if (a.aux_n != nullptr) {
          if (a.aux_n == a.aux_in) {
#pragma unroll
            for (int k = 0; k < Nf; ++k) xn[k] = xi[k];
          } else {
            const double* pn = a.aux_n + base;
#pragma unroll
            for (int k = 0; k < Nf; ++k) xn[k] = pn[k * Np];
          }
        }
        if (a.acc_in != nullptr) {
          const double* pa = a.acc_in + base;
#pragma unroll
          for (int k = 0; k < Nf; ++k) xa[k] = pa[k * Np];
        }
        // surface part: LIFT of the direction's flux tile, accumulated into the same registers
        const double* gd = gt + dd * C::gtile_doubles;
#pragma unroll
        for (int ks = 0; ks < KFT; ++ks) {
          double bf[NT];
#pragma unroll
          for (int t = 0; t < NT; ++t) bf[t] = gd[(bcol + 2 * t) * SG + 4 * ks + c];
          const double af = sAlift[(nb * KFT + ks) * 32 + lane];
#pragma unroll
          for (int t = 0; t < NT; ++t) dmma(V[t][0], V[t][1], af, bf[t]);
        }
        if (evalid) {
#pragma unroll
          for (int k = 0; k < Nf; ++k) {
            const int64_t idx = base + k * Np;
            const double gg = V[k >> 1][k & 1] - sig * xi[k];
            if (a.G_out) a.G_out[idx] = gg;
            if (a.aux_out) a.aux_out[idx] = fma(a.cx_g, gg, fma(a.cx_acc, xa[k], a.cx_n * xn[k]));
            if (a.acc_out) a.acc_out[idx] = fma(a.cy_g, gg, fma(a.cy_acc, xa[k], a.cy_n * xn[k]));
          }
        }
      }
    }
  }
}

// ------------------------------------------------------------------------------------------------------------------
template <int DIM, int N>
static cudaError_t launch_pml_mma_one(const PmlArgs& a, int num_sms, cudaStream_t s, bool configure_only) {
  using C = pmlmma::Cfg<DIM, N>;
  if constexpr (!C::supported) {
    return cudaErrorInvalidValue;
  } else {
    if (configure_only)
      return cudaFuncSetAttribute(pml_mma_kernel<DIM, N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem_bytes);
    const int64_t nquads = (a.Kpml + C::EG - 1) / C::EG;
    if (nquads == 0) return cudaSuccess;
    int64_t grid = (nquads + C::TEAMS - 1) / C::TEAMS;
    if (grid > num_sms) grid = num_sms;
    pml_mma_kernel<DIM, N><<<(int)grid, C::Threads, C::smem_bytes, s>>>(a);
    return cudaGetLastError();
  }
}

#define ALEGB_PMLMMA_DISPATCH(...)                                   \
  switch (dim * 10 + N) {                                            \
    case 21: return launch_pml_mma_one<2, 1>(__VA_ARGS__);           \
    case 22: return launch_pml_mma_one<2, 2>(__VA_ARGS__);           \
    case 23: return launch_pml_mma_one<2, 3>(__VA_ARGS__);           \
    case 24: return launch_pml_mma_one<2, 4>(__VA_ARGS__);           \
    case 25: return launch_pml_mma_one<2, 5>(__VA_ARGS__);           \
    case 31: return launch_pml_mma_one<3, 1>(__VA_ARGS__);           \
    case 32: return launch_pml_mma_one<3, 2>(__VA_ARGS__);           \
    case 33: return launch_pml_mma_one<3, 3>(__VA_ARGS__);           \
    case 34: return launch_pml_mma_one<3, 4>(__VA_ARGS__);           \
    default: return cudaErrorInvalidValue;                           \
  }

cudaError_t launch_pml_mma(int dim, int N, const PmlArgs& a, int num_sms, cudaStream_t s) {
  ALEGB_PMLMMA_DISPATCH(a, num_sms, s, false)
}
cudaError_t configure_pml_mma(int dim, int N) {
  PmlArgs a{};
  ALEGB_PMLMMA_DISPATCH(a, 0, nullptr, true)
}

}  // namespace alegb
