// Fused stage kernel, pipelined tensor-core version (DMMA, mma.sync.m8n8k4.f64) for sm_100a.
//
// Why this shape (profiles/r1_v2_mma_stage_kernel.md): on the 3-D configurations the stage is bound by the fp64
// datapath (380 flop per degree of freedom against 38 B), and the warp-per-4-elements DMMA kernel kept that datapath
// only ~50 % busy because each of its 8 warps serialised  tile load -> contraction -> neighbour gathers -> contraction
// -> update loads  with every global-memory latency exposed.  Here a persistent CTA is split into
//
//   producer warps  stream "quads" (4 consecutive elements) into a ring of shared-memory slots: the q tile
//                   (cp.async, padded rows), per-element metric data, per-face data, and the complete upwind flux
//                   tile of the quad (a5: trace gather through vmapP, boundary states, eq. 7) -- all global-memory
//                   latency of a3-a5 lives here, overlapped with the contractions of earlier quads;
//   consumer warps  take work items (quad, block of 8 nodes): D_r,D_s,D_t contraction on the tensor cores (a3),
//                   point-wise volume terms on the accumulator registers (a3, a4), LIFT contraction into the same
//                   registers (a5), SARK update and stores (a6).
//
// Slots are handed over with mbarriers (full: producers -> consumers, empty: consumers -> producers).
// DMMA operand layout as in stage_mma.cu: rows = nodes (blocks of 8), columns = (element 0..3) x (field pair
// member), so lane (g = lane/4, c = lane%4) of a consumer holds every field of node 8*nb+g of element c.
#include "alegb_internal.h"
#include "device_common.cuh"

namespace alegb {

namespace pipe {

__host__ __device__ constexpr int stride_pad(int x) {
  // smallest s >= x with s = 4 (mod 8): the B-fragment loads of a half-warp (4 rows x 4 consecutive doubles) then
  // fall on 16 distinct 8-byte banks
  int s = x;
  while (s % 8 != 4) ++s;
  return s;
}

// LAYER: the instantiation for meshes with an absorbing layer (a8 fused in, see the consumers): a slot carries DIM
// more flux tiles (the directional pieces of reading R12), so the ring is as deep as shared memory allows.
template <int DIM, int N, bool LAYER = false>
struct Cfg {
  static constexpr int Np = DIM == 2 ? (N + 1) * (N + 2) / 2 : (N + 1) * (N + 2) * (N + 3) / 6;
  static constexpr int Nfp = DIM == 2 ? N + 1 : (N + 1) * (N + 2) / 2;
  static constexpr int Nfaces = DIM + 1;
  static constexpr int NFN = Nfaces * Nfp;
  static constexpr int Nf = DIM == 2 ? 6 : 10;
  static constexpr int NT = Nf / 2;            // column tiles (field pairs)
  static constexpr int NB = (Np + 7) / 8;      // node blocks (row tiles) = work items per quad
  static constexpr int KS = (Np + 3) / 4;      // k-steps of the volume contraction
  static constexpr int KFT = (NFN + 3) / 4;    // k-steps of the surface contraction (all faces packed: m = f*Nfp + mm)
  static constexpr int S = stride_pad(4 * KS);     // node stride of a q-tile row
  static constexpr int SG = stride_pad(4 * KFT);   // face-node stride of a flux-tile row
  static constexpr int EG = 4;                 // elements per quad
  // warps: 3-D 4 + 8 (3 per SM sub-partition -> up to 168 registers); 2-D 6 + 10 (< 128 registers, so 4 per sub-partition fit)
  static constexpr int PW = DIM == 2 ? 6 : 4;  // producer warps
  static constexpr int CW = DIM == 2 ? 10 : 8; // consumer warps
  // Producer groups.  3-D: the four producer warps work on ONE quad together (a quad is 1400 doubles of q and 240
  // flux tasks at N=4) and the ring has 4 slots (a 5th costs more in L1 capacity than it gains).  2-D: a quad is a
  // few hundred doubles and 36 DMMA per item, the per-quad latency chain of the producers (indices -> copies ->
  // barrier -> flux) is what bounds the kernel (profiles/r1_v12_cfg3_stage_kernel.md), so every producer warp
  // streams quads of its own (warp w takes quads w, w+6, ...) into a 16-slot ring.  3-D N <= 3 sits in between:
  // two groups of two warps, ring of 8 (config 5: stage kernel 4.94 -> 4.56 ms).
  static constexpr int PG = DIM == 2 ? 32 : (N <= 3 && !LAYER ? 64 : PW * 32);   // threads of one producer group
  static constexpr int NS_want = PG == 32 ? 16 : (PG == 64 ? 8 : 4);   // slots in the ring, if they fit
  static constexpr int NG = PW * 32 / PG;      // producer groups
  static constexpr int NTILE = LAYER ? 1 + DIM : 1;   // flux tiles per slot: the full flux (+ one per direction)
  static constexpr int TAG0 = PG >= 64 ? 32 : EG;   // first thread of a group that fetches boundary tags
  static constexpr int Threads = (PW + CW) * 32;
  static constexpr int PT = PG;                // threads producing one quad
  static constexpr int NTASK = EG * NFN;       // flux tasks per quad
  static constexpr int ROUNDS = (NTASK + PT - 1) / PT;
  // per-element geometry records, copied raw from the geometry kernel's arrays
  static constexpr int VG = DIM * DIM + 1;         // vgeo: d xi_a / d x_d, J
  static constexpr int VV = (DIM + 1) * DIM;       // vvel: vertex velocities
  static constexpr int SGE = Nfaces * (DIM + 2);   // sgeo: per face unit normal, sJ, Fscale
  // slot layout, in doubles
  static constexpr int off_gt = EG * Nf * S;
  static constexpr int tile_doubles = EG * Nf * SG;
  static constexpr int off_vg = off_gt + NTILE * tile_doubles;
  static constexpr int off_vv = off_vg + EG * VG;
  static constexpr int off_sg = off_vv + EG * VV;
  static constexpr int off_int = off_sg + EG * SGE;          // ints: pml[EG], tag[EG*Nfaces]
  static constexpr int slot_doubles = off_int + (EG + EG * Nfaces + 1) / 2 + 1;
  static constexpr int avol_doubles = DIM * NB * KS * 32;
  static constexpr int alift_doubles = NB * KFT * 32;
  static constexpr int lam_doubles = NB * 8 * (DIM + 1);
  static constexpr size_t fixed_bytes = (size_t)(avol_doubles + alift_doubles + lam_doubles) * 8 + (size_t)NFN * 4 + 16;
  static constexpr int NS_fit = (int)((227 * 1024 - fixed_bytes) / ((size_t)slot_doubles * 8 + 16));
  static constexpr int NS = NS_want < NS_fit ? NS_want : NS_fit;
  static constexpr size_t smem_bytes = fixed_bytes + (size_t)NS * slot_doubles * 8 + 2 * (NS > 0 ? NS : 0) * 8;
  static constexpr bool supported = NS >= NG && NS >= (LAYER ? 3 : 2);
};

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("{\n\t.reg .b64 st;\n\tmbarrier.arrive.shared::cta.b64 st, [%0];\n\t}" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!done);
}
__device__ __forceinline__ void cp_async8(double* dst, const double* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NPENDING>
__device__ __forceinline__ void cp_async_wait_group() { asm volatile("cp.async.wait_group %0;" ::"n"(NPENDING) : "memory"); }
__device__ __forceinline__ void prefetch_l2(const void* p, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}
template <int NTHREADS>
__device__ __forceinline__ void producer_sync(int group) {   // the threads of one producer group
  if constexpr (NTHREADS == 32) __syncwarp();
  else if (group == 0) asm volatile("bar.sync 1, %0;" ::"n"(NTHREADS) : "memory");
  else asm volatile("bar.sync %0, %1;" ::"r"(1 + group), "n"(NTHREADS) : "memory");
}

}  // namespace pipe

template <int DIM, int N, bool LAYER>
__global__ void __launch_bounds__(pipe::Cfg<DIM, N, LAYER>::Threads, 1) stage_pipe_kernel(StageArgs a) {
  using namespace pipe;
  using C = Cfg<DIM, N, LAYER>;
  constexpr int Np = C::Np, Nfp = C::Nfp, Nfaces = C::Nfaces, NFN = C::NFN, Nf = C::Nf, NT = C::NT, NB = C::NB;
  constexpr int KS = C::KS, KFT = C::KFT, S = C::S, SG = C::SG, EG = C::EG, NS = C::NS, PT = C::PT;
  extern __shared__ double smem[];
  double* sAvol = smem;                              // [DIM][NB][KS][32] fragment order
  double* sAlift = sAvol + C::avol_doubles;          // [NB][KFT][32]
  double* slam = sAlift + C::alift_doubles;          // [NB*8][DIM+1], rows >= Np repeat the last node
  double* sslots = slam + C::lam_doubles;            // [NS][slot_doubles]
  uint64_t* full = reinterpret_cast<uint64_t*>(sslots + NS * C::slot_doubles);
  uint64_t* empty = full + NS;
  int* sfmask = reinterpret_cast<int*>(empty + NS);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  for (int x = tid; x < C::avol_doubles; x += C::Threads) sAvol[x] = a.Avol[x];
  for (int x = tid; x < C::alift_doubles; x += C::Threads) sAlift[x] = a.AliftP[x];
  for (int x = tid; x < NB * 8; x += C::Threads) {
    const int n = x < Np ? x : Np - 1;
#pragma unroll
    for (int v = 0; v <= DIM; ++v) slam[x * (DIM + 1) + v] = a.lam[n * (DIM + 1) + v];
  }
  for (int x = tid; x < NFN; x += C::Threads) sfmask[x] = a.fmask[x];
  // zero the slots once: the k-padding of both tiles (j >= Np, m >= NFN) is never written again and multiplies as 0
  for (int x = tid; x < NS * C::slot_doubles; x += C::Threads) sslots[x] = 0.0;
  if (tid == 0) {
    for (int s = 0; s < NS; ++s) {
      mbar_init(&full[s], PT);
      mbar_init(&empty[s], C::CW * 32);   // every consumer warp takes part in every hand-over (see the consumers)
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  const double cs = a.c;
  // the quads of this launch: all of the mesh, or a list (meshes with an absorbing layer run the plain instantiation
  // over the quads outside the layer and the LAYER instantiation over the quads that touch it)
  const int64_t nquads = a.quad_list != nullptr ? a.nquads_list : (a.K + EG - 1) / EG;
  auto quad_of = [&](int ql) -> int64_t {
    const int64_t idx = (int64_t)ql * gridDim.x + blockIdx.x;
    if (a.quad_list == nullptr) return idx;
    return idx < nquads ? (int64_t)__ldg(a.quad_list + idx) : 0;
  };
  const int nq_cta = (int)((nquads - blockIdx.x + gridDim.x - 1) / gridDim.x);   // quads blockIdx.x + ql*gridDim.x

  if (warp < C::PW) {
    // =================================================================================================== producers
    // Every global read of a quad is asynchronous (cp.async straight into its slot) and issued one quad ahead of
    // the flux arithmetic, so the producers never sit on a load: a group's iteration issues its next quad, then
    // computes the current one.
    const int pt = C::NG == 1 ? tid : tid % PT, grp = C::NG == 1 ? 0 : tid / PT;   // thread within its producer group, group
    constexpr int ROUNDS = C::ROUNDS;
    int task_fe[ROUNDS], task_m[ROUNDS];
#pragma unroll
    for (int r = 0; r < ROUNDS; ++r) {
      const int task = r * PT + pt;
      task_fe[r] = task / NFN;
      task_m[r] = task - task_fe[r] * NFN;
    }
    int idx_next[ROUNDS];   // vmapP entries of my face nodes in the quad that is issued next
    int meta_next = 0;      // pml index (threads < EG) / boundary tag (threads TAG0 .. TAG0+EG*Nfaces) of that quad

    auto load_indices = [&](int ql) {
      const int64_t e0 = quad_of(ql) * EG;
#pragma unroll
      for (int r = 0; r < ROUNDS; ++r) {
        const int64_t ee = e0 + task_fe[r];
        idx_next[r] = (ql < nq_cta && r * PT + pt < C::NTASK && ee < a.K) ? __ldg(a.vmapP + ee * NFN + task_m[r]) : -1;
      }
    };
    auto issue = [&](int ql) {
      const int64_t e0 = quad_of(ql) * EG;
      const int nel = (a.K - e0) < EG ? (int)(a.K - e0) : EG;
      const int slot = ql % NS, use = ql / NS;
      double* qt = sslots + slot * C::slot_doubles;
      if (use > 0) mbar_wait(&empty[slot], (use - 1) & 1);
      // q tile of the quad, rows (element, field), node stride S
      {
        const double* src = a.q_in + e0 * Nf * Np;
        const int total = nel * Nf * Np;
        for (int x = pt; x < total; x += PT) {
          const int row = x / Np, j = x - row * Np;
          cp_async8(qt + row * S + j, src + x);
        }
      }
      // exterior traces q+ of my face nodes, into the flux tile (the flux overwrites them in place)
#pragma unroll
      for (int r = 0; r < ROUNDS; ++r) {
        const int idP = idx_next[r];
        if (idP >= 0) {
          const int eP = idP / Np, nP = idP - eP * Np;
          const double* qp = a.q_in + (int64_t)eP * Nf * Np + nP;
          double* dst = qt + C::off_gt + task_fe[r] * Nf * SG + task_m[r];
#pragma unroll
          for (int k = 0; k < Nf; ++k) cp_async8(dst + k * SG, qp + k * Np);
        }
      }
      // geometric factors of the quad's elements, raw (a2's output; contiguous per quad)
      for (int x = pt; x < nel * C::VG; x += PT) cp_async8(qt + C::off_vg + x, a.vgeo + e0 * C::VG + x);
      for (int x = pt; x < nel * C::VV; x += PT) cp_async8(qt + C::off_vv + x, a.vvel + e0 * C::VV + x);
      for (int x = pt; x < nel * C::SGE; x += PT) cp_async8(qt + C::off_sg + x, a.sgeo + e0 * C::SGE + x);
      // integer records, through a register (stored one iteration later)
      meta_next = pt < EG ? -1 : 0;
      if (pt < EG) {
        if (pt < nel && a.pml_index != nullptr && a.aux != nullptr) meta_next = __ldg(a.pml_index + e0 + pt);
      } else if (pt >= C::TAG0 && pt < C::TAG0 + EG * Nfaces) {
        const int ef = pt - C::TAG0;
        if (ef < nel * Nfaces && a.EToB != nullptr) meta_next = a.EToB[e0 * Nfaces + ef];
      }
      // L2 prefetch of the a6 inputs the consumers will read for this quad
      if (pt == PT - 1) {
        const uint32_t bytes = (uint32_t)(nel * Nf * Np * 8);
        const int64_t off = e0 * Nf * Np;
        if (a.q_n != nullptr && a.q_n != a.q_in && (a.q_out || a.acc_out)) prefetch_l2(a.q_n + off, bytes);
        if (a.F0_in != nullptr) prefetch_l2(a.F0_in + off, bytes);
        if (a.acc_in != nullptr) prefetch_l2(a.acc_in + off, bytes);
      }
      load_indices(ql + C::NG);
    };

    load_indices(grp);
    if (grp < nq_cta) issue(grp);
    cp_async_commit();
    for (int ql = grp; ql < nq_cta; ql += C::NG) {
      const int64_t e0 = quad_of(ql) * EG;
      const int nel = (a.K - e0) < EG ? (int)(a.K - e0) : EG;
      const int slot = ql % NS;
      double* qt = sslots + slot * C::slot_doubles;
      double* gt = qt + C::off_gt;
      const double* svv = qt + C::off_vv;
      const double* ssg = qt + C::off_sg;
      int* si = reinterpret_cast<int*>(qt + C::off_int);
      const int meta_cur = meta_next;
      if (ql + C::NG < nq_cta) issue(ql + C::NG);
      cp_async_commit();
      if (pt < EG) si[pt] = meta_cur;
      else if (pt >= C::TAG0 && pt < C::TAG0 + EG * Nfaces) si[EG + pt - C::TAG0] = meta_cur;
      cp_async_wait_group<1>();   // everything of quad ql has landed (the group's next quad may still be in flight)
      producer_sync<PT>(grp);
      // ---- a5: upwind flux at my face nodes (eq. 7; reading R7), in place over the gathered q+
#pragma unroll
      for (int r = 0; r < ROUNDS; ++r) {
        const int fe = task_fe[r], m = task_m[r];
        if (r * PT + pt >= C::NTASK || fe >= nel) continue;
        const int f = m / Nfp;
        const int n = sfmask[m];
        double qM[Nf], qP[Nf];
#pragma unroll
        for (int k = 0; k < Nf; ++k) {
          qM[k] = qt[(fe * Nf + k) * S + n];
          qP[k] = gt[(fe * Nf + k) * SG + m];
        }
        const double* fd = ssg + (fe * Nfaces + f) * (DIM + 2);
        double nh[DIM], vG[DIM];
#pragma unroll
        for (int d = 0; d < DIM; ++d) nh[d] = fd[d];
        const double Fscale = fd[DIM + 1];
        node_velocity<DIM>(slam + n * (DIM + 1), svv + fe * C::VV, vG);   // P1 mesh velocity at the node (L152, L196)
        double vn = 0.0;
#pragma unroll
        for (int d = 0; d < DIM; ++d) vn = fma(vG[d], nh[d], vn);
        const int tag = si[EG + fe * Nfaces + f];
        if (tag == 1) {          // wall moving with the mesh (reading R11)
#pragma unroll
          for (int k = 0; k < Nf; ++k) qP[k] = qM[k];
#pragma unroll
          for (int d = 0; d < DIM; ++d) qP[1 + d] = 2.0 * qM[0] * vG[d] / cs - qM[1 + d];
        } else if (tag != 0) {   // far field
#pragma unroll
          for (int k = 0; k < Nf; ++k) qP[k] = a.q_inf[k];
        }
        double fl[Nf];
        upwind_flux<DIM>(qM, qP, nh, cs, vn, Fscale, fl);
#pragma unroll
        for (int k = 0; k < Nf; ++k) gt[(fe * Nf + k) * SG + m] = fl[k];
        if constexpr (LAYER) {
          // a8 (reading R12): the directional pieces Fscale ( -1/2 n_d c A^_d [q] + 1/2 n_d^2 |A_n| [q] ) of the quads
          // that touch the absorbing layer, one more flux tile per direction
          bool inlayer = false;
#pragma unroll
          for (int el = 0; el < EG; ++el) inlayer |= si[el] >= 0;
          if (inlayer) {
            if (r == 0 && pt < EG && si[pt] >= 0) {   // pull the element's auxiliary rows towards L2 for the consumers
              const int64_t off = (int64_t)si[pt] * DIM * Nf * Np;
              const uint32_t bytes = (uint32_t)(DIM * Nf * Np * 8);
              prefetch_l2(a.aux + off, bytes);
              if (a.layer.aux_n != nullptr && a.layer.aux_n != a.aux) prefetch_l2(a.layer.aux_n + off, bytes);
              if (a.layer.acc_in != nullptr) prefetch_l2(a.layer.acc_in + off, bytes);
            }
#pragma unroll
            for (int dd = 0; dd < DIM; ++dd) {
              double fd2[Nf];
              directional_flux<DIM>(dd, qM, qP, nh, cs, Fscale, fd2);
#pragma unroll
              for (int k = 0; k < Nf; ++k) gt[(1 + dd) * C::tile_doubles + (fe * Nf + k) * SG + m] = fd2[k];
            }
          }
        }
      }
      mbar_arrive(&full[slot]);
    }
  } else {
    // =================================================================================================== consumers
    const int cw = warp - C::PW;
    const int g = lane >> 2, c = lane & 3;
    // B-fragment column of this lane: column g  <->  element g/2, field 2t + (g&1); k index = c
    const int bcol = (g >> 1) * Nf + (g & 1);
    const bool qn_in_tile = a.q_n == a.q_in;
    const bool want_update = a.q_out != nullptr || a.acc_out != nullptr;
    const int nitems = nq_cta * NB;
    // mbarrier waits test a phase PARITY, so a waiter must never be two phases away from the barrier.  A warp has
    // an item only in some quads (items cw, cw + CW, ...; NB <= CW items per quad); were it to skip the others, it
    // could reach a slot whose previous use is not even full yet -- the parity test then passes and it reads stale
    // data -- or fall two uses behind and wait forever (seen as a hang with two producer groups and a ring of 4, and
    // reproduced for 3-D N = 1 in a scheduling simulation).  So every consumer warp takes part in the hand-over of
    // EVERY quad, in order: it waits for `full`, works if it has an item there, and arrives on `empty`.
    static_assert(NB <= C::CW, "at most one item per quad and consumer warp");
    int next_q = 0;   // first quad this warp has not yet taken part in
    auto pass_quads = [&](int upto) {
      for (; next_q < upto; ++next_q) {
        mbar_wait(&full[next_q % NS], (next_q / NS) & 1);
        mbar_arrive(&empty[next_q % NS]);
      }
    };
    for (int it = cw; it < nitems; it += C::CW) {
      const int ql = it / NB, nb = it - ql * NB;
      pass_quads(ql);
      next_q = ql + 1;
      const int64_t quad = quad_of(ql);
      const int64_t e0 = quad * EG;
      const int nel = (a.K - e0) < EG ? (int)(a.K - e0) : EG;
      const int slot = ql % NS, use = ql / NS;
      const double* qt = sslots + slot * C::slot_doubles;
      const double* gt = qt + C::off_gt;
      const double* svg = qt + C::off_vg + c * C::VG;
      const double* svv = qt + C::off_vv + c * C::VV;
      const int* si = reinterpret_cast<const int*>(qt + C::off_int);
      mbar_wait(&full[slot], use & 1);

      // ---- a3: reference derivatives D_a q of all fields at nodes 8nb..8nb+7 of the 4 elements (L103, L195)
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
      // ---- point-wise volume terms at node n of element c (eq. 9 first term, L107; a4 relaxation L115)
      const int n = 8 * nb + g;
      const int nn = n < Np ? n : Np - 1;
      double V[NT][2];
      {
        double G[DIM * DIM], w[DIM], vG[DIM];
#pragma unroll
        for (int x = 0; x < DIM * DIM; ++x) G[x] = svg[x];
        node_velocity<DIM>(slam + n * (DIM + 1), svv, vG);   // P1 mesh velocity at the node (L152, L192)
#pragma unroll
        for (int r = 0; r < DIM; ++r) {
          double s = 0.0;
#pragma unroll
          for (int d = 0; d < DIM; ++d) s = fma(vG[d], G[r * DIM + d], s);
          w[r] = s;   // w_r = v_G . grad(xi_r)
        }
        double st[Nf], qn[Nf], nt[Nf];
        hermite_apply<DIM>(
            [&](int d, int j) {
              double s = 0.0;
#pragma unroll
              for (int r = 0; r < DIM; ++r) s = fma(G[r * DIM + d], acc[r][j >> 1][j & 1], s);
              return s;   // d q_j / d x_d
            },
            st);
#pragma unroll
        for (int k = 0; k < Nf; ++k) qn[k] = qt[(c * Nf + k) * S + nn];
        relaxation_term<DIM>(a, qn, e0 + (c < nel ? c : 0), nn, Np, nt);
#pragma unroll
        for (int k = 0; k < Nf; ++k) {
          double v = fma(-cs, st[k], nt[k]);
#pragma unroll
          for (int r = 0; r < DIM; ++r) v = fma(w[r], acc[r][k >> 1][k & 1], v);
          V[k >> 1][k & 1] = v;
        }
      }
      const bool evalid = c < nel && n < Np;
      const int64_t e = e0 + (c < nel ? c : 0);
      const int64_t base = e * Nf * Np + nn;
      const int pml = si[c];
      if (pml >= 0) {   // absorbing layer (reading R12): - sum_d sigma_d q~^d
#pragma unroll
        for (int d = 0; d < DIM; ++d) {
          const double sig = a.pml_sigma[(int64_t)pml * DIM + d];
#pragma unroll
          for (int k = 0; k < Nf; ++k)
            V[k >> 1][k & 1] -= sig * a.aux[(((int64_t)pml * DIM + d) * Nf + k) * Np + nn];
        }
      }
      // ---- a6 inputs, requested before the LIFT contraction so that their latency hides behind it (one uniform
      //      branch per array, straight-line loads with immediate offsets inside)
      double uq[Nf], uf[Nf], ua[Nf];
#pragma unroll
      for (int k = 0; k < Nf; ++k) { uq[k] = 0.0; uf[k] = 0.0; ua[k] = 0.0; }
      if (evalid && want_update) {
        if (qn_in_tile) {
#pragma unroll
          for (int k = 0; k < Nf; ++k) uq[k] = qt[(c * Nf + k) * S + nn];
        } else if (a.q_n != nullptr) {
          const double* pq = a.q_n + base;
#pragma unroll
          for (int k = 0; k < Nf; ++k) uq[k] = __ldg(pq + k * Np);
        }
        if (a.F0_in != nullptr) {
          const double* pf = a.F0_in + base;
#pragma unroll
          for (int k = 0; k < Nf; ++k) uf[k] = __ldg(pf + k * Np);
        }
        if (a.acc_in != nullptr) {
          const double* pa = a.acc_in + base;
#pragma unroll
          for (int k = 0; k < Nf; ++k) ua[k] = __ldg(pa + k * Np);
        }
      }
      // ---- a5: LIFT contraction of the quad's flux tile into the same registers (L103, L196)
#pragma unroll
      for (int ks = 0; ks < KFT; ++ks) {
        double bf[NT];
#pragma unroll
        for (int t = 0; t < NT; ++t) bf[t] = gt[(bcol + 2 * t) * SG + 4 * ks + c];
        const double af = sAlift[(nb * KFT + ks) * 32 + lane];
#pragma unroll
        for (int t = 0; t < NT; ++t) dmma(V[t][0], V[t][1], af, bf[t]);
      }
      // all reads of the slot are done (quads in the absorbing layer: after their directional contractions below)
      bool inlayer = false;
      if constexpr (LAYER) {
        if (a.layer.on) {
#pragma unroll
          for (int el = 0; el < EG; ++el) inlayer |= si[el] >= 0;
        }
      }
      if (!inlayer) mbar_arrive(&empty[slot]);
      // ---- a6: SARK stage update (L132-134), straight from the accumulator registers; one uniform branch per output
      if (evalid) {
        if (a.F_out != nullptr) {
          double* of = a.F_out + base;
#pragma unroll
          for (int k = 0; k < Nf; ++k) of[k * Np] = V[k >> 1][k & 1];
        }
        // the coefficients depend on the field only through stiff / non-stiff (StageCoef): two values each
        const bool hf = a.F0_in != nullptr, ha = a.acc_in != nullptr;
        auto combine = [&](const double* cn, const double* cf0, double cacc, const double* cf, double* out) {
          const double n0 = cn[0], n1 = cn[DIM + 1], f00 = cf0[0], f01 = cf0[DIM + 1], g0 = cf[0], g1 = cf[DIM + 1];
          if (hf && ha) {
#pragma unroll
            for (int k = 0; k < Nf; ++k)
              out[k * Np] = fma(k > DIM ? g1 : g0, V[k >> 1][k & 1],
                                fma(cacc, ua[k], fma(k > DIM ? f01 : f00, uf[k], (k > DIM ? n1 : n0) * uq[k])));
          } else if (hf) {
#pragma unroll
            for (int k = 0; k < Nf; ++k)
              out[k * Np] = fma(k > DIM ? g1 : g0, V[k >> 1][k & 1], fma(k > DIM ? f01 : f00, uf[k], (k > DIM ? n1 : n0) * uq[k]));
          } else if (ha) {
#pragma unroll
            for (int k = 0; k < Nf; ++k)
              out[k * Np] = fma(k > DIM ? g1 : g0, V[k >> 1][k & 1], fma(cacc, ua[k], (k > DIM ? n1 : n0) * uq[k]));
          } else {
#pragma unroll
            for (int k = 0; k < Nf; ++k) out[k * Np] = fma(k > DIM ? g1 : g0, V[k >> 1][k & 1], (k > DIM ? n1 : n0) * uq[k]);
          }
        };
        if (a.q_out != nullptr) combine(a.coef.cq_n, a.coef.cq_f0, a.coef.cq_acc, a.coef.cq_f, a.q_out + base);
        if (a.acc_out != nullptr) combine(a.coef.ca_n, a.coef.ca_f0, a.coef.ca_acc, a.coef.ca_f, a.acc_out + base);
      }
      if constexpr (LAYER) {
        if (inlayer) {
          // ---- a8, fused: auxiliary fields of the absorbing layer (reading R12) for the layer elements of this quad,
          //   d/dt q~^d = -c A^_d d_d q + LIFT( directional flux tile d ) - sigma_d q~^d,   classic RK4 weights.
          // D_a q is still in the accumulator registers and the exterior traces were gathered once for all tiles;
          // the separate kernel (pml_mma.cu) re-read the q tile, re-gathered q+ and repeated the D_a contraction.
          const int64_t p = pml >= 0 ? pml : 0;          // clamped: valid addresses in every lane, stores predicated
          const bool pvalid = evalid && pml >= 0;
          double Vd[DIM][NT][2];
          {   // volume parts -c A^_dd d_dd q of all directions on the accumulator registers (D_a q is dead afterwards)
            double Gm[DIM * DIM];
#pragma unroll
            for (int x = 0; x < DIM * DIM; ++x) Gm[x] = svg[x];
#pragma unroll
            for (int dd = 0; dd < DIM; ++dd) {
              double st[Nf];
              hermite_apply<DIM>(
                  [&](int d, int j) {
                    if (d != dd) return 0.0;
                    double s = 0.0;
#pragma unroll
                    for (int r = 0; r < DIM; ++r) s = fma(Gm[r * DIM + dd], acc[r][j >> 1][j & 1], s);
                    return s;   // d q_j / d x_dd
                  },
                  st);
#pragma unroll
              for (int k = 0; k < Nf; ++k) Vd[dd][k >> 1][k & 1] = -cs * st[k];
            }
          }
          // surface parts: LIFT of the directional flux tiles, all directions back to back, then the slot is free
#pragma unroll
          for (int dd = 0; dd < DIM; ++dd) {
            const double* gd = gt + (1 + dd) * C::tile_doubles;
#pragma unroll
            for (int ks = 0; ks < KFT; ++ks) {
              double bf[NT];
#pragma unroll
              for (int t = 0; t < NT; ++t) bf[t] = gd[(bcol + 2 * t) * SG + 4 * ks + c];
              const double af = sAlift[(nb * KFT + ks) * 32 + lane];
#pragma unroll
              for (int t = 0; t < NT; ++t) dmma(Vd[dd][t][0], Vd[dd][t][1], af, bf[t]);
            }
          }
          mbar_arrive(&empty[slot]);
          // RK combination of the auxiliary state, direction by direction (straight-line loads behind uniform branches)
#pragma unroll
          for (int dd = 0; dd < DIM; ++dd) {
            const double sig = a.pml_sigma[p * DIM + dd];
            const int64_t pb = ((p * DIM + dd) * Nf) * Np + nn;
            double xi[Nf], xn[Nf], xa[Nf];
            {
              const double* pi = a.aux + pb;
#pragma unroll
              for (int k = 0; k < Nf; ++k) xi[k] = pi[k * Np];
            }
#pragma unroll
            for (int k = 0; k < Nf; ++k) { xn[k] = 0.0; xa[k] = 0.0; }
            if (a.layer.aux_n != nullptr) {
              if (a.layer.aux_n == a.aux) {
#pragma unroll
                for (int k = 0; k < Nf; ++k) xn[k] = xi[k];
              } else {
                const double* pn = a.layer.aux_n + pb;
#pragma unroll
                for (int k = 0; k < Nf; ++k) xn[k] = pn[k * Np];
              }
            }
            if (a.layer.acc_in != nullptr) {
              const double* pa = a.layer.acc_in + pb;
#pragma unroll
              for (int k = 0; k < Nf; ++k) xa[k] = pa[k * Np];
            }
            if (pvalid) {
#pragma unroll
              for (int k = 0; k < Nf; ++k) {
                const int64_t idx = pb + k * Np;
                const double gg = Vd[dd][k >> 1][k & 1] - sig * xi[k];
                if (a.layer.G_out) a.layer.G_out[idx] = gg;
                if (a.layer.aux_out) a.layer.aux_out[idx] = fma(a.layer.cx_g, gg, fma(a.layer.cx_acc, xa[k], a.layer.cx_n * xn[k]));
                if (a.layer.acc_out) a.layer.acc_out[idx] = fma(a.layer.cy_g, gg, fma(a.layer.cy_acc, xa[k], a.layer.cy_n * xn[k]));
              }
            }
          }
        }
      }
    }
    pass_quads(nq_cta);
  }
}

// ------------------------------------------------------------------------------------------------------------------
template <int DIM, int N, bool LAYER>
static cudaError_t launch_pipe_inst(const StageArgs& a, int num_sms, cudaStream_t s, bool configure_only) {
  using C = pipe::Cfg<DIM, N, LAYER>;
  if constexpr (!C::supported) {
    return cudaErrorInvalidValue;
  } else {
    if (configure_only)
      return cudaFuncSetAttribute(stage_pipe_kernel<DIM, N, LAYER>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem_bytes);
    const int64_t nquads = a.quad_list != nullptr ? a.nquads_list : (a.K + C::EG - 1) / C::EG;
    if (nquads == 0) return cudaSuccess;
    int64_t grid = nquads < num_sms ? nquads : num_sms;
    stage_pipe_kernel<DIM, N, LAYER><<<(int)grid, C::Threads, C::smem_bytes, s>>>(a);
    return cudaGetLastError();
  }
}
// a.layer.on selects the instantiation with the absorbing layer fused in (configure: both, the plain one decides)
template <int DIM, int N>
static cudaError_t launch_pipe_one(const StageArgs& a, int num_sms, cudaStream_t s, bool configure_only) {
  if (configure_only) {
    cudaError_t e = launch_pipe_inst<DIM, N, false>(a, num_sms, s, true);
    if (e == cudaSuccess && pipe::Cfg<DIM, N, true>::supported) e = launch_pipe_inst<DIM, N, true>(a, num_sms, s, true);
    return e;
  }
  if (a.layer.on) return launch_pipe_inst<DIM, N, true>(a, num_sms, s, false);
  return launch_pipe_inst<DIM, N, false>(a, num_sms, s, false);
}

#define ALEGB_PIPE_DISPATCH(...)                                  \
  switch (dim * 10 + N) {                                         \
    case 21: return launch_pipe_one<2, 1>(__VA_ARGS__);           \
    case 22: return launch_pipe_one<2, 2>(__VA_ARGS__);           \
    case 23: return launch_pipe_one<2, 3>(__VA_ARGS__);           \
    case 24: return launch_pipe_one<2, 4>(__VA_ARGS__);           \
    case 25: return launch_pipe_one<2, 5>(__VA_ARGS__);           \
    case 31: return launch_pipe_one<3, 1>(__VA_ARGS__);           \
    case 32: return launch_pipe_one<3, 2>(__VA_ARGS__);           \
    case 33: return launch_pipe_one<3, 3>(__VA_ARGS__);           \
    case 34: return launch_pipe_one<3, 4>(__VA_ARGS__);           \
    default: return cudaErrorInvalidValue;                        \
  }

cudaError_t launch_stage_pipe(int dim, int N, const StageArgs& a, int num_sms, cudaStream_t s) {
  ALEGB_PIPE_DISPATCH(a, num_sms, s, false)
}
cudaError_t configure_stage_pipe(int dim, int N) {
  StageArgs a{};
  ALEGB_PIPE_DISPATCH(a, 0, nullptr, true)
}
bool stage_pipe_layer_supported(int dim, int N) {
  switch (dim * 10 + N) {
    case 21: return pipe::Cfg<2, 1, true>::supported;
    case 22: return pipe::Cfg<2, 2, true>::supported;
    case 23: return pipe::Cfg<2, 3, true>::supported;
    case 24: return pipe::Cfg<2, 4, true>::supported;
    case 25: return pipe::Cfg<2, 5, true>::supported;
    case 31: return pipe::Cfg<3, 1, true>::supported;
    case 32: return pipe::Cfg<3, 2, true>::supported;
    case 33: return pipe::Cfg<3, 3, true>::supported;
    case 34: return pipe::Cfg<3, 4, true>::supported;
    default: return false;
  }
}

// The hand-over parameters of Cfg<DIM,N>, for tests/test_pipe_protocol.py (alegb_pipe_config): the simulation must
// model the kernel that is compiled, not a re-typed copy of its constants.
template <int DIM, int N, bool LAYER>
static bool pipe_config_one(PipeConfig& c) {
  using C = pipe::Cfg<DIM, N, LAYER>;
  if (!C::supported) return false;
  c.producer_groups = C::NG; c.slots = C::NS; c.items_per_quad = C::NB; c.consumer_warps = C::CW;
  c.warps_per_group = C::PG / 32; c.producer_warps = C::PW; c.elements_per_quad = C::EG; c.smem_bytes = (int)C::smem_bytes;
  return true;
}
template <bool LAYER>
static bool pipe_config_any(int dim, int N, PipeConfig& c) {
  switch (dim * 10 + N) {
    case 21: return pipe_config_one<2, 1, LAYER>(c);
    case 22: return pipe_config_one<2, 2, LAYER>(c);
    case 23: return pipe_config_one<2, 3, LAYER>(c);
    case 24: return pipe_config_one<2, 4, LAYER>(c);
    case 25: return pipe_config_one<2, 5, LAYER>(c);
    case 31: return pipe_config_one<3, 1, LAYER>(c);
    case 32: return pipe_config_one<3, 2, LAYER>(c);
    case 33: return pipe_config_one<3, 3, LAYER>(c);
    case 34: return pipe_config_one<3, 4, LAYER>(c);
    default: return false;
  }
}
bool stage_pipe_config(int dim, int N, PipeConfig& c, bool layer) {
  return layer ? pipe_config_any<true>(dim, N, c) : pipe_config_any<false>(dim, N, c);
}

}  // namespace alegb
