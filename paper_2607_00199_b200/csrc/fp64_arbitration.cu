// Microbenchmarks behind the design of the fused stage kernel (profiles/r1_fp64_arbitration.md):
//   --latency   DMMA (mma.sync.m8n8k4.f64) issue rate against independent accumulator chains per warp and warps per SM;
//   --mix       DMMA warps and DFMA warps sharing an SM sub-partition: how much of the fp64 datapath a DFMA warp
//               gets next to one or two DMMA warps (issue arbitration), against its instruction-level parallelism;
//   --contract  the stage kernel's two contraction loops in isolation (operands in shared memory, same layouts).
// Built by paper_2607_00199_b200/build.py into paper_2607_00199_b200/fp64_arbitration; not part of the library.
#include <cstdio>
#include <cstring>
#include <cuda_runtime.h>
__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// ---- --latency
template <int CH>
__global__ void k_latency(double* out, int iters, long long* cyc) {
  double c0[CH], c1[CH];
  for (int i = 0; i < CH; ++i) { c0[i] = threadIdx.x * 1e-9; c1[i] = i; }
  double a = 1.0 + threadIdx.x * 1e-12, b = 1.0 - threadIdx.x * 1e-12;
  long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < CH; ++i) dmma(c0[i], c1[i], a, b);
  }
  long long t1 = clock64();
  double s = 0; for (int i = 0; i < CH; ++i) s += c0[i] + c1[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
  if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}
template <int CH> void run_latency(int warps, double* d, long long* dc) {
  int iters = 4000;
  k_latency<CH><<<148, warps * 32>>>(d, iters, dc); cudaDeviceSynchronize();
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  cudaEventRecord(e0); k_latency<CH><<<148, warps * 32>>>(d, iters, dc); cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1);
  long long c; cudaMemcpy(&c, dc, 8, cudaMemcpyDeviceToHost);
  double flop = 148.0 * warps * iters * CH * 512.0;
  printf("chains %2d warps/SM %2d : %6.2f TFLOP/s, %.1f clk per DMMA per warp (=%.1f clk per chain step)\n", CH, warps, flop / ms / 1e9, (double)c / iters / CH, (double)c / iters);
}

// ---- --mix
// warps [0, nm) run DMMA (8 chains) for `iters`; warps [nm, nm+nf) run DFMA with CH chains until a flag says the DMMA warps are done
template <int CH>
__global__ void k_mix(double* out, int iters, int nm, long long* cyc, long long* nfma) {
  __shared__ volatile int done;
  if (threadIdx.x == 0) done = 0;
  __syncthreads();
  int warp = threadIdx.x >> 5;
  double a = 1.0 + threadIdx.x * 1e-12, b = 1.0 - threadIdx.x * 1e-12;
  if (warp < nm) {
    double c0[8], c1[8];
    for (int i = 0; i < 8; ++i) { c0[i] = threadIdx.x * 1e-9; c1[i] = i; }
    long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int i = 0; i < 8; ++i) dmma(c0[i], c1[i], a, b);
    }
    long long t1 = clock64();
    double s = 0; for (int i = 0; i < 8; ++i) s += c0[i] + c1[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) { done = 1; if (blockIdx.x == 0) *cyc = t1 - t0; }
  } else {
    double x[CH];
    for (int i = 0; i < CH; ++i) x[i] = i + threadIdx.x;
    long long n = 0;
    while (!done) {
#pragma unroll
      for (int r = 0; r < 8; ++r)
#pragma unroll
        for (int i = 0; i < CH; ++i) x[i] = fma(x[i], a, b);
      n += 8 * CH;
    }
    double s = 0; for (int i = 0; i < CH; ++i) s += x[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if ((threadIdx.x & 31) == 0 && warp == nm && blockIdx.x == 0) *nfma = n;
  }
}
template <int CH> void run_mix(int nm, int nf, double* d, long long* dc) {
  int iters = 4000;
  cudaMemset(dc, 0, 16);
  k_mix<CH><<<148, (nm + nf) * 32>>>(d, iters, nm, dc, dc + 1); cudaDeviceSynchronize();
  long long c[2]; cudaMemcpy(c, dc, 16, cudaMemcpyDeviceToHost);
  double clk_per_dmma_smsp = (double)c[0] / (iters * 8.0) / (nm / 4.0);   // pipe clocks per DMMA on one sub-partition
  double dfma_clk = nf ? (double)c[0] / (double)c[1] : 0;                 // clocks per DFMA of one DFMA warp
  double pipe = (16.0 * iters * 8.0 * (nm / 4.0) + 2.0 * c[1] * (nf / 4.0)) / c[0];
  printf("DMMA warps/SMSP %d, DFMA warps/SMSP %d chains %2d: %.1f clk per DMMA per SMSP (16 = peak), DFMA warp issues one per %.1f clk, pipe busy %.0f %%\n",
         nm / 4, nf / 4, CH, clk_per_dmma_smsp, dfma_clk, 100 * pipe);
}

// ---- --contract
constexpr int Nf=10,NT=5,NB=5,KS=9,KFT=15,S=36,SG=60,DIM=3;
template <int MODE>   // 0: vol+lift as in the kernel; 1: vol only; 2: lift only; 3: lift with two node blocks per pass; 4: vol + lift2
__global__ void k_contract(double* out, int iters) {
  extern __shared__ double sm[];
  double* sAvol = sm; double* sAlift = sAvol + DIM*NB*KS*32; double* qt = sAlift + NB*KFT*32; double* gt = qt + 40*S;
  for (int x = threadIdx.x; x < DIM*NB*KS*32 + NB*KFT*32 + 40*S + 40*SG; x += blockDim.x) sm[x] = 1e-3 * (x % 7);
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, g = lane >> 2, c = lane & 3;
  const int bcol = (g >> 1) * Nf + (g & 1);
  double tot = 0;
  for (int it = 0; it < iters; ++it) {
    const int nb = (warp + it) % NB, nb2 = (nb + 1) % NB;
    double acc[DIM][NT][2], V[NT][2], V2[NT][2];
    for (int d = 0; d < DIM; ++d) for (int t = 0; t < NT; ++t) acc[d][t][0] = acc[d][t][1] = 0;
    for (int t = 0; t < NT; ++t) V[t][0] = V[t][1] = V2[t][0] = V2[t][1] = 0;
    if (MODE == 0 || MODE == 1 || MODE == 4) {
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
      for (int t = 0; t < NT; ++t) { V[t][0] = acc[0][t][0] + acc[1][t][0] + acc[2][t][0]; V[t][1] = acc[0][t][1] + acc[1][t][1] + acc[2][t][1]; }
    }
    if (MODE == 0 || MODE == 2) {
#pragma unroll
      for (int ks = 0; ks < KFT; ++ks) {
        double bf[NT];
#pragma unroll
        for (int t = 0; t < NT; ++t) bf[t] = gt[(bcol + 2 * t) * SG + 4 * ks + c];
        const double af = sAlift[(nb * KFT + ks) * 32 + lane];
#pragma unroll
        for (int t = 0; t < NT; ++t) dmma(V[t][0], V[t][1], af, bf[t]);
      }
    }
    if (MODE == 3 || MODE == 4) {
#pragma unroll
      for (int ks = 0; ks < KFT; ++ks) {
        double bf[NT];
#pragma unroll
        for (int t = 0; t < NT; ++t) bf[t] = gt[(bcol + 2 * t) * SG + 4 * ks + c];
        const double af = sAlift[(nb * KFT + ks) * 32 + lane], af2 = sAlift[(nb2 * KFT + ks) * 32 + lane];
#pragma unroll
        for (int t = 0; t < NT; ++t) { dmma(V[t][0], V[t][1], af, bf[t]); dmma(V2[t][0], V2[t][1], af2, bf[t]); }
      }
    }
    for (int t = 0; t < NT; ++t) tot += V[t][0] + V[t][1] + V2[t][0] + V2[t][1];
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = tot;
}
template <int MODE> void run_contract(int warps, double* d, const char* name) {
  int iters = 2000; size_t smem = (DIM*NB*KS*32 + NB*KFT*32 + 40*S + 40*SG) * 8;
  cudaFuncSetAttribute(k_contract<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  k_contract<MODE><<<148, warps * 32, smem>>>(d, 10); cudaDeviceSynchronize();
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  cudaEventRecord(e0); k_contract<MODE><<<148, warps * 32, smem>>>(d, iters); cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1);
  int nd = (MODE == 0 ? 210 : MODE == 1 ? 135 : MODE == 2 ? 75 : MODE == 3 ? 150 : 285);
  double flop = 148.0 * warps * iters * nd * 512.0;
  printf("%-28s warps/SM %2d : %6.2f TFLOP/s (%.0f %% of 37.2)  err=%s\n", name, warps, flop / ms / 1e9, flop / ms / 1e9 / 37.2 * 100, cudaGetErrorString(cudaGetLastError()));
}

int main(int argc, char** argv) {
  const bool all = argc < 2;
  auto want = [&](const char* f) { if (all) return true; for (int i = 1; i < argc; ++i) if (!strcmp(argv[i], f)) return true; return false; };
  double* d; long long* dc; cudaMalloc(&d, 148 * 1024 * 8); cudaMalloc(&dc, 16);
  if (want("--latency"))
    for (int w : {4, 8, 12, 16}) { run_latency<1>(w, d, dc); run_latency<2>(w, d, dc); run_latency<4>(w, d, dc); run_latency<5>(w, d, dc); run_latency<8>(w, d, dc); run_latency<15>(w, d, dc); }
  if (want("--mix")) {
    run_mix<1>(4, 0, d, dc);
    for (int nm : {4, 8}) for (int nf : {4, 8}) { run_mix<1>(nm, nf, d, dc); run_mix<2>(nm, nf, d, dc); run_mix<4>(nm, nf, d, dc); run_mix<16>(nm, nf, d, dc); }
  }
  if (want("--contract"))
    for (int w : {4, 8, 12, 16}) { run_contract<0>(w, d, "vol+lift"); run_contract<1>(w, d, "vol only"); run_contract<2>(w, d, "lift only"); }
  return 0;
}
