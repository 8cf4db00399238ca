// Measured fp64 ceiling of the device, for the roofline bench.py reports (alegb_measure_fp64_peak).
//
// MEASURED_PEAKS.json holds no fp64 figure and tcgen05 has no fp64 kind, so the stage kernels' binding roof -- the
// fp64 datapath reached through DMMA (mma.sync.m8n8k4.f64) and DFMA -- was so far DERIVED from unit counts and the
// clock (148 SM x 64 FMA/clk x 2 x 1.965 GHz = 37.2 TFLOP/s).  These two kernels measure it on the device the
// context runs on, at the clocks it runs at: register-resident chains with nothing else in the loop, 8 independent
// accumulator sets per warp / thread so that the pipe latency is covered, every SM filled with 16 warps.
// Not part of the hot path (measurement).
#include "alegb_internal.h"

namespace alegb {

namespace {

constexpr int kChains = 8;        // independent accumulators per thread
constexpr int kInner = 64;        // unrolled chain length per outer iteration
static __device__ double g_peak_sink[32];

__global__ void __launch_bounds__(512) dmma_peak_kernel(int outer, double seed) {
  double c0[kChains], c1[kChains];
  const double a = seed + 1e-9 * threadIdx.x, b = 1.0 - 1e-9 * threadIdx.x;
#pragma unroll
  for (int i = 0; i < kChains; ++i) { c0[i] = i; c1[i] = -i; }
  for (int o = 0; o < outer; ++o) {
#pragma unroll
    for (int k = 0; k < kInner / kChains; ++k) {
#pragma unroll
      for (int i = 0; i < kChains; ++i)
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                     : "+d"(c0[i]), "+d"(c1[i])
                     : "d"(a), "d"(b));
    }
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < kChains; ++i) s += c0[i] + c1[i];
  if (s == 0.123456789) g_peak_sink[threadIdx.x & 31] = s;   // never true: keeps the chains alive
}

__global__ void __launch_bounds__(512) dfma_peak_kernel(int outer, double seed) {
  double c[kChains];
  const double a = seed + 1e-9 * threadIdx.x, b = 1e-9 * threadIdx.x;
#pragma unroll
  for (int i = 0; i < kChains; ++i) c[i] = i;
  for (int o = 0; o < outer; ++o) {
#pragma unroll
    for (int k = 0; k < kInner / kChains; ++k) {
#pragma unroll
      for (int i = 0; i < kChains; ++i) c[i] = fma(c[i], a, b);
    }
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < kChains; ++i) s += c[i];
  if (s == 0.123456789) g_peak_sink[threadIdx.x & 31] = s;
}

}  // namespace

// TFLOP/s of each kind on the current device: best of `reps` timed launches after one warm-up, CUDA events on `s`.
cudaError_t measure_fp64_peak(int num_sms, int reps, double* dmma_tflops, double* dfma_tflops, cudaStream_t s) {
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  cudaError_t e = cudaEventCreate(&e0);
  if (e != cudaSuccess) return e;
  e = cudaEventCreate(&e1);
  if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
  const int blocks = num_sms, threads = 512, outer = 4096;
  const double warps = (double)blocks * threads / 32.0, lanes = (double)blocks * threads;
  // one DMMA = an 8x8x4 product per warp = 512 flop; one DFMA = 2 flop per lane
  const double flop_dmma = warps * (double)outer * kInner * 512.0, flop_dfma = lanes * (double)outer * kInner * 2.0;
  double best[2] = {0.0, 0.0};
  for (int kind = 0; kind < 2 && e == cudaSuccess; ++kind) {
    for (int r = 0; r <= reps && e == cudaSuccess; ++r) {
      cudaEventRecord(e0, s);
      if (kind == 0) dmma_peak_kernel<<<blocks, threads, 0, s>>>(outer, 0.999);
      else dfma_peak_kernel<<<blocks, threads, 0, s>>>(outer, 0.999);
      cudaEventRecord(e1, s);
      e = cudaEventSynchronize(e1);
      if (e != cudaSuccess) break;
      e = cudaGetLastError();
      float ms = 0.f;
      if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
      if (e == cudaSuccess && r > 0 && ms > 0.f) {
        const double tf = (kind == 0 ? flop_dmma : flop_dfma) / (ms * 1e-3) / 1e12;
        if (tf > best[kind]) best[kind] = tf;
      }
    }
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  if (e != cudaSuccess) return e;
  *dmma_tflops = best[0];
  *dfma_tflops = best[1];
  return cudaSuccess;
}

}  // namespace alegb
