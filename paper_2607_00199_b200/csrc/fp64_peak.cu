// Microbenchmark behind the "alu" roofline denominator: peak fp64 throughput of the SM's fp64 pipe with
// plain DFMA, with tensor-core DMMA (mma.sync.m8n8k4.f64), with both interleaved in one warp and with both split
// across warps -- the last two show that DFMA and DMMA share one pipe on sm_100a (no overlap).
// Built by paper_2607_00199_b200/build.py into paper_2607_00199_b200/fp64_peak; not part of the library.
#include <cstdio>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("ERR %s line %d\n",cudaGetErrorString(e),__LINE__);return 1;}}while(0)

__device__ __forceinline__ void dmma(double &c0,double &c1,double a,double b){
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};":"+d"(c0),"+d"(c1):"d"(a),"d"(b));
}
template<int MODE> // 0 dfma, 1 dmma, 2 both interleaved in-warp, 3 split by warp parity
__global__ void __launch_bounds__(256) k(double *out,int iters,double a,double b,long long *cyc){
  double f[16]; double c[16];
  #pragma unroll
  for(int i=0;i<16;i++){f[i]=threadIdx.x*1e-3+i; c[i]=i;}
  int warp=threadIdx.x>>5;
  long long t0=clock64();
  for(int it=0;it<iters;it++){
    if(MODE==0 || MODE==2 || (MODE==3 && (warp&1))){
      #pragma unroll
      for(int i=0;i<16;i++) f[i]=fma(f[i],a,b);
    }
    if(MODE==1 || MODE==2 || (MODE==3 && !(warp&1))){
      #pragma unroll
      for(int i=0;i<8;i++) dmma(c[2*i],c[2*i+1],a,b);
    }
  }
  long long t1=clock64();
  double s=0; 
  #pragma unroll
  for(int i=0;i<16;i++) s+=f[i]+c[i];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
  if(threadIdx.x==0&&blockIdx.x==0) *cyc=t1-t0;
}
template<int MODE> int run(const char*name,int bps){
  int nb=148*bps, iters=20000; double *out; long long *cyc; CK(cudaMalloc(&out,nb*256*8)); CK(cudaMalloc(&cyc,8));
  cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  k<MODE><<<nb,256>>>(out,1000,0.999,1e-9,cyc); CK(cudaDeviceSynchronize());
  cudaEventRecord(e0); k<MODE><<<nb,256>>>(out,iters,0.999,1e-9,cyc); cudaEventRecord(e1); CK(cudaDeviceSynchronize());
  float ms; cudaEventElapsedTime(&ms,e0,e1); long long hc; cudaMemcpy(&hc,cyc,8,cudaMemcpyDeviceToHost);
  double nwarps=(double)nb*8, fl_dfma=0, fl_dmma=0;
  if(MODE==0||MODE==2) fl_dfma=nwarps*32*16*2.0*iters; if(MODE==3) fl_dfma=nwarps/2*32*16*2.0*iters;
  if(MODE==1||MODE==2) fl_dmma=nwarps*8*512.0*iters; if(MODE==3) fl_dmma=nwarps/2*8*512.0*iters;
  printf("%-28s bps=%d ms=%.3f dfma=%.2f TF dmma=%.2f TF total=%.2f TF  clk=%.0f MHz\n",name,bps,ms,fl_dfma/ms*1e-9,fl_dmma/ms*1e-9,(fl_dfma+fl_dmma)/ms*1e-9, hc/(ms*1e3));
  cudaFree(out); cudaFree(cyc); return 0;
}
int main(){
  for(int bps=1;bps<=4;bps*=2){
    run<0>("dfma",bps); run<1>("dmma m8n8k4",bps); run<2>("both in-warp",bps); run<3>("split by warp",bps);
  }
  return 0;
}
