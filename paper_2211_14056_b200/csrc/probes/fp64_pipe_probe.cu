// fp64_pipe_probe.cu — stand-alone measurement (not part of libmadme.so): DFMA peak and latency, DMMA m8n8k4 peak and
// latency, and DFMA + DMMA issued concurrently, on every SM.  BASELINE.json:north_star makes FP64 tensor cores
// conditional on a measurement; profiles/r2_probes.md records the result (they share one pipe on B200).
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o fp64_pipe_probe fp64_pipe_probe.cu && ./fp64_pipe_probe
#include <cstdio>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("err %s line %d\n", cudaGetErrorString(e), __LINE__); return 1;}}while(0)

template<int CH> __global__ void dfma_k(double* out, int iters, double a, double b){
  double acc[CH];
  for(int i=0;i<CH;++i) acc[i]=threadIdx.x*1e-3+i;
  for(int it=0; it<iters; ++it){
#pragma unroll
    for(int i=0;i<CH;++i) acc[i]=fma(acc[i],a,b);
  }
  double s=0; for(int i=0;i<CH;++i) s+=acc[i];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
__device__ __forceinline__ void dmma(double& d0,double& d1,double a,double b){
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};":"+d"(d0),"+d"(d1):"d"(a),"d"(b));
}
template<int CH> __global__ void dmma_k(double* out, int iters, double a, double b){
  double c0[CH],c1[CH];
  for(int i=0;i<CH;++i){c0[i]=threadIdx.x*1e-3+i;c1[i]=i;}
  for(int it=0; it<iters; ++it){
#pragma unroll
    for(int i=0;i<CH;++i) dmma(c0[i],c1[i],a,b);
  }
  double s=0; for(int i=0;i<CH;++i) s+=c0[i]+c1[i];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
// warps < nmma do DMMA (CH chains), the rest DFMA (CH chains); iterations tuned separately
template<int CH> __global__ void mix_k(double* out, int it_mma, int it_fma, int nmma, double a, double b){
  int w=threadIdx.x>>5;
  double s=0;
  if(w<nmma){
    double c0[CH],c1[CH];
    for(int i=0;i<CH;++i){c0[i]=threadIdx.x*1e-3+i;c1[i]=i;}
    for(int it=0; it<it_mma; ++it){
#pragma unroll
      for(int i=0;i<CH;++i) dmma(c0[i],c1[i],a,b);
    }
    for(int i=0;i<CH;++i) s+=c0[i]+c1[i];
  } else {
    double acc[CH];
    for(int i=0;i<CH;++i) acc[i]=threadIdx.x*1e-3+i;
    for(int it=0; it<it_fma; ++it){
#pragma unroll
      for(int i=0;i<CH;++i) acc[i]=fma(acc[i],a,b);
    }
    for(int i=0;i<CH;++i) s+=acc[i];
  }
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
// same warp interleaves 1 DMMA + R DFMA
template<int R> __global__ void inter_k(double* out, int iters, double a, double b){
  double c0[4],c1[4],acc[4*R];
  for(int i=0;i<4;++i){c0[i]=threadIdx.x*1e-3+i;c1[i]=i;}
  for(int i=0;i<4*R;++i) acc[i]=threadIdx.x*1e-3+i;
  for(int it=0; it<iters; ++it){
#pragma unroll
    for(int i=0;i<4;++i){ dmma(c0[i],c1[i],a,b);
#pragma unroll
      for(int r=0;r<R;++r) acc[i*R+r]=fma(acc[i*R+r],a,b);
    }
  }
  double s=0; for(int i=0;i<4;++i) s+=c0[i]+c1[i]; for(int i=0;i<4*R;++i) s+=acc[i];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
}
int main(){
  cudaDeviceProp p; CK(cudaGetDeviceProperties(&p,0));
  int sms=p.multiProcessorCount; int clk; cudaDeviceGetAttribute(&clk,cudaDevAttrClockRate,0);
  printf("%s SMs %d clock %d kHz\n",p.name,sms,clk);
  double* out; CK(cudaMalloc(&out,sizeof(double)*sms*1024*4));
  cudaEvent_t e0,e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  float ms; double ghz=clk*1e-6;
  auto rep=[&](const char* name,double flops,float ms,int){ printf("%-46s %8.3f ms  %7.2f TFLOP/s  %6.2f flop/clk/SM (of 128)\n",name,ms,flops/ms*1e-9,flops/(ms*1e-3)/(sms*ghz*1e9)); };
#define RUN(label, flops, ...) { __VA_ARGS__; CK(cudaDeviceSynchronize()); cudaEventRecord(e0); __VA_ARGS__; cudaEventRecord(e1); CK(cudaEventSynchronize(e1)); cudaEventElapsedTime(&ms,e0,e1); rep(label,flops,ms,0);} 
  int it=1<<16;
  // DFMA peak vs warps/SM and chains
  for(int wps: {4,8,16,32}){
    char l[96]; int thr=wps*32>1024?1024:wps*32; int bl=sms*((wps*32+thr-1)/thr);
    snprintf(l,96,"DFMA 8 chains, %d warps/SM",wps); RUN(l, 2.0*8*it*(double)bl*thr, (dfma_k<8><<<bl,thr>>>(out,it,1.0000001,1e-9)));
    snprintf(l,96,"DFMA 4 chains, %d warps/SM",wps); RUN(l, 2.0*4*it*(double)bl*thr, (dfma_k<4><<<bl,thr>>>(out,it,1.0000001,1e-9)));
    snprintf(l,96,"DFMA 2 chains, %d warps/SM",wps); RUN(l, 2.0*2*it*(double)bl*thr, (dfma_k<2><<<bl,thr>>>(out,it,1.0000001,1e-9)));
    snprintf(l,96,"DFMA 1 chain, %d warps/SM",wps); RUN(l, 2.0*1*it*(double)bl*thr, (dfma_k<1><<<bl,thr>>>(out,it,1.0000001,1e-9)));
  }
  // latency: 1 warp per SM, 1 chain
  { RUN("DFMA latency: 1 warp/SM 1 chain", 2.0*it*(double)sms*32, (dfma_k<1><<<sms,32>>>(out,it,1.0000001,1e-9)));
    printf("   -> cycles per dependent DFMA: %.2f\n", ms*1e-3*ghz*1e9/it); }
  { RUN("DMMA latency: 1 warp/SM 1 chain", 512.0*it*(double)sms, (dmma_k<1><<<sms,32>>>(out,it,1.0000001,1e-9)));
    printf("   -> cycles per dependent DMMA: %.2f\n", ms*1e-3*ghz*1e9/it); }
  for(int wps: {4,8,16}){
    char l[96];
    snprintf(l,96,"DMMA 8 chains, %d warps/SM",wps); RUN(l, 512.0*8*it*(double)sms*wps, (dmma_k<8><<<sms,wps*32>>>(out,it,1.0000001,1e-9)));
    snprintf(l,96,"DMMA 4 chains, %d warps/SM",wps); RUN(l, 512.0*4*it*(double)sms*wps, (dmma_k<4><<<sms,wps*32>>>(out,it,1.0000001,1e-9)));
    snprintf(l,96,"DMMA 1 chain, %d warps/SM",wps); RUN(l, 512.0*1*it*(double)sms*wps, (dmma_k<1><<<sms,wps*32>>>(out,it,1.0000001,1e-9)));
  }
  // mixed: 4 DMMA warps + 4 DFMA warps per SM (8 chains each): equal flops per warp per iteration? DMMA: 512/inst/warp, DFMA 64/inst/warp
  { int itm=it, itf=it*8; double fl=(512.0*8*itm*4 + 64.0*8*itf*4)*sms;
    RUN("MIX 4 DMMA warps + 4 DFMA warps (equal flops)", fl, (mix_k<8><<<sms,256>>>(out,itm,itf,4,1.0000001,1e-9)));
    RUN("  ref: DMMA part alone (4 warps)", 512.0*8*itm*4*sms, (mix_k<8><<<sms,128>>>(out,itm,itf,4,1.0000001,1e-9)));
    RUN("  ref: DFMA part alone (4 warps)", 64.0*8*itf*4*sms, (mix_k<8><<<sms,128>>>(out,itm,itf,0,1.0000001,1e-9)));
  }
  { RUN("INTERLEAVE 1 DMMA : 8 DFMA per warp, 8 warps", (512.0+64*8)*4*it*(double)sms*8, (inter_k<8><<<sms,256>>>(out,it,1.0000001,1e-9)));
    RUN("INTERLEAVE 1 DMMA : 4 DFMA per warp, 8 warps", (512.0+64*4)*4*it*(double)sms*8, (inter_k<4><<<sms,256>>>(out,it,1.0000001,1e-9)));
    RUN("INTERLEAVE 1 DMMA : 2 DFMA per warp, 8 warps", (512.0+64*2)*4*it*(double)sms*8, (inter_k<2><<<sms,256>>>(out,it,1.0000001,1e-9))); }
  return 0;
}
