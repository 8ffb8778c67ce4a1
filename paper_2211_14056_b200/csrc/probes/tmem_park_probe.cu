// tmem_park_probe.cu — stand-alone measurement (not part of libmadme.so): tensor memory as a parking lot for registers.
// 8 warps x 96 registers per thread, tcgen05.st -> tcgen05.ld round trip, checked and timed (profiles/r2_probes.md);
// csrc/tmem.cuh is the product form.
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o tmem_park_probe tmem_park_probe.cu && ./tmem_park_probe
#include <cstdio>
#include <cuda_runtime.h>
#include <cstdint>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("err %s line %d\n", cudaGetErrorString(e), __LINE__); return 1;}}while(0)

__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t* r){
  asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
   :: "r"(taddr), "r"(r[0]),"r"(r[1]),"r"(r[2]),"r"(r[3]),"r"(r[4]),"r"(r[5]),"r"(r[6]),"r"(r[7]),"r"(r[8]),"r"(r[9]),"r"(r[10]),"r"(r[11]),"r"(r[12]),"r"(r[13]),"r"(r[14]),"r"(r[15]),
      "r"(r[16]),"r"(r[17]),"r"(r[18]),"r"(r[19]),"r"(r[20]),"r"(r[21]),"r"(r[22]),"r"(r[23]),"r"(r[24]),"r"(r[25]),"r"(r[26]),"r"(r[27]),"r"(r[28]),"r"(r[29]),"r"(r[30]),"r"(r[31]) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t* r){
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
   : "=r"(r[0]),"=r"(r[1]),"=r"(r[2]),"=r"(r[3]),"=r"(r[4]),"=r"(r[5]),"=r"(r[6]),"=r"(r[7]),"=r"(r[8]),"=r"(r[9]),"=r"(r[10]),"=r"(r[11]),"=r"(r[12]),"=r"(r[13]),"=r"(r[14]),"=r"(r[15]),
     "=r"(r[16]),"=r"(r[17]),"=r"(r[18]),"=r"(r[19]),"=r"(r[20]),"=r"(r[21]),"=r"(r[22]),"=r"(r[23]),"=r"(r[24]),"=r"(r[25]),"=r"(r[26]),"=r"(r[27]),"=r"(r[28]),"=r"(r[29]),"=r"(r[30]),"=r"(r[31]) : "r"(taddr) : "memory");
}
__global__ void __launch_bounds__(256,1) k(double* out, long long* cyc, int iters){
  __shared__ uint32_t base_s;
  const int warp=threadIdx.x>>5, lane=threadIdx.x&31;
  if(warp==0){
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 256;" :: "r"((uint32_t)__cvta_generic_to_shared(&base_s)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t base=base_s;
  const uint32_t taddr = base + ((uint32_t)(32*(warp&3))<<16) + (warp>>2)*128;
  double j[48];
  for(int i=0;i<48;++i) j[i]=1.0+ i*0.001 + threadIdx.x + blockIdx.x*1000.0;
  long long t0=clock64();
  for(int it=0; it<iters; ++it){
    uint32_t* r=reinterpret_cast<uint32_t*>(j);
    tmem_st32(taddr, r); tmem_st32(taddr+32, r+32); tmem_st32(taddr+64, r+64);
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
    for(int i=0;i<48;++i) j[i]=-1.0;   // clobber
    tmem_ld32(taddr, r); tmem_ld32(taddr+32, r+32); tmem_ld32(taddr+64, r+64);
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
    for(int i=0;i<48;++i) j[i]+=1.0;
  }
  long long t1=clock64();
  double s=0; for(int i=0;i<48;++i) s+=j[i];
  out[blockIdx.x*blockDim.x+threadIdx.x]=s;
  if(threadIdx.x==0) cyc[blockIdx.x]=t1-t0;
  __syncthreads();
  if(warp==0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 256;" :: "r"(base) : "memory");
}
int main(){
  int nb=148, iters=100;
  double* out; long long* cyc; CK(cudaMalloc(&out,sizeof(double)*nb*256)); CK(cudaMalloc(&cyc,8*nb));
  k<<<nb,256>>>(out,cyc,iters); CK(cudaDeviceSynchronize());
  static double h[148*256]; long long hc[148];
  CK(cudaMemcpy(h,out,sizeof(h),cudaMemcpyDeviceToHost)); CK(cudaMemcpy(hc,cyc,sizeof(hc),cudaMemcpyDeviceToHost));
  int bad=0;
  for(int b=0;b<nb;++b) for(int t=0;t<256;++t){ double e=0; for(int i=0;i<48;++i) e+=1.0+i*0.001+t+b*1000.0+iters; if(fabs(h[b*256+t]-e)>1e-6*fabs(e)){ if(bad<5) printf("mismatch b%d t%d got %f exp %f\n",b,t,h[b*256+t],e); ++bad;} }
  printf("tmem round trip: %d mismatches; %.1f cycles per st96+ld96 round trip (8 warps)\n",bad,(double)hc[0]/iters);
  return bad!=0;
}
