// dmma_dot_probe.cu — stand-alone measurement (not part of libmadme.so): the dot stage of me_eval (step a7: J += U . C for
// one leg split, 8 helicity variants of the open current U x 4 of the propagated current C = the 32 helicity combinations of
// one event, one warp per event) in the CUDA-core form the kernel uses and as an FP64 tensor-core contraction.
// BASELINE.json:north_star: "uses FP64 tensor cores only if ncu shows it beats the CUDA-core form"; VERDICT r1 asked for the
// dot stages to be measured, not argued (profiles/r2_probes.md has the result).
//
// Real form of the complex contraction T[a][b] = sum_c U[a][c] C[b][c] (c = 4 components): an 8 x 8 x 8 real product
//   T[a][2b + im] = sum_k A[a][k] B[k][2b + im],  A[a][k] = (Ur | Ui)[a][k mod 4],
//   B[k][2b] = (Cr | -Ci)[b][k mod 4],  B[k][2b+1] = (Ci | Cr)[b][k mod 4]
// = two mma.sync.m8n8k4.f64.  The accumulator fragment leaves lane l with (T_re, T_im) of (a, b) = (l / 4, l % 4): the
// kernel's "lane = helicity combination" layout for THIS split.  Other leg splits put other helicity bits on the U side,
// so their fragments must be permuted across lanes before they can be added to the same J: variant `perm` pays that with
// shuffles, variant `ideal` pretends every split had the same layout (an upper bound for the tensor-core form).
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o dmma_dot_probe dmma_dot_probe.cu && ./dmma_dot_probe
#include <cstdio>
#include <cmath>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("err %s line %d\n", cudaGetErrorString(e), __LINE__); return 1;}}while(0)

constexpr int NS = 16;            // leg splits per repetition (the operands of each live in shared memory)
constexpr int WARPS = 8;          // warps per CTA = events per CTA, as in me_eval
constexpr int SPLIT_DOUBLES = 128;   // U: 4 lines x 16 doubles (8 variants x (re, im)), C: 4 lines x 16 doubles (4 variants used)
constexpr int EV_DOUBLES = NS * SPLIT_DOUBLES + 2;   // event stride = 16 B mod 128 B, as in the kernel

__device__ __forceinline__ void dmma(double& d0, double& d1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// mode 0: DFMA form (the kernel's dot_acc), 1: DMMA + lane permutation per split, 2: DMMA, same layout for every split
template <int MODE>
__global__ void __launch_bounds__(32 * WARPS, 1) dot_k(const double* __restrict__ in, double* __restrict__ out, int reps) {
  extern __shared__ __align__(16) double sm[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double* ev = sm + warp * EV_DOUBLES;
  for (int i = lane; i < NS * SPLIT_DOUBLES; i += 32) ev[i] = in[(blockIdx.x * WARPS + warp) * NS * SPLIT_DOUBLES + i];
  __syncwarp();
  constexpr int NF = 8;            // colour flows fed in turn (the kernel holds 24: independent accumulator chains)
  double jr[NF], ji[NF];
#pragma unroll
  for (int f = 0; f < NF; ++f) { jr[f] = 0.0; ji[f] = 0.0; }
  const int a = lane >> 2, b = lane & 3;
  for (int r = 0; r < reps; ++r) {
    asm volatile("" ::: "memory");   // the operands are re-read from shared memory in every repetition, as in the kernel
#pragma unroll
    for (int s = 0; s < NS; ++s) {
      const double* U = ev + s * SPLIT_DOUBLES;        // component c, variant v: U[16 c + 2 v], +1 imaginary
      const double* C = U + 64;
      if (MODE == 0) {
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const double2 u = *reinterpret_cast<const double2*>(U + 16 * c + 2 * a);
          const double2 v = *reinterpret_cast<const double2*>(C + 16 * c + 2 * b);
          jr[s % NF] = fma(u.x, v.x, fma(-u.y, v.y, jr[s % NF]));
          ji[s % NF] = fma(u.x, v.y, fma(u.y, v.x, ji[s % NF]));
        }
      } else {
        // fragments: A[row = lane / 4][k = lane % 4], B[k = lane % 4][n = lane / 4], n = 2 b' + im
        const int k = lane & 3, n = lane >> 2, bb = n >> 1, im = n & 1;
        double t0 = 0.0, t1 = 0.0;
        const double ar = U[16 * k + 2 * a], ai = U[16 * k + 2 * a + 1];
        const double cr = C[16 * k + 2 * bb], ci = C[16 * k + 2 * bb + 1];
        dmma(t0, t1, ar, im ? ci : cr);
        dmma(t0, t1, ai, im ? cr : -ci);
        if (MODE == 1) {   // this split's (a, b) -> the lane that holds that helicity combination in J's layout
          const int src = ((lane << (s % 5)) | (lane >> (5 - s % 5))) & 31;
          t0 = __shfl_sync(0xffffffffu, t0, src);
          t1 = __shfl_sync(0xffffffffu, t1, src);
        }
        jr[s % NF] += t0;
        ji[s % NF] += t1;
      }
    }
  }
  double sr = 0.0, si = 0.0;
#pragma unroll
  for (int f = 0; f < NF; ++f) { sr += jr[f]; si += ji[f]; }
  out[(blockIdx.x * blockDim.x + threadIdx.x) * 2] = sr;
  out[(blockIdx.x * blockDim.x + threadIdx.x) * 2 + 1] = si;
}

int main() {
  int dev = 0, sms = 0, khz = 0;
  CK(cudaGetDevice(&dev));
  CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  CK(cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev));
  const int n_in = sms * WARPS * NS * SPLIT_DOUBLES;
  double* h = new double[n_in];
  unsigned long long x = 88172645463325252ull;
  for (int i = 0; i < n_in; ++i) { x ^= x << 13; x ^= x >> 7; x ^= x << 17; h[i] = (double)(x >> 11) / 9007199254740992.0 - 0.5; }
  double *d_in, *d_out;
  CK(cudaMalloc(&d_in, sizeof(double) * n_in));
  CK(cudaMalloc(&d_out, sizeof(double) * sms * 32 * WARPS * 2));
  CK(cudaMemcpy(d_in, h, sizeof(double) * n_in, cudaMemcpyHostToDevice));
  const int smem = WARPS * EV_DOUBLES * 8;
  CK(cudaFuncSetAttribute(dot_k<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  CK(cudaFuncSetAttribute(dot_k<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  CK(cudaFuncSetAttribute(dot_k<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  const int reps = 20000;
  double ref[64];
  const char* names[3] = {"DFMA form (kernel)", "DMMA + lane permutation per split", "DMMA, one layout for all splits (bound)"};
  for (int mode = 0; mode < 3; ++mode) {
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    for (int pass = 0; pass < 2; ++pass) {
      CK(cudaEventRecord(e0));
      if (mode == 0) dot_k<0><<<sms, 32 * WARPS, smem>>>(d_in, d_out, reps);
      if (mode == 1) dot_k<1><<<sms, 32 * WARPS, smem>>>(d_in, d_out, reps);
      if (mode == 2) dot_k<2><<<sms, 32 * WARPS, smem>>>(d_in, d_out, reps);
      CK(cudaEventRecord(e1));
      CK(cudaDeviceSynchronize());
    }
    float ms = 0;
    CK(cudaEventElapsedTime(&ms, e0, e1));
    double o[64];
    CK(cudaMemcpy(o, d_out, sizeof o, cudaMemcpyDeviceToHost));
    double dev_max = 0;
    if (mode == 0) for (int i = 0; i < 64; ++i) ref[i] = o[i];
    if (mode == 2) for (int i = 0; i < 64; ++i) dev_max = fmax(dev_max, fabs(o[i] - ref[i]) / (fabs(ref[i]) + 1e-300));
    // one contraction = 32 helicity combinations x 4 complex MACs = 512 real FMAs = 1024 flop per warp and split
    const double contractions = (double)sms * WARPS * NS * reps;
    const double cyc = ms * 1e-3 * khz * 1e3;
    printf("%-44s %8.3f ms  %6.2f cycles per contraction and SM-warp-slot  %6.1f flop/clk/SM%s\n", names[mode], ms,
           cyc / (NS * (double)reps), contractions * 1024.0 / cyc / sms, mode == 2 ? "" : "");
    if (mode == 2) printf("   DMMA (one layout) against DFMA result, first 32 lanes: max relative difference %.2e\n", dev_max);
  }
  return 0;
}
