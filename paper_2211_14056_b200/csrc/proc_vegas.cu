// proc_vegas.cu — the fused Vegas integrand for ONE process: compiled once per process with -DMADME_PROC=<process>.
#include "common.cuh"
#include "vegas_kernels.cuh"

#ifndef MADME_PROC
#error "compile with -DMADME_PROC=<process>"
#endif
#define MADME_CAT_(a, b, c) a##b##c
#define MADME_CAT(a, b, c) MADME_CAT_(a, b, c)

namespace madme {
// a named namespace per (process, file): this file is compiled several times into one library
namespace MADME_CAT(tu_, MADME_PROC, _v) {
using P = MADME_PROC;

// me_init: the kernel attribute is per device, the launch geometry and the size of the survivor staging are fixed
int prepare(me_handle* h) {
  constexpr int W = P::N_WARPS;   // threads per CTA = 32 W, each generates one event per batch
  CU(cudaFuncSetAttribute(vegas_integrand_kernel<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, h->smem_bytes));
  int per_sm = 0;
  CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, vegas_integrand_kernel<P>, 32 * W, h->smem_bytes));
  if (per_sm < 1) return fail(ME_ECUDA, "vegas_integrand kernel does not fit on an SM%s%s");
  if (JPark<P>::ON && per_sm * JPark<P>::COLS > 512) per_sm = 512 / JPark<P>::COLS;
  h->vegas_grid = h->sms * per_sm;
  h->vegas_stage_len = static_cast<long long>(h->vegas_grid) * 32 * W * (4 * (P::N_EXT - 2) + 4);
  return ME_OK;
}

int integrand(me_handle* h, const VegasArgs& a, double* f, unsigned long long* idx, int words, cudaStream_t s) {
  constexpr int W = P::N_WARPS;
  const long long need = (a.n_ev + 32 * W - 1) / (32 * W);
  const int grid = static_cast<int>(need < h->vegas_grid ? need : h->vegas_grid);
  vegas_integrand_kernel<P><<<grid, 32 * W, h->smem_bytes, s>>>(a, f, idx, words, h->vegas_stage);
  CU(cudaGetLastError());
  return ME_OK;
}

const ProcOps ops = {prepare, nullptr, nullptr, integrand};
}  // namespace tu_<process>

const ProcOps* MADME_CAT(ops_, MADME_PROC, _vegas)() { return &MADME_CAT(tu_, MADME_PROC, _v)::ops; }
}  // namespace madme
