// proc_eval.cu — me_eval for ONE process: compiled once per process with -DMADME_PROC=<process> (build.py).
// W (events = warps per CTA) is a run-time choice among the compiled instances; MADME_WARPS overrides it — the
// threads-per-block scan of PAPER.md:78-84 (Fig. 3) is repeated with it.
#include "common.cuh"
#include "me_kernel.cuh"

#ifndef MADME_PROC
#error "compile with -DMADME_PROC=<process>"
#endif
#define MADME_CAT_(a, b, c) a##b##c
#define MADME_CAT(a, b, c) MADME_CAT_(a, b, c)

namespace madme {
// a named namespace per (process, file): this file is compiled several times into one library
namespace MADME_CAT(tu_, MADME_PROC, _e) {
using P = MADME_PROC;

template <int W> int geom(int* regs, int* ctas) {
  cudaFuncAttributes fa;
  CU(cudaFuncGetAttributes(&fa, me_eval_kernel<P, W>));
  const int bytes = W * EventSmem<P>::DOUBLES * 8;
  if (cudaFuncSetAttribute(me_eval_kernel<P, W>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes) != cudaSuccess) {
    (void)cudaGetLastError();
    *ctas = 0;
    return ME_OK;
  }
  *regs = fa.numRegs;
  CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas, me_eval_kernel<P, W>, 32 * W, bytes));
  return ME_OK;
}

int fill(me_handle* h) {
  h->n_ext = P::N_EXT; h->n_hel = P::N_HEL; h->n_flow = P::N_FLOW; h->n_diag = P::N_DIAGRAMS;
  h->n_terms = P::N_TERMS; h->n_diag4g = P::N_DIAGRAMS_4G; h->n_cur = P::N_CURRENTS; h->flops = P::FLOPS_PER_EVENT;
  const double g2 = P::QED ? 4.0 * PS_PI * h->par.alpha_em : 4.0 * PS_PI * h->par.alpha_s;  // g^2
  double c = 1.0;
  for (int i = 0; i < P::COUPLING_POWER / 2; ++i) c *= g2;
  h->scale = c / (double(P::CF_DEN) * double(P::AVG_DEN));
  int dev = 0;
  CU(cudaGetDevice(&dev));
  CU(cudaDeviceGetAttribute(&h->sms, cudaDevAttrMultiProcessorCount, dev));
  const int cand[4] = {1, 2, 4, 8};
  int regs[4] = {0, 0, 0, 0}, ctas[4] = {0, 0, 0, 0}, rc;
  if ((rc = geom<1>(&regs[0], &ctas[0])) || (rc = geom<2>(&regs[1], &ctas[1])) || (rc = geom<4>(&regs[2], &ctas[2])) ||
      (rc = geom<8>(&regs[3], &ctas[3])))
    return rc;
  int pick = -1;
  const char* env = getenv("MADME_WARPS");
  if (env) {
    for (int k = 0; k < 4; ++k)
      if (atoi(env) == cand[k] && ctas[k] > 0) pick = k;
    if (pick < 0) return fail(ME_EINVAL, "MADME_WARPS must be 1, 2, 4 or 8 (and fit on an SM)%s%s");
  } else {
    // most resident warps per SM; ties go to the larger CTA (fuller lanes in the current stages)
    int best = 0;
    for (int k = 0; k < 4; ++k)
      if (cand[k] * ctas[k] >= best && ctas[k] > 0) { best = cand[k] * ctas[k]; pick = k; }
    if (pick < 0) return fail(ME_ECUDA, "me_eval kernel does not fit on an SM%s%s");
  }
  h->warps = cand[pick];
  h->regs = regs[pick];
  h->ctas_per_sm = ctas[pick];
  h->smem_bytes = h->warps * EventSmem<P>::DOUBLES * 8;
  h->grid = h->sms * h->ctas_per_sm;
  return ME_OK;
}

int eval(me_handle* h, const double* mom, double* me2, double* hel, long long n, cudaStream_t s) {
  const long long need = (n + h->warps - 1) / h->warps;
  const int grid = static_cast<int>(need < h->grid ? need : h->grid), T = 32 * h->warps;
  switch (h->warps) {
    case 1: me_eval_kernel<P, 1><<<grid, T, h->smem_bytes, s>>>(mom, me2, hel, n, h->mass, h->scale); break;
    case 2: me_eval_kernel<P, 2><<<grid, T, h->smem_bytes, s>>>(mom, me2, hel, n, h->mass, h->scale); break;
    case 4: me_eval_kernel<P, 4><<<grid, T, h->smem_bytes, s>>>(mom, me2, hel, n, h->mass, h->scale); break;
    default: me_eval_kernel<P, 8><<<grid, T, h->smem_bytes, s>>>(mom, me2, hel, n, h->mass, h->scale); break;
  }
  CU(cudaGetLastError());
  return ME_OK;
}

const ProcOps ops = {fill, eval, nullptr};
}  // namespace tu_<process>

const ProcOps* MADME_CAT(ops_, MADME_PROC, _eval)() { return &MADME_CAT(tu_, MADME_PROC, _e)::ops; }
}  // namespace madme
