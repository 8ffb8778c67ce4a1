// proc_eval.cu — me_eval for ONE process: compiled once per process with -DMADME_PROC=<process> (build.py).
// A CTA is 8 warps = 8 events (me_kernel.cuh); the events-per-CTA scan of PAPER.md:78-84 (Fig. 3) was done on the
// round-1 kernel (profiles/r1_block_size_scan.md).
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

int geom(me_handle* h) {
  cudaFuncAttributes fa;
  CU(cudaFuncGetAttributes(&fa, me_eval_kernel<P>));
  const int bytes = P::W_EVENTS * EventSmem<P>::DOUBLES * 8;
  CU(cudaFuncSetAttribute(me_eval_kernel<P>, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  int ctas = 0;
  CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas, me_eval_kernel<P>, 32 * P::N_WARPS, bytes));
  if (ctas < 1) return fail(ME_ECUDA, "me_eval kernel does not fit on an SM%s%s");
  // tensor memory: 512 columns per SM shared by the resident CTAs
  if (JPark<P>::ON && ctas * JPark<P>::COLS > 512) ctas = 512 / JPark<P>::COLS;
  h->warps = P::W_EVENTS;
  h->regs = fa.numRegs;
  h->ctas_per_sm = ctas;
  h->smem_bytes = bytes;
  h->grid = h->sms * ctas;
  return ME_OK;
}

int fill(me_handle* h) {
  h->n_ext = P::N_EXT; h->n_hel = P::N_HEL; h->n_flow = P::N_FLOW; h->n_diag = P::N_DIAGRAMS;
  h->n_terms = P::N_TERMS; h->n_diag4g = P::N_DIAGRAMS_4G; h->n_cur = P::N_CURRENTS; h->flops = P::FLOPS_PER_EVENT;
  h->qed = P::QED;
  h->mass = P::QED ? 0.0 : h->par.m_top;
  // final-state particle i (leg i + 2): its mass, and whether the jet cuts apply to it (massless coloured partons)
  for (int i = 0; i < PS_MAX_FINAL; ++i) h->masses[i] = ((P::FINAL_MASSIVE_MASK >> i) & 1) ? h->par.m_top : 0.0;
  h->gluon_mask = P::JET_MASK;
  h->beam_kind[0] = P::BEAM_KIND_0; h->beam_kind[1] = P::BEAM_KIND_1;
  const double g2 = P::QED ? 4.0 * PS_PI * h->par.alpha_em : 4.0 * PS_PI * h->par.alpha_s;  // g^2
  double c = 1.0;
  for (int i = 0; i < P::COUPLING_POWER / 2; ++i) c *= g2;
  h->scale = c / (double(P::CF_DEN) * double(P::AVG_DEN));
  int dev = 0;
  CU(cudaGetDevice(&dev));
  CU(cudaDeviceGetAttribute(&h->sms, cudaDevAttrMultiProcessorCount, dev));
  return geom(h);
}

int eval(me_handle* h, const double* mom, double* me2, double* hel, long long n, cudaStream_t s) {
  const long long need = (n + P::W_EVENTS - 1) / P::W_EVENTS;
  const int grid = static_cast<int>(need < h->grid ? need : h->grid);
  me_eval_kernel<P><<<grid, 32 * P::N_WARPS, h->smem_bytes, s>>>(mom, me2, hel, n, h->mass, h->scale);
  CU(cudaGetLastError());
  return ME_OK;
}

const ProcOps ops = {nullptr, fill, eval, nullptr};
}  // namespace tu_<process>

const ProcOps* MADME_CAT(ops_, MADME_PROC, _eval)() { return &MADME_CAT(tu_, MADME_PROC, _e)::ops; }
}  // namespace madme
