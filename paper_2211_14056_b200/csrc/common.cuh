// common.cuh — shared by the translation units of libmadme.so: error reporting, the handle, and the table of
// per-process entry points (each process's kernels are compiled in their own translation units).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "../../include/madme.h"
#include "vegas_common.cuh"

namespace madme {

extern thread_local char g_err[512];
inline int fail(int code, const char* fmt, const char* a = "", const char* b = "") {
  snprintf(g_err, sizeof g_err, fmt, a, b);
  return code;
}
inline int cuda_fail(cudaError_t e, const char* where) { return fail(ME_ECUDA, "%s: %s", where, cudaGetErrorString(e)); }
#define CU(call)                                                  \
  do {                                                            \
    cudaError_t e__ = (call);                                     \
    if (e__ != cudaSuccess) return madme::cuda_fail(e__, #call);  \
  } while (0)

struct ProcOps;

}  // namespace madme

struct me_handle {
  const madme::ProcOps* ev = nullptr;  // the process's me_eval entry points (proc_eval.cu)
  const madme::ProcOps* vg = nullptr;  // its fused Vegas integrand (proc_vegas.cu); QCD processes only
  bool qed = false;
  me_params par;
  int n_ext, n_hel, n_flow, n_diag, n_terms, n_diag4g, n_cur;
  double mass, scale, flops;
  double masses[madme::PS_MAX_FINAL];
  unsigned gluon_mask;
  int beam_kind[2] = {0, 0};  // toy density of each beam in the hadronic Vegas mode: 0 gluon, 1 quark, 2 antiquark
  // launch geometry of the CTA-per-W-events kernels
  int warps, grid, smem_bytes, regs, ctas_per_sm, sms;
  int device = 0;  // the device that was current in me_init: every call runs there
  // vegas scratch: per-event buffers sized by me_reserve, fixed-size buffers by me_init; calls never allocate
  int vegas_grid = 0;  // CTAs of the fused integrand kernel (fixed at me_init)
  long long* block_counts = nullptr;  // vegas_unweight: accepted events per 256-event block [scratch_ev / 256 + 2]
  double* f_scratch = nullptr;
  unsigned long long* idx_scratch = nullptr;
  long long scratch_ev = 0;
  double* partial = nullptr;
  long long partial_len = 0;
  double* sums_d = nullptr;
  double* sums_h = nullptr;  // pinned
  double* vegas_stage = nullptr;  // per-CTA survivor staging of the fused integrand (L2 resident)
  long long vegas_stage_len = 0;
};

namespace madme {

struct ProcOps {
  int (*prepare)(me_handle* h);  // vegas: per-device kernel attribute, launch geometry, staging size (me_init)
  int (*fill)(me_handle* h);  // constants of the generated program + launch geometry
  int (*eval)(me_handle* h, const double* mom, double* me2, double* hel, long long n, cudaStream_t s);
  int (*integrand)(me_handle* h, const VegasArgs& a, double* f, unsigned long long* idx, int words, cudaStream_t s);
};
#define MADME_DECLARE_OPS(P) const ProcOps* ops_##P##_eval(); const ProcOps* ops_##P##_vegas();
// every process of gen/diagrams.py::PROCESSES (build.py compiles proc_eval.cu / proc_vegas.cu once for each)
#define MADME_FOR_EACH_PROCESS(X) \
  X(epem_mupmum) X(gg_ttx) X(gg_ttxg) X(gg_ttxgg) X(gg_ttxggg) X(qqx_ttx) X(qqx_ttxg) X(qg_ttxq) X(qqx_ttxgg) X(qg_ttxqg) X(qxg_ttxqx) X(qxg_ttxqxg)
MADME_FOR_EACH_PROCESS(MADME_DECLARE_OPS)

}  // namespace madme
