// madme.cu — the C ABI of include/madme.h on top of the sm_100a kernels.  No CPU path: without a CUDA device
// every compute call fails with ME_ENODEV.  The per-process kernels are compiled in their own translation units
// (proc_eval.cu, proc_vegas.cu with -DMADME_PROC=<process>) and reached through ProcOps.
#include "common.cuh"
#include "phase_space.cuh"

using namespace madme;

thread_local char madme::g_err[512] = "";

namespace {

bool have_device() {
  static int state = -1;
  if (state < 0) {
    int n = 0;
    state = (cudaGetDeviceCount(&n) == cudaSuccess && n > 0) ? 1 : 0;
    if (!state) (void)cudaGetLastError();
  }
  return state == 1;
}
bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

// ---- stand-alone phase-space kernels: one event per thread ------------------------------------------------
__global__ void philox_kernel(unsigned long long seed, unsigned iteration, long long first, int n_dim, double* __restrict__ out,
                              long long n_ev) {
  const long long ev = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (ev >= n_ev) return;
  double u[VEGAS_MAX_DIM];
  philox_fill<VEGAS_MAX_DIM>(seed, iteration, static_cast<uint64_t>(first + ev), n_dim, u);
#pragma unroll
  for (int d = 0; d < VEGAS_MAX_DIM; ++d)
    if (d < n_dim) out[ev * n_dim + d] = u[d];
}

struct RamboArgs {
  double sqrt_s, w0;
  double masses[PS_MAX_FINAL];
  int ps_mode;
};
template <int N>
__global__ void rambo_kernel(const double* __restrict__ rand, RamboArgs a, double* __restrict__ mom, double* __restrict__ wgt,
                             long long n_ev) {
  const long long ev = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (ev >= n_ev) return;
  constexpr int DMAX = 4 * N;
  const int n_dim = a.ps_mode == 0 ? 4 * N : 3 * N - 4;
  double r[DMAX], p[N][4];
#pragma unroll
  for (int d = 0; d < DMAX; ++d) r[d] = d < n_dim ? rand[ev * n_dim + d] : 0.5;
  const double w = rambo_event<N>(r, a.sqrt_s, a.masses, a.ps_mode, a.w0, p);
  double* o = mom + ev * (4 * (N + 2));
  const double e = 0.5 * a.sqrt_s;
  reinterpret_cast<double2*>(o)[0] = make_double2(e, 0.0);
  reinterpret_cast<double2*>(o)[1] = make_double2(0.0, e);
  reinterpret_cast<double2*>(o)[2] = make_double2(e, 0.0);
  reinterpret_cast<double2*>(o)[3] = make_double2(0.0, -e);
#pragma unroll
  for (int i = 0; i < N; ++i) {
    reinterpret_cast<double2*>(o)[4 + 2 * i] = make_double2(p[i][0], p[i][1]);
    reinterpret_cast<double2*>(o)[5 + 2 * i] = make_double2(p[i][2], p[i][3]);
  }
  wgt[ev] = w;
}
template <int N>
__global__ void cuts_kernel(const double* __restrict__ mom, unsigned gluon_mask, double ptj_min, double dr_min, int* __restrict__ pass,
                            long long n_ev) {
  const long long ev = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (ev >= n_ev) return;
  double p[N][4];
  const double2* in = reinterpret_cast<const double2*>(mom + ev * (4 * (N + 2)));
#pragma unroll
  for (int i = 0; i < N; ++i) {
    const double2 a = in[4 + 2 * i], b = in[5 + 2 * i];
    p[i][0] = a.x; p[i][1] = a.y; p[i][2] = b.x; p[i][3] = b.y;
  }
  pass[ev] = passes_cuts<N>(p, gluon_mask, ptj_min, dr_min) ? 1 : 0;
}
__global__ void vegas_map_kernel(const double* __restrict__ edges, int n_dim, int n_bins, const double* __restrict__ y,
                                 double* __restrict__ x, double* __restrict__ jac, int* __restrict__ idx, long long n) {
  const long long ev = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (ev >= n) return;
  double j = 1.0;
  for (int d = 0; d < n_dim; ++d) {
    int bin;
    x[ev * n_dim + d] = vegas_map_1d(edges + d * (n_bins + 1), n_bins, y[ev * n_dim + d], j, bin);
    idx[ev * n_dim + d] = bin;
  }
  jac[ev] = j;
}

// fp64 roofline denominator: 8 independent DFMA chains per thread, register resident
__global__ void __launch_bounds__(256) dfma_probe_kernel(long long n_iter, double* sink) {
  double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
  const double m = 0.999999999, c = 1e-9;
  for (long long it = 0; it < n_iter; ++it) {
#pragma unroll
    for (int k = 0; k < 256; ++k) {
      a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
      a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
  }
  const double s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
  if (s == 123.456) *sink = s;
}

inline int blocks_for(long long n, int threads) { return static_cast<int>((n + threads - 1) / threads); }

int ensure_scratch(me_handle* h, long long n_ev, int idx_words, int n_chunks, int n_out) {
  if (n_ev > h->scratch_ev) {
    if (h->f_scratch) cudaFree(h->f_scratch);
    if (h->idx_scratch) cudaFree(h->idx_scratch);
    h->f_scratch = nullptr; h->idx_scratch = nullptr; h->scratch_ev = 0;
    CU(cudaMalloc(&h->f_scratch, sizeof(double) * n_ev));
    CU(cudaMalloc(&h->idx_scratch, sizeof(unsigned long long) * 2 * n_ev));
    h->scratch_ev = n_ev;
  }
  (void)idx_words;
  const long long need = static_cast<long long>(n_chunks) * n_out;
  if (need > h->partial_len) {
    if (h->partial) cudaFree(h->partial);
    h->partial = nullptr; h->partial_len = 0;
    CU(cudaMalloc(&h->partial, sizeof(double) * need));
    h->partial_len = need;
  }
  return ME_OK;
}

}  // namespace

extern "C" {

const char* me_last_error(void) { return g_err; }

int me_init(const char* process, const me_params* params, me_handle** out) {
  if (!process || !params || !out) return fail(ME_EINVAL, "me_init: null argument%s%s");
  *out = nullptr;
  Proc pr;
  if (!strcmp(process, "epem_mupmum")) pr = P_EPEM;
  else if (!strcmp(process, "gg_ttx")) pr = P_GGTT;
  else if (!strcmp(process, "gg_ttxg")) pr = P_GGTTG;
  else if (!strcmp(process, "gg_ttxgg")) pr = P_GGTTGG;
  else return fail(ME_EPROCESS, "me_init: unknown process '%s'%s", process);
  if (params->w_top != 0.0) return fail(ME_EINVAL, "me_init: w_top must be 0 (no width in propagators)%s%s");
  if (!have_device()) return fail(ME_ENODEV, "me_init: no CUDA device (this library has no CPU path)%s%s");
  me_handle* h = new me_handle();
  h->proc = pr;
  h->par = *params;
  h->mass = (pr == P_EPEM) ? 0.0 : params->m_top;
  for (int i = 0; i < PS_MAX_FINAL; ++i) h->masses[i] = 0.0;
  h->gluon_mask = 0;
  if (pr != P_EPEM) { h->masses[0] = h->masses[1] = params->m_top; }
  if (pr == P_GGTTG) h->gluon_mask = 0x4;
  if (pr == P_GGTTGG) h->gluon_mask = 0xC;
  int rc;
  switch (pr) {
    case P_EPEM: rc = ops_epem_mupmum_eval()->fill(h); break;
    case P_GGTT: rc = ops_gg_ttx_eval()->fill(h); break;
    case P_GGTTG: rc = ops_gg_ttxg_eval()->fill(h); break;
    default: rc = ops_gg_ttxgg_eval()->fill(h); break;
  }
  if (rc == ME_OK) {
    cudaError_t e = cudaMalloc(&h->sums_d, sizeof(double) * (3 + VEGAS_MAX_DIM * VEGAS_MAX_BINS));
    if (e == cudaSuccess) e = cudaMallocHost(&h->sums_h, sizeof(double) * 4);
    if (e != cudaSuccess) rc = cuda_fail(e, "me_init scratch");
  }
  if (rc != ME_OK) { me_free(h); return rc; }
  *out = h;
  return ME_OK;
}

void me_free(me_handle* h) {
  if (!h) return;
  if (h->f_scratch) cudaFree(h->f_scratch);
  if (h->idx_scratch) cudaFree(h->idx_scratch);
  if (h->partial) cudaFree(h->partial);
  if (h->sums_d) cudaFree(h->sums_d);
  if (h->sums_h) cudaFreeHost(h->sums_h);
  if (h->vegas_stage) cudaFree(h->vegas_stage);
  delete h;
}

int me_n_external(const me_handle* h) { return h ? h->n_ext : ME_EINVAL; }
int me_n_final(const me_handle* h) { return h ? h->n_ext - 2 : ME_EINVAL; }
long long me_info(const me_handle* h, int what) {
  if (!h) return ME_EINVAL;
  switch (what) {
    case 0: return h->n_diag;
    case 1: return h->n_terms;
    case 2: return h->n_diag4g;
    case 3: return h->n_flow;
    case 4: return h->n_hel;
    case 5: return h->n_cur;
    case 6: return h->smem_bytes / h->warps;
    case 7: return h->warps;
    case 8: return h->regs;
    case 9: return h->ctas_per_sm;
    case 10: return h->sms;
    default: return ME_EINVAL;
  }
}
double me_flops_per_event(const me_handle* h) { return h ? h->flops : 0.0; }

static int eval_common(me_handle* h, const double* momenta, double* me2, double* hel, long long n_ev, void* stream) {
  if (!h || n_ev < 0) return fail(ME_EINVAL, "me_eval: null handle or negative n_ev%s%s");
  if (n_ev == 0) return ME_OK;  // an empty batch needs no buffers
  if (!momenta || (!me2 && !hel)) return fail(ME_EINVAL, "me_eval: null buffer%s%s");
  if (!aligned16(momenta)) return fail(ME_EINVAL, "me_eval: momenta must be 16-byte aligned%s%s");
  if (n_ev == 0) return ME_OK;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  switch (h->proc) {
    case P_EPEM: return ops_epem_mupmum_eval()->eval(h, momenta, me2, hel, n_ev, s);
    case P_GGTT: return ops_gg_ttx_eval()->eval(h, momenta, me2, hel, n_ev, s);
    case P_GGTTG: return ops_gg_ttxg_eval()->eval(h, momenta, me2, hel, n_ev, s);
    default: return ops_gg_ttxgg_eval()->eval(h, momenta, me2, hel, n_ev, s);
  }
}
int me_eval(me_handle* h, const double* momenta, double* me2, long long n_ev, void* stream) {
  if (!me2 && n_ev > 0) return fail(ME_EINVAL, "me_eval: me2 is null%s%s");
  return eval_common(h, momenta, me2, nullptr, n_ev, stream);
}
int me_eval_helicities(me_handle* h, const double* momenta, double* me2_hel, long long n_ev, void* stream) {
  if (!me2_hel && n_ev > 0) return fail(ME_EINVAL, "me_eval_helicities: me2_hel is null%s%s");
  return eval_common(h, momenta, nullptr, me2_hel, n_ev, stream);
}

int philox_uniform(uint64_t seed, uint64_t iteration, long long first_event, int n_dim, double* rand, long long n_ev, void* stream) {
  if ((!rand && n_ev > 0) || n_ev < 0 || first_event < 0) return fail(ME_EINVAL, "philox_uniform: null pointer or negative count%s%s");
  if (n_dim < 1 || n_dim > VEGAS_MAX_DIM) return fail(ME_EDIM, "philox_uniform: n_dim out of range 1..24%s%s");
  if (!have_device()) return fail(ME_ENODEV, "philox_uniform: no CUDA device%s%s");
  if (n_ev == 0) return ME_OK;
  philox_kernel<<<blocks_for(n_ev, 256), 256, 0, static_cast<cudaStream_t>(stream)>>>(seed, static_cast<unsigned>(iteration),
                                                                                      first_event, n_dim, rand, n_ev);
  CU(cudaGetLastError());
  return ME_OK;
}

int rambo_generate(const double* rand, double sqrt_s, const double* masses, int n_final, int ps_mode, double* momenta,
                   double* weights, long long n_ev, void* stream) {
  if (!masses || n_ev < 0 || (n_ev > 0 && (!rand || !momenta || !weights))) return fail(ME_EINVAL, "rambo_generate: null pointer or negative count%s%s");
  if (n_final < 2 || n_final > PS_MAX_FINAL || (ps_mode != 0 && ps_mode != 1)) return fail(ME_EDIM, "rambo_generate: n_final 2..6, ps_mode 0|1%s%s");
  if (!(sqrt_s > 0.0)) return fail(ME_EINVAL, "rambo_generate: sqrt_s must be positive%s%s");
  if (!aligned16(momenta)) return fail(ME_EINVAL, "rambo_generate: momenta must be 16-byte aligned%s%s");
  double msum = 0.0;
  RamboArgs a;
  for (int i = 0; i < PS_MAX_FINAL; ++i) a.masses[i] = 0.0;
  for (int i = 0; i < n_final; ++i) { a.masses[i] = masses[i]; msum += masses[i]; }
  if (!(msum < sqrt_s)) return fail(ME_EINVAL, "rambo_generate: sum of masses >= sqrt_s%s%s");
  if (!have_device()) return fail(ME_ENODEV, "rambo_generate: no CUDA device%s%s");
  if (n_ev == 0) return ME_OK;
  a.sqrt_s = sqrt_s; a.ps_mode = ps_mode; a.w0 = rambo_volume(n_final, sqrt_s * sqrt_s);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int T = 128, B = blocks_for(n_ev, T);
  switch (n_final) {
    case 2: rambo_kernel<2><<<B, T, 0, s>>>(rand, a, momenta, weights, n_ev); break;
    case 3: rambo_kernel<3><<<B, T, 0, s>>>(rand, a, momenta, weights, n_ev); break;
    case 4: rambo_kernel<4><<<B, T, 0, s>>>(rand, a, momenta, weights, n_ev); break;
    case 5: rambo_kernel<5><<<B, T, 0, s>>>(rand, a, momenta, weights, n_ev); break;
    default: rambo_kernel<6><<<B, T, 0, s>>>(rand, a, momenta, weights, n_ev); break;
  }
  CU(cudaGetLastError());
  return ME_OK;
}

int apply_cuts(const double* momenta, int n_final, const int* is_gluon, double ptj_min, double dr_min, int* pass, long long n_ev,
               void* stream) {
  if (!is_gluon || n_ev < 0 || (n_ev > 0 && (!momenta || !pass))) return fail(ME_EINVAL, "apply_cuts: null pointer or negative count%s%s");
  if (n_final < 2 || n_final > PS_MAX_FINAL) return fail(ME_EDIM, "apply_cuts: n_final 2..6%s%s");
  if (!aligned16(momenta)) return fail(ME_EINVAL, "apply_cuts: momenta must be 16-byte aligned%s%s");
  if (!have_device()) return fail(ME_ENODEV, "apply_cuts: no CUDA device%s%s");
  if (n_ev == 0) return ME_OK;
  unsigned mask = 0;
  for (int i = 0; i < n_final; ++i) if (is_gluon[i]) mask |= 1u << i;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int T = 128, B = blocks_for(n_ev, T);
  switch (n_final) {
    case 2: cuts_kernel<2><<<B, T, 0, s>>>(momenta, mask, ptj_min, dr_min, pass, n_ev); break;
    case 3: cuts_kernel<3><<<B, T, 0, s>>>(momenta, mask, ptj_min, dr_min, pass, n_ev); break;
    case 4: cuts_kernel<4><<<B, T, 0, s>>>(momenta, mask, ptj_min, dr_min, pass, n_ev); break;
    case 5: cuts_kernel<5><<<B, T, 0, s>>>(momenta, mask, ptj_min, dr_min, pass, n_ev); break;
    default: cuts_kernel<6><<<B, T, 0, s>>>(momenta, mask, ptj_min, dr_min, pass, n_ev); break;
  }
  CU(cudaGetLastError());
  return ME_OK;
}

int vegas_map(const double* edges, int n_dim, int n_bins, const double* y, double* x, double* jac, int* idx, long long n, void* stream) {
  if (!edges || n < 0 || (n > 0 && (!y || !x || !jac || !idx))) return fail(ME_EINVAL, "vegas_map: null pointer or negative count%s%s");
  if (n_dim < 1 || n_dim > VEGAS_MAX_DIM || n_bins < 1 || n_bins > VEGAS_MAX_BINS) return fail(ME_EDIM, "vegas_map: n_dim 1..24, n_bins 1..255%s%s");
  if (!have_device()) return fail(ME_ENODEV, "vegas_map: no CUDA device%s%s");
  if (n == 0) return ME_OK;
  vegas_map_kernel<<<blocks_for(n, 256), 256, 0, static_cast<cudaStream_t>(stream)>>>(edges, n_dim, n_bins, y, x, jac, idx, n);
  CU(cudaGetLastError());
  return ME_OK;
}

int vegas_refine(double* edges, int n_dim, int n_bins, const double* S, double alpha, void* stream) {
  if (!edges || !S) return fail(ME_EINVAL, "vegas_refine: null pointer%s%s");
  if (n_dim < 1 || n_dim > VEGAS_MAX_DIM || n_bins < 1 || n_bins > VEGAS_MAX_BINS) return fail(ME_EDIM, "vegas_refine: n_dim 1..24, n_bins 1..255%s%s");
  if (!have_device()) return fail(ME_ENODEV, "vegas_refine: no CUDA device%s%s");
  vegas_refine_kernel<<<1, 32, 0, static_cast<cudaStream_t>(stream)>>>(edges, n_dim, n_bins, S, alpha);
  CU(cudaGetLastError());
  return ME_OK;
}

int vegas_integrand(me_handle* h, const vegas_grid* g, double sqrt_s, long long first_event, long long n_ev, double* sums,
                    double* f_out, void* stream) {
  if (!h || !g || !g->edges || !sums || n_ev < 0 || first_event < 0) return fail(ME_EINVAL, "vegas_integrand: null pointer or negative count%s%s");
  if (h->proc == P_EPEM) return fail(ME_EINVAL, "vegas_integrand: QCD processes only%s%s");
  const int nf = h->n_ext - 2, D = g->n_dim, nb = g->n_bins;
  if (g->ps_mode < 0 || g->ps_mode > 2 || D != (g->ps_mode == 0 ? 4 * nf : g->ps_mode == 1 ? 3 * nf - 4 : 3 * nf - 2))
    return fail(ME_EDIM, "vegas_integrand: n_dim must be 4 n_final (ps_mode 0), 3 n_final - 4 (1) or 3 n_final - 2 (2)%s%s");
  if (nb < 1 || nb > VEGAS_MAX_BINS || D * nb + 3 > 512 * VEGAS_RED_PER_THREAD)
    return fail(ME_EDIM, "vegas_integrand: n_bins 1..255 and n_dim*n_bins <= 2045%s%s");
  if (!(sqrt_s > 2.0 * h->par.m_top)) return fail(ME_EINVAL, "vegas_integrand: sqrt_s below threshold%s%s");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int n_out = 3 + D * nb, words = (D + 7) / 8;
  if (n_ev == 0) { CU(cudaMemsetAsync(sums, 0, sizeof(double) * n_out, s)); return ME_OK; }
  // fixed-shape reduction: chunk = ceil(n_ev / 1024) rounded up to a multiple of the tile -> n_chunks <= 1024
  long long chunk = (n_ev + 1023) / 1024;
  chunk = ((chunk + VEGAS_RED_TILE - 1) / VEGAS_RED_TILE) * VEGAS_RED_TILE;
  const int n_chunks = static_cast<int>((n_ev + chunk - 1) / chunk);
  int rc = ensure_scratch(h, n_ev, words, n_chunks, n_out);
  if (rc) return rc;
  VegasArgs a;
  a.edges = g->edges; a.n_dim = D; a.n_bins = nb; a.ps_mode = g->ps_mode; a.seed = g->seed;
  a.iteration = static_cast<unsigned>(g->iteration); a.first_event = first_event; a.n_ev = n_ev; a.sqrt_s = sqrt_s;
  a.w0 = rambo_volume(nf, sqrt_s * sqrt_s); a.prefactor = PB_GEV2 / (2.0 * sqrt_s * sqrt_s);
  for (int i = 0; i < PS_MAX_FINAL; ++i) a.masses[i] = h->masses[i];
  a.gluon_mask = h->gluon_mask; a.ptj_min = h->par.ptj_min; a.dr_min = h->par.dr_min; a.mass = h->mass; a.scale = h->scale;
  double* f = f_out ? f_out : h->f_scratch;
  switch (h->proc) {
    case P_GGTT: rc = ops_gg_ttx_vegas()->integrand(h, a, f, h->idx_scratch, words, s); break;
    case P_GGTTG: rc = ops_gg_ttxg_vegas()->integrand(h, a, f, h->idx_scratch, words, s); break;
    default: rc = ops_gg_ttxgg_vegas()->integrand(h, a, f, h->idx_scratch, words, s); break;
  }
  if (rc) return rc;
  vegas_reduce_chunks<<<n_chunks, 512, 0, s>>>(f, h->idx_scratch, words, D, nb, n_ev, chunk, h->partial);
  CU(cudaGetLastError());
  vegas_reduce_final<<<blocks_for(n_out, 128), 128, 0, s>>>(h->partial, n_chunks, n_out, sums);
  CU(cudaGetLastError());
  return ME_OK;
}

int vegas_iterate(me_handle* h, vegas_grid* g, double sqrt_s, long long n_ev, vegas_result* result, void* stream) {
  if (!h || !g || !result || n_ev < 2) return fail(ME_EINVAL, "vegas_iterate: null pointer or n_ev < 2%s%s");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  int rc = vegas_integrand(h, g, sqrt_s, 0, n_ev, h->sums_d, nullptr, s);
  if (rc) return rc;
  vegas_refine_kernel<<<1, 32, 0, s>>>(g->edges, g->n_dim, g->n_bins, h->sums_d + 3, g->alpha);
  CU(cudaGetLastError());
  CU(cudaMemcpyAsync(h->sums_h, h->sums_d, sizeof(double) * 3, cudaMemcpyDeviceToHost, s));
  CU(cudaStreamSynchronize(s));
  const double N = static_cast<double>(n_ev), I = h->sums_h[0] / N;
  result->integral = I;
  result->variance = (h->sums_h[1] / N - I * I) / (N - 1.0);
  result->sum_w = h->sums_h[0];
  result->sum_w2 = h->sums_h[1];
  result->n_pass = static_cast<long long>(h->sums_h[2]);
  g->iteration += 1;
  return ME_OK;
}

int fp64_peak_probe(long long n_iter, double* sink, double* n_dfma, void* stream) {
  if (!sink || !n_dfma || n_iter < 1) return fail(ME_EINVAL, "fp64_peak_probe: bad argument%s%s");
  if (!have_device()) return fail(ME_ENODEV, "fp64_peak_probe: no CUDA device%s%s");
  int dev = 0, sms = 0;
  CU(cudaGetDevice(&dev));
  CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int blocks = sms * 8, threads = 256;
  dfma_probe_kernel<<<blocks, threads, 0, static_cast<cudaStream_t>(stream)>>>(n_iter, sink);
  CU(cudaGetLastError());
  *n_dfma = double(blocks) * threads * double(n_iter) * 8.0 * 256.0;
  return ME_OK;
}

}  // extern "C"
