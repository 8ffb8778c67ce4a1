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

// A handle lives on the device that was current in me_init: calls run there and restore the caller's device.
struct DeviceGuard {
  int prev = -1;
  bool ok = true;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; prev = -1; return; }
    if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    else if (prev == dev) prev = -1;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define ON_DEVICE_OF(h) DeviceGuard guard__((h)->device); if (!guard__.ok) return fail(ME_ECUDA, "cannot switch to the handle's device%s%s")
constexpr int VEGAS_MAX_CHUNKS = 1024, VEGAS_MAX_OUT = 512 * VEGAS_RED_PER_THREAD;

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

// ---- unweighting: hit-or-miss with a dedicated Philox counter word, order-preserving compaction ----
__device__ __forceinline__ bool unweight_keep(double f, double w_max, unsigned long long seed, unsigned iteration, long long event) {
  if (!(f > 0.0)) return false;
  const uint4 w = philox4x32_10(make_uint4(static_cast<uint32_t>(event), static_cast<uint32_t>(static_cast<unsigned long long>(event) >> 32),
                                           0x7fffffffu, iteration),
                                make_uint2(static_cast<uint32_t>(seed), static_cast<uint32_t>(seed >> 32)));
  return philox_u01(w.x, w.y) * w_max < f;
}
// pass 1: kept events per 256-event block (+ overweight count); pass 2 (one block): exclusive scan; pass 3: write
__global__ void __launch_bounds__(256) unweight_count_kernel(const double* __restrict__ f, long long n_ev, double w_max, unsigned long long seed,
                                                             unsigned iteration, long long first_event, long long* __restrict__ block_counts,
                                                             unsigned long long* __restrict__ n_over) {
  const long long e = static_cast<long long>(blockIdx.x) * 256 + threadIdx.x;
  const double v = e < n_ev ? f[e] : 0.0;
  const bool keep = e < n_ev && unweight_keep(v, w_max, seed, iteration, first_event + e);
  const int c = __syncthreads_count(keep);
  const int o = __syncthreads_count(e < n_ev && v > w_max);
  if (threadIdx.x == 0) {
    block_counts[blockIdx.x] = c;
    if (o) atomicAdd(n_over, static_cast<unsigned long long>(o));   // an integer count: order does not matter
  }
}
__global__ void __launch_bounds__(1024) unweight_scan_kernel(long long* __restrict__ block_counts, long long n_blocks, long long* __restrict__ counts) {
  __shared__ long long part[1024];
  const long long per = (n_blocks + 1023) / 1024, lo = threadIdx.x * per, hi = min(n_blocks, lo + per);
  long long s = 0;
  for (long long i = lo; i < hi; ++i) s += block_counts[i];
  part[threadIdx.x] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    long long run = 0;
    for (int i = 0; i < 1024; ++i) { const long long t = part[i]; part[i] = run; run += t; }
    counts[0] = run;
  }
  __syncthreads();
  long long run = part[threadIdx.x];
  for (long long i = lo; i < hi; ++i) { const long long t = block_counts[i]; block_counts[i] = run; run += t; }
}
__global__ void __launch_bounds__(256) unweight_write_kernel(const double* __restrict__ f, long long n_ev, double w_max, unsigned long long seed,
                                                             unsigned iteration, long long first_event, const long long* __restrict__ block_offsets,
                                                             long long* __restrict__ accepted) {
  __shared__ int warp_count[8];
  const long long e = static_cast<long long>(blockIdx.x) * 256 + threadIdx.x;
  const bool keep = e < n_ev && unweight_keep(f[e], w_max, seed, iteration, first_event + e);
  const unsigned mask = __ballot_sync(0xffffffffu, keep);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) warp_count[warp] = __popc(mask);
  __syncthreads();
  if (keep) {
    long long pos = block_offsets[blockIdx.x] + __popc(mask & ((1u << lane) - 1u));
    for (int k = 0; k < warp; ++k) pos += warp_count[k];
    accepted[pos] = first_event + e;
  }
}
__global__ void max_weight_kernel(const double* __restrict__ f, long long n_ev, double* __restrict__ w_max) {
  // grid-stride maximum; the maximum does not depend on the order, so one atomic per block is deterministic
  double m = 0.0;
  for (long long e = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x; e < n_ev; e += static_cast<long long>(gridDim.x) * blockDim.x)
    m = fmax(m, f[e]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0 && m > 0.0)
    atomicMax(reinterpret_cast<unsigned long long*>(w_max), static_cast<unsigned long long>(__double_as_longlong(m)));  // non-negative doubles order like integers
}

// the kinematics of listed events (same device functions as the fused integrand)
template <int NF>
__global__ void vegas_generate_kernel(VegasArgs a, const long long* __restrict__ ids, long long n, double* __restrict__ mom_out,
                                      double* __restrict__ wgt_out) {
  const long long k = static_cast<long long>(blockIdx.x) * blockDim.x + threadIdx.x;
  if (k >= n) return;
  double p[NF][4], y[VEGAS_MAX_DIM], x[VEGAS_MAX_DIM];
  philox_fill<VEGAS_MAX_DIM>(a.seed, a.iteration, static_cast<uint64_t>(ids[k]), a.n_dim, y);
  double jac = 1.0;
#pragma unroll
  for (int d = 0; d < VEGAS_MAX_DIM; ++d) {
    int bin;
    x[d] = d < a.n_dim ? vegas_map_1d(a.edges + d * (a.n_bins + 1), a.n_bins, y[d], jac, bin) : 0.5;
  }
  double w = 0.0, rs = a.sqrt_s;
  bool ok = true;
  if (a.ps_mode == 2) {
    double msum = 0.0;
#pragma unroll
    for (int i = 0; i < NF; ++i) msum += a.masses[i];
    rs = sqrt(x[0] * x[1]) * a.sqrt_s;
    ok = rs > msum;
    if (ok) w = jac * toy_density(a.beam_kind[0], x[0]) * toy_density(a.beam_kind[1], x[1]) * rambo_event<NF>(x + 2, rs, a.masses, 1, rambo_volume(NF, rs * rs), p) *
                (PB_GEV2 / (2.0 * rs * rs));
  } else {
    w = jac * rambo_event<NF>(x, a.sqrt_s, a.masses, a.ps_mode, a.w0, p) * a.prefactor;
  }
  double* o = mom_out + k * (4 * (NF + 2));
  const double e = 0.5 * rs;
  o[0] = e; o[1] = 0.0; o[2] = 0.0; o[3] = e;
  o[4] = e; o[5] = 0.0; o[6] = 0.0; o[7] = -e;
#pragma unroll
  for (int i = 0; i < NF; ++i)
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) o[8 + 4 * i + mu] = ok ? p[i][mu] : 0.0;
  wgt_out[k] = w;
}

int check_grid(const me_handle* h, const vegas_grid* g, double sqrt_s, const char* who) {
  if (h->qed) return fail(ME_EINVAL, "%s: QCD processes only%s", who);
  const int nf = h->n_ext - 2, D = g->n_dim, nb = g->n_bins;
  if (g->ps_mode < 0 || g->ps_mode > 2 || D != (g->ps_mode == 0 ? 4 * nf : g->ps_mode == 1 ? 3 * nf - 4 : 3 * nf - 2))
    return fail(ME_EDIM, "%s: n_dim must be 4 n_final (ps_mode 0), 3 n_final - 4 (1) or 3 n_final - 2 (2)%s", who);
  if (D > VEGAS_MAX_DIM || nb < 1 || nb > VEGAS_MAX_BINS || D * nb + 3 > VEGAS_MAX_OUT)
    return fail(ME_EDIM, "%s: n_bins 1..255 and n_dim*n_bins <= 2045%s", who);
  if (!(sqrt_s > 2.0 * h->par.m_top)) return fail(ME_EINVAL, "%s: sqrt_s below threshold%s", who);
  return ME_OK;
}
void fill_args(const me_handle* h, const vegas_grid* g, double sqrt_s, long long first_event, long long n_ev, VegasArgs& a) {
  const int nf = h->n_ext - 2;
  a.edges = g->edges; a.n_dim = g->n_dim; a.n_bins = g->n_bins; a.ps_mode = g->ps_mode; a.seed = g->seed;
  a.iteration = static_cast<unsigned>(g->iteration); a.first_event = first_event; a.n_ev = n_ev; a.sqrt_s = sqrt_s;
  a.w0 = rambo_volume(nf, sqrt_s * sqrt_s); a.prefactor = PB_GEV2 / (2.0 * sqrt_s * sqrt_s);
  for (int i = 0; i < PS_MAX_FINAL; ++i) a.masses[i] = h->masses[i];
  a.gluon_mask = h->gluon_mask; a.beam_kind[0] = h->beam_kind[0]; a.beam_kind[1] = h->beam_kind[1]; a.ptj_min = h->par.ptj_min; a.dr_min = h->par.dr_min; a.mass = h->mass; a.scale = h->scale;
}

}  // namespace

extern "C" {

const char* me_last_error(void) { return g_err; }

int me_init(const char* process, const me_params* params, me_handle** out) {
  if (!process || !params || !out) return fail(ME_EINVAL, "me_init: null argument%s%s");
  *out = nullptr;
  struct Entry { const char* name; const ProcOps* (*ev)(); const ProcOps* (*vg)(); };
#define MADME_ENTRY(P) {#P, ops_##P##_eval, ops_##P##_vegas},
  static const Entry table[] = {MADME_FOR_EACH_PROCESS(MADME_ENTRY)};
#undef MADME_ENTRY
  const Entry* pe = nullptr;
  for (const Entry& e : table)
    if (!strcmp(process, e.name)) pe = &e;
  if (!pe) return fail(ME_EPROCESS, "me_init: unknown process '%s'%s", process);
  if (params->w_top != 0.0) return fail(ME_EINVAL, "me_init: w_top must be 0 (no width in propagators)%s%s");
  if (!have_device()) return fail(ME_ENODEV, "me_init: no CUDA device (this library has no CPU path)%s%s");
  me_handle* h = new me_handle();
  if (cudaGetDevice(&h->device) != cudaSuccess) { delete h; return fail(ME_ECUDA, "me_init: cudaGetDevice failed%s%s"); }
  h->ev = pe->ev();
  h->par = *params;
  // fill: the constants of the generated program (legs, masses of the final state, which final partons are jets,
  // coupling and averaging factors) and the launch geometry
  int rc = h->ev->fill(h);
  const bool qed = h->qed;
  if (rc == ME_OK && !qed) {
    h->vg = pe->vg();
    rc = h->vg->prepare(h);
  }
  if (rc == ME_OK) {
    // the fixed-size scratch of the Vegas path: sums, reduction partials, survivor staging, unweighting counters
    cudaError_t e = cudaMalloc(&h->sums_d, sizeof(double) * (VEGAS_MAX_OUT + 8));
    if (e == cudaSuccess) e = cudaMallocHost(&h->sums_h, sizeof(double) * 4);
    if (e == cudaSuccess && !qed) {
      h->partial_len = static_cast<long long>(VEGAS_MAX_CHUNKS) * VEGAS_MAX_OUT;
      e = cudaMalloc(&h->partial, sizeof(double) * h->partial_len);
      if (e == cudaSuccess) e = cudaMalloc(&h->vegas_stage, sizeof(double) * h->vegas_stage_len);
    }
    if (e != cudaSuccess) rc = cuda_fail(e, "me_init scratch");
  }
  if (rc != ME_OK) { me_free(h); return rc; }
  *out = h;
  return ME_OK;
}

void me_free(me_handle* h) {
  if (!h) return;
  DeviceGuard guard(h->device);
  if (h->block_counts) cudaFree(h->block_counts);
  if (h->f_scratch) cudaFree(h->f_scratch);
  if (h->idx_scratch) cudaFree(h->idx_scratch);
  if (h->partial) cudaFree(h->partial);
  if (h->sums_d) cudaFree(h->sums_d);
  if (h->sums_h) cudaFreeHost(h->sums_h);
  if (h->vegas_stage) cudaFree(h->vegas_stage);
  delete h;
}

int me_reserve(me_handle* h, long long max_events) {
  if (!h || max_events < 0) return fail(ME_EINVAL, "me_reserve: null handle or negative count%s%s");
  if (max_events <= h->scratch_ev) return ME_OK;
  ON_DEVICE_OF(h);
  CU(cudaDeviceSynchronize());  // earlier work may still use the buffers that are replaced
  if (h->f_scratch) cudaFree(h->f_scratch);
  if (h->idx_scratch) cudaFree(h->idx_scratch);
  if (h->block_counts) cudaFree(h->block_counts);
  h->f_scratch = nullptr; h->idx_scratch = nullptr; h->block_counts = nullptr; h->scratch_ev = 0;
  CU(cudaMalloc(&h->f_scratch, sizeof(double) * max_events));
  CU(cudaMalloc(&h->idx_scratch, sizeof(unsigned long long) * VEGAS_IDX_WORDS * max_events));
  CU(cudaMalloc(&h->block_counts, sizeof(long long) * (max_events / 256 + 2)));
  h->scratch_ev = max_events;
  return ME_OK;
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
    case 11: return h->scratch_ev;
    case 12: return h->device;
    case 13: return static_cast<long long>(reinterpret_cast<uintptr_t>(h->f_scratch));
    default: return ME_EINVAL;
  }
}
double me_flops_per_event(const me_handle* h) { return h ? h->flops : 0.0; }

static int eval_common(me_handle* h, const double* momenta, double* me2, double* hel, long long n_ev, void* stream) {
  if (!h || n_ev < 0) return fail(ME_EINVAL, "me_eval: null handle or negative n_ev%s%s");
  if (n_ev == 0) return ME_OK;  // an empty batch needs no buffers
  if (!momenta || (!me2 && !hel)) return fail(ME_EINVAL, "me_eval: null buffer%s%s");
  if (!aligned16(momenta)) return fail(ME_EINVAL, "me_eval: momenta must be 16-byte aligned%s%s");
  if (!have_device()) return fail(ME_ENODEV, "me_eval: no CUDA device%s%s");
  ON_DEVICE_OF(h);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  return h->ev->eval(h, momenta, me2, hel, n_ev, s);
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
  int rc = check_grid(h, g, sqrt_s, "vegas_integrand");
  if (rc) return rc;
  if (n_ev > h->scratch_ev) return fail(ME_EINVAL, "vegas_integrand: n_ev exceeds the reserved scratch: call me_reserve(h, n_ev) first%s%s");
  ON_DEVICE_OF(h);
  const int D = g->n_dim, nb = g->n_bins;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int n_out = 3 + D * nb, words = (D + 7) / 8;
  if (n_ev == 0) { CU(cudaMemsetAsync(sums, 0, sizeof(double) * n_out, s)); return ME_OK; }
  // fixed-shape reduction: chunk = ceil(n_ev / 1024) rounded up to a multiple of the tile -> n_chunks <= 1024
  long long chunk = (n_ev + VEGAS_MAX_CHUNKS - 1) / VEGAS_MAX_CHUNKS;
  chunk = ((chunk + VEGAS_RED_TILE - 1) / VEGAS_RED_TILE) * VEGAS_RED_TILE;
  const int n_chunks = static_cast<int>((n_ev + chunk - 1) / chunk);
  VegasArgs a;
  fill_args(h, g, sqrt_s, first_event, n_ev, a);
  double* f = f_out ? f_out : h->f_scratch;
  rc = h->vg->integrand(h, a, f, h->idx_scratch, words, s);
  if (rc) return rc;
  vegas_reduce_chunks<<<n_chunks, 512, 0, s>>>(f, h->idx_scratch, words, D, nb, n_ev, chunk, h->partial);
  CU(cudaGetLastError());
  vegas_reduce_final<<<blocks_for(n_out, 128), 128, 0, s>>>(h->partial, n_chunks, n_out, sums);
  CU(cudaGetLastError());
  return ME_OK;
}

int vegas_combine(const double* parts, int n_parts, int n_out, double* sums, void* stream) {
  if (!parts || !sums || n_parts < 1 || n_out < 1) return fail(ME_EINVAL, "vegas_combine: null pointer or empty input%s%s");
  if (!have_device()) return fail(ME_ENODEV, "vegas_combine: no CUDA device%s%s");
  vegas_reduce_final<<<blocks_for(n_out, 128), 128, 0, static_cast<cudaStream_t>(stream)>>>(parts, n_parts, n_out, sums);
  CU(cudaGetLastError());
  return ME_OK;
}

int vegas_finish(const double* sums, long long n_total, vegas_result* result, void* stream) {
  if (!sums || !result || n_total < 2) return fail(ME_EINVAL, "vegas_finish: null pointer or n_total < 2%s%s");
  if (!have_device()) return fail(ME_ENODEV, "vegas_finish: no CUDA device%s%s");
  double host[3];
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  CU(cudaMemcpyAsync(host, sums, sizeof host, cudaMemcpyDeviceToHost, s));
  CU(cudaStreamSynchronize(s));
  const double N = static_cast<double>(n_total), I = host[0] / N;
  result->integral = I;
  result->variance = (host[1] / N - I * I) / (N - 1.0);
  result->sum_w = host[0];
  result->sum_w2 = host[1];
  result->n_pass = static_cast<long long>(host[2]);
  return ME_OK;
}

int vegas_iterate(me_handle* h, vegas_grid* g, double sqrt_s, long long n_ev, vegas_result* result, void* stream) {
  if (!h || !g || !result || n_ev < 2) return fail(ME_EINVAL, "vegas_iterate: null pointer or n_ev < 2%s%s");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  int rc = vegas_integrand(h, g, sqrt_s, 0, n_ev, h->sums_d, nullptr, s);
  if (rc) return rc;
  ON_DEVICE_OF(h);
  vegas_refine_kernel<<<1, 32, 0, s>>>(g->edges, g->n_dim, g->n_bins, h->sums_d + 3, g->alpha);
  CU(cudaGetLastError());
  rc = vegas_finish(h->sums_d, n_ev, result, stream);
  if (rc) return rc;
  g->iteration += 1;
  return ME_OK;
}

int vegas_max_weight(const double* f, long long n_ev, double* w_max, void* stream) {
  if (!w_max || n_ev < 0 || (n_ev > 0 && !f)) return fail(ME_EINVAL, "vegas_max_weight: null pointer or negative count%s%s");
  if (!have_device()) return fail(ME_ENODEV, "vegas_max_weight: no CUDA device%s%s");
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  CU(cudaMemsetAsync(w_max, 0, sizeof(double), s));
  if (n_ev == 0) return ME_OK;
  const int blocks = static_cast<int>(n_ev / 256 + 1 < 1184 ? n_ev / 256 + 1 : 1184);
  max_weight_kernel<<<blocks, 256, 0, s>>>(f, n_ev, w_max);
  CU(cudaGetLastError());
  return ME_OK;
}

int vegas_unweight(me_handle* h, const double* f, long long n_ev, double w_max, uint64_t seed, uint64_t iteration, long long first_event,
                   long long* accepted, long long* counts, void* stream) {
  if (!h || !counts || n_ev < 0 || first_event < 0 || (n_ev > 0 && (!f || !accepted)))
    return fail(ME_EINVAL, "vegas_unweight: null pointer or negative count%s%s");
  if (!(w_max > 0.0)) return fail(ME_EINVAL, "vegas_unweight: w_max must be positive%s%s");
  if (n_ev > h->scratch_ev) return fail(ME_EINVAL, "vegas_unweight: n_ev exceeds the reserved scratch: call me_reserve(h, n_ev) first%s%s");
  ON_DEVICE_OF(h);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  CU(cudaMemsetAsync(counts, 0, 2 * sizeof(long long), s));
  if (n_ev == 0) return ME_OK;
  const long long n_blocks = (n_ev + 255) / 256;
  unweight_count_kernel<<<static_cast<unsigned>(n_blocks), 256, 0, s>>>(f, n_ev, w_max, seed, static_cast<unsigned>(iteration), first_event,
                                                                        h->block_counts, reinterpret_cast<unsigned long long*>(counts + 1));
  CU(cudaGetLastError());
  unweight_scan_kernel<<<1, 1024, 0, s>>>(h->block_counts, n_blocks, counts);
  CU(cudaGetLastError());
  unweight_write_kernel<<<static_cast<unsigned>(n_blocks), 256, 0, s>>>(f, n_ev, w_max, seed, static_cast<unsigned>(iteration), first_event,
                                                                        h->block_counts, accepted);
  CU(cudaGetLastError());
  return ME_OK;
}

int vegas_generate(me_handle* h, const vegas_grid* g, double sqrt_s, const long long* event_ids, long long n, double* momenta,
                   double* weights, void* stream) {
  if (!h || !g || !g->edges || n < 0 || (n > 0 && (!event_ids || !momenta || !weights)))
    return fail(ME_EINVAL, "vegas_generate: null pointer or negative count%s%s");
  int rc = check_grid(h, g, sqrt_s, "vegas_generate");
  if (rc) return rc;
  if (n == 0) return ME_OK;
  ON_DEVICE_OF(h);
  VegasArgs a;
  fill_args(h, g, sqrt_s, 0, n, a);
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  const int T = 128, B = blocks_for(n, T);
  switch (h->n_ext - 2) {
    case 2: vegas_generate_kernel<2><<<B, T, 0, s>>>(a, event_ids, n, momenta, weights); break;
    case 3: vegas_generate_kernel<3><<<B, T, 0, s>>>(a, event_ids, n, momenta, weights); break;
    case 4: vegas_generate_kernel<4><<<B, T, 0, s>>>(a, event_ids, n, momenta, weights); break;
    case 5: vegas_generate_kernel<5><<<B, T, 0, s>>>(a, event_ids, n, momenta, weights); break;
    default: return fail(ME_EINVAL, "vegas_generate: 2 to 5 final-state particles%s%s");
  }
  CU(cudaGetLastError());
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
