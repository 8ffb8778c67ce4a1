// unweight_static.cu — vegas_unweight_static: the hit-or-miss unweighting of vegas_unweight (DESIGN.md
// R-N4) for callers that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc.  vegas_unweight keeps its scratch (kept events per 256-event block) in a buffer that me_reserve sizes with
// cudaMalloc; this variant keeps it in a FILE-SCOPE device array of fixed size, so that the entry point needs no handle, no
// me_reserve and calls no cudaMalloc, cudaFree or allocating library routine.  The price:
//   * at most VEGAS_UNWEIGHT_STATIC_MAX_EVENTS (2^22) events per call; larger calls are rejected with ME_EINVAL;
//   * every GPU that loads the library holds the array (128 KB + 16 B) until the process exits;
//   * every call on a device shares the one array, which keeps the last call's contents: calls that overlap on the GPU
//     (different streams, or a captured graph replayed while another call runs) RACE.  One call at a time per device.
// Nothing in the array has to start at zero: pass 1 writes every entry that passes 2 and 3 read.  counts[] is the
// caller's and is cleared by the call (a memset node under capture).
// The existing path (madme.cu::vegas_unweight) is untouched; tests/test_zz_no_alloc.py holds the two to the same output.
#include "common.cuh"
#include "phase_space.cuh"

using namespace madme;

namespace {

constexpr long long MAX_EVENTS = VEGAS_UNWEIGHT_STATIC_MAX_EVENTS;
constexpr int BLOCK = 256;
constexpr long long MAX_BLOCKS = (MAX_EVENTS + BLOCK - 1) / BLOCK;
constexpr int MAX_DEVICES = 64;

// The scratch.  In HOST code this name is a host-side stand-in, not a device address: the address a kernel may use comes
// from cudaGetSymbolAddress (static_init below), once per device, with that device current.
static __device__ __align__(256) long long g_block_counts[MAX_BLOCKS + 2];

long long* g_scratch_of_device[MAX_DEVICES] = {};   // device address of g_block_counts on each device, 0 = not set up

// the decision of DESIGN.md R-N4: kept iff f > 0 and u w_max < f, u = Philox uniform of counter (event lo, event hi,
// 0x7fffffff, iteration), words 0-1
__device__ __forceinline__ bool keep_event(double f, double w_max, unsigned long long seed, unsigned iteration, long long event) {
  if (!(f > 0.0)) return false;
  const uint4 w = philox4x32_10(make_uint4(static_cast<uint32_t>(event), static_cast<uint32_t>(static_cast<unsigned long long>(event) >> 32),
                                           0x7fffffffu, iteration),
                                make_uint2(static_cast<uint32_t>(seed), static_cast<uint32_t>(seed >> 32)));
  return philox_u01(w.x, w.y) * w_max < f;
}

// pass 1: kept events of each 256-event block -> scratch[block]; events above w_max counted into counts[1]
__global__ void __launch_bounds__(BLOCK) static_count_kernel(const double* __restrict__ f, long long n_ev, double w_max, unsigned long long seed,
                                                             unsigned iteration, long long first_event, long long* __restrict__ scratch,
                                                             unsigned long long* __restrict__ n_over) {
  const long long e = static_cast<long long>(blockIdx.x) * BLOCK + threadIdx.x;
  const double v = e < n_ev ? f[e] : 0.0;
  const bool keep = e < n_ev && keep_event(v, w_max, seed, iteration, first_event + e);
  const int c = __syncthreads_count(keep);
  const int o = __syncthreads_count(e < n_ev && v > w_max);
  if (threadIdx.x == 0) {
    scratch[blockIdx.x] = c;
    if (o) atomicAdd(n_over, static_cast<unsigned long long>(o));
  }
}
// pass 2 (one block): exclusive scan of scratch[0 .. n_blocks) in place, total -> counts[0]
__global__ void __launch_bounds__(1024) static_scan_kernel(long long* __restrict__ scratch, long long n_blocks, long long* __restrict__ counts) {
  __shared__ long long part[1024];
  const long long per = (n_blocks + 1023) / 1024, lo = threadIdx.x * per, hi = min(n_blocks, lo + per);
  long long s = 0;
  for (long long i = lo; i < hi; ++i) s += scratch[i];
  part[threadIdx.x] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    long long run = 0;
    for (int i = 0; i < 1024; ++i) { const long long t = part[i]; part[i] = run; run += t; }
    counts[0] = run;
  }
  __syncthreads();
  long long run = part[threadIdx.x];
  for (long long i = lo; i < hi; ++i) { const long long t = scratch[i]; scratch[i] = run; run += t; }
}
// pass 3: the global indices of the kept events, in ascending order
__global__ void __launch_bounds__(BLOCK) static_write_kernel(const double* __restrict__ f, long long n_ev, double w_max, unsigned long long seed,
                                                             unsigned iteration, long long first_event, const long long* __restrict__ offsets,
                                                             long long* __restrict__ accepted) {
  __shared__ int warp_count[BLOCK / 32];
  const long long e = static_cast<long long>(blockIdx.x) * BLOCK + threadIdx.x;
  const bool keep = e < n_ev && keep_event(f[e], w_max, seed, iteration, first_event + e);
  const unsigned mask = __ballot_sync(0xffffffffu, keep);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) warp_count[warp] = __popc(mask);
  __syncthreads();
  if (keep) {
    long long pos = offsets[blockIdx.x] + __popc(mask & ((1u << lane) - 1u));
    for (int k = 0; k < warp; ++k) pos += warp_count[k];
    accepted[pos] = first_event + e;
  }
}

bool device_present() {
  int n = 0;
  const bool ok = cudaGetDeviceCount(&n) == cudaSuccess && n > 0;
  if (!ok) (void)cudaGetLastError();
  return ok;
}

// the device address of the scratch on the CURRENT device (set-up, once per device)
int static_init(long long** out) {
  int dev = 0;
  CU(cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEVICES) return fail(ME_EINVAL, "vegas_unweight_static: device ordinal beyond 63%s%s");
  if (!g_scratch_of_device[dev]) {
    long long* p = nullptr;
    CU(cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_block_counts));
    if (!p) return fail(ME_ECUDA, "vegas_unweight_static: cudaGetSymbolAddress returned a null address%s%s");
    g_scratch_of_device[dev] = p;
  }
  if (out) *out = g_scratch_of_device[dev];
  return ME_OK;
}

}  // namespace

extern "C" {

int vegas_unweight_static_init(void) {
  if (!device_present()) return fail(ME_ENODEV, "vegas_unweight_static_init: no CUDA device%s%s");
  return static_init(nullptr);
}

int vegas_unweight_static(const double* f, long long n_ev, double w_max, uint64_t seed, uint64_t iteration, long long first_event,
                          long long* accepted, long long* counts, void* stream) {
  if (!counts || n_ev < 0 || first_event < 0 || (n_ev > 0 && (!f || !accepted)))
    return fail(ME_EINVAL, "vegas_unweight_static: null pointer or negative count%s%s");
  if (!(w_max > 0.0)) return fail(ME_EINVAL, "vegas_unweight_static: w_max must be positive%s%s");
  if (n_ev > MAX_EVENTS)
    return fail(ME_EINVAL, "vegas_unweight_static: n_ev exceeds VEGAS_UNWEIGHT_STATIC_MAX_EVENTS (4194304): split the call or use vegas_unweight%s%s");
  if (!device_present()) return fail(ME_ENODEV, "vegas_unweight_static: no CUDA device%s%s");
  long long* scratch = nullptr;
  const int rc = static_init(&scratch);   // a table look-up after the first call on this device
  if (rc) return rc;
  cudaStream_t s = static_cast<cudaStream_t>(stream);
  CU(cudaMemsetAsync(counts, 0, 2 * sizeof(long long), s));
  if (n_ev == 0) return ME_OK;
  const long long n_blocks = (n_ev + BLOCK - 1) / BLOCK;
  static_count_kernel<<<static_cast<unsigned>(n_blocks), BLOCK, 0, s>>>(f, n_ev, w_max, seed, static_cast<unsigned>(iteration), first_event, scratch,
                                                                        reinterpret_cast<unsigned long long*>(counts + 1));
  CU(cudaGetLastError());
  static_scan_kernel<<<1, 1024, 0, s>>>(scratch, n_blocks, counts);
  CU(cudaGetLastError());
  static_write_kernel<<<static_cast<unsigned>(n_blocks), BLOCK, 0, s>>>(f, n_ev, w_max, seed, static_cast<unsigned>(iteration), first_event, scratch,
                                                                        accepted);
  CU(cudaGetLastError());
  return ME_OK;
}

}  // extern "C"
