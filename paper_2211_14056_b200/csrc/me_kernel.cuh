// me_kernel.cuh — the me_eval kernel: a CTA of W warps evaluates W events at a time.
//
// the tensorised generator materialises every wavefunction as an HBM tensor over events and
// its footprint grows with the number of diagrams; the paper's CUDA op keeps them in per-thread storage
// (PAPER.md:70-72).  Here an event's wavefunctions live in a private slice of SHARED MEMORY (BASE + one ROUND
// region, generated/*.inc), every off-shell current is computed once per combination of the helicities of ITS OWN
// legs ("helicity recycling", me_tasks.cuh) and HBM sees 32 n_ext bytes in and 8 bytes out per event.
//
// Two mappings alternate inside the CTA (the barrier between them is __syncthreads, or __syncwarp when W = 1):
//   current stages (a5, a6): the 32 W threads share the (task row, event) pairs of the stage, W events of the same
//       row side by side on neighbouring lanes — every warp iteration runs ONE vertex routine on full lanes;
//   dot stages (a7-a10): warp w owns event w, lane = helicity combination, J (the colour-flow vector) in registers.
#pragma once
#include "generated/epem_mupmum.inc"
#include "generated/gg_ttx.inc"
#include "generated/gg_ttxg.inc"
#include "generated/gg_ttxgg.inc"

namespace madme {

// per-process tables in global memory (read through L1; a few KB, shared by every warp)
template <class P> struct Tables;
#define MADME_DEF_TABLES(P, U)                                                  \
  __device__ const MeRow U##_tasks_d[] = U##_TASK_TABLE;                        \
  __device__ const int U##_masks_d[] = U##_SUB_MASKS;                           \
  __device__ const int U##_kind_d[] = U##_LEG_KIND;                             \
  __device__ const int U##_massive_d[] = U##_LEG_MASSIVE;                       \
  __device__ const int U##_extoff_d[] = U##_EXT_OFF;                            \
  template <> struct Tables<P> {                                                \
    static __device__ __forceinline__ const MeRow* tasks() { return U##_tasks_d; }   \
    static __device__ __forceinline__ const int* masks() { return U##_masks_d; }     \
    static __device__ __forceinline__ const int* kind() { return U##_kind_d; }       \
    static __device__ __forceinline__ const int* massive() { return U##_massive_d; } \
    static __device__ __forceinline__ const int* ext_off() { return U##_extoff_d; }  \
  };
MADME_DEF_TABLES(epem_mupmum, EPEM_MUPMUM)
MADME_DEF_TABLES(gg_ttx, GG_TTX)
MADME_DEF_TABLES(gg_ttxg, GG_TTXG)
MADME_DEF_TABLES(gg_ttxgg, GG_TTXGG)

// doubles of shared memory per event: momenta [n_ext][4] + the generated scratch layout; the stride between the
// events of a CTA is = 2 doubles (16 B) mod 16 doubles (128 B), so that the same object of neighbouring events
// (neighbouring lanes in the current stages) falls into different banks.
template <class P> struct EventSmem {
  static constexpr int RAW = 4 * P::N_EXT + P::SMEM_DOUBLES;
  static constexpr int DOUBLES = ((RAW + 13) / 16) * 16 + 2;
};

template <int W> __device__ __forceinline__ void cta_sync() {
  if (W == 1) __syncwarp();
  else __syncthreads();
}

// rows [begin, end) for all W events of the CTA: item = (row, event), event fastest.  The row of the NEXT iteration is
// fetched before the current one is executed (the table is constant: its latency stays off the dependent chain); the
// loop is unrolled by two with the rows in alternating registers, so that no register copy waits on the fetch.
__device__ __forceinline__ void run_row(const uint4 q, double* sm, double mass) {
  MeRow r;
  r.x = q.x; r.y = q.y; r.z = q.z; r.w = q.w;
  me_run_row(r, sm, mass);
}
// `first` holds this thread's first row of the stage on entry (fetched during the previous stage) and of the NEXT
// stage on return (stages are multiples of 32 rows, so that row is end + t / W): its latency hides behind the barrier
// and the dot products in between.
template <int W>
__device__ __forceinline__ void run_rows(const uint4* __restrict__ tab, int begin, int end, int n_rows, double* smem, int ev_stride,
                                         double mass, uint4& first) {
  const int t = threadIdx.x;
  const int ev = t % W;
  double* sm = smem + ev * ev_stride;
  int row = begin + t / W;
  uint4 a = first;
  first = __ldg(tab + min(end + t / W, n_rows));
  if (row >= end) return;
#pragma unroll 1
  for (;;) {
    const uint4 b = __ldg(tab + min(row + 32, n_rows));
    run_row(a, sm, mass);
    row += 32;
    if (row >= end) break;
    a = __ldg(tab + min(row + 32, n_rows));
    run_row(b, sm, mass);
    row += 32;
    if (row >= end) break;
  }
}

// |M|^2 of the W events whose momenta sit at the head of each event slice ([n_ext][4]).  Returns, on every lane of
// warp w, the helicity- and colour-summed, averaged value of event w.  hel_out (optional, global [N_HEL], per warp)
// receives each helicity combination's share.
template <class P, int W>
__device__ __forceinline__ double cta_me2(double* smem, double mass, double scale, double* hel_out) {
  constexpr int STRIDE = EventSmem<P>::DOUBLES;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const uint4* tab = reinterpret_cast<const uint4*>(Tables<P>::tasks());
  // a5: subset momenta / denominators and external wavefunctions, items = (subset or leg, event)
  {
    const int t = threadIdx.x, ev = t % W;
    double* mom_s = smem + ev * STRIDE;
    me_phase0(t / W, 32, mom_s + 4 * P::N_EXT, mom_s, P::N_EXT, P::N_SUB, Tables<P>::masks(), Tables<P>::kind(),
              Tables<P>::massive(), Tables<P>::ext_off(), mass);
  }
  cta_sync<W>();
  double* base = smem + 4 * P::N_EXT;  // event e's scratch = base + e * STRIDE
  static_assert(P::N_HEL_EVAL <= 32, "one helicity combination per lane");
  double jr[P::N_FLOW], ji[P::N_FLOW];
#pragma unroll
  for (int f = 0; f < P::N_FLOW; ++f) { jr[f] = 0.0; ji[f] = 0.0; }
  const double* my = base + warp * STRIDE;
  int row = 0;
  uint4 first = __ldg(tab + threadIdx.x / W);
  // ONE copy of the row interpreter and one of each round's dot products in the instruction stream: the phase loop
  // must stay rolled (unrolled it is > 600 KB of SASS and the kernel starves on instruction fetch)
#pragma unroll 1
  for (int p = 0; p < P::N_PHASES; ++p) {
    const int end = P::phase_end(p);
    run_rows<W>(tab, row, end, P::N_ROWS, base, STRIDE, mass, first);
    row = end;
    cta_sync<W>();
    const int r = P::phase_dots(p);
    if (r >= 0) {
      if (lane < P::N_HEL_EVAL) P::dots(r, my, lane, jr, ji);
      cta_sync<W>();
    }
  }
  double v = (lane < P::N_HEL_EVAL) ? P::colour(jr, ji) : 0.0;
  if (hel_out && lane < P::N_HEL_EVAL) {  // full index: leg 0 at +1 is bit 0; the parity partner has every helicity flipped
    const int hf = (lane << 1) | 1;
    hel_out[hf] = v * scale;
    hel_out[(P::N_HEL - 1) ^ hf] = v * scale;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return 2.0 * v * scale;
}

// W events per CTA (blockDim.x = 32 W); persistent grid, batches of W consecutive events.  MADME_OCC_WARPS is the number
// of resident warps per SM the register allocation is bounded for (8 -> up to 255 registers, 12 -> 168).
#ifndef MADME_OCC_WARPS
#define MADME_OCC_WARPS 8
#endif
template <class P, int W>
__global__ void __launch_bounds__(32 * W, (MADME_OCC_WARPS + W - 1) / W) me_eval_kernel(const double* __restrict__ momenta, double* __restrict__ me2,
                                                         double* __restrict__ me2_hel, long long n_ev, double mass, double scale) {
  extern __shared__ __align__(16) double smem[];
  constexpr int STRIDE = EventSmem<P>::DOUBLES;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long n_batches = (n_ev + W - 1) / W;
  for (long long b = blockIdx.x; b < n_batches; b += gridDim.x) {
    // events past the end repeat the last one (computed, not stored)
    const long long ev = min(b * W + warp, n_ev - 1);
    if (lane < 4 * P::N_EXT) smem[warp * STRIDE + lane] = momenta[ev * (4 * P::N_EXT) + lane];
    cta_sync<W>();
    const double r = cta_me2<P, W>(smem, mass, scale, (me2_hel && b * W + warp < n_ev) ? me2_hel + ev * P::N_HEL : nullptr);
    if (lane == 0 && me2 && b * W + warp < n_ev) me2[ev] = r;
    cta_sync<W>();
  }
}

}  // namespace madme
