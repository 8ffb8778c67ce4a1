// me_kernel.cuh — the me_eval kernel: one warp per event, one helicity combination per lane per pass.
//
// the tensorised generator materialises every wavefunction as an HBM tensor over events and
// its footprint grows with the number of diagrams; the paper's CUDA op keeps them in per-thread storage
// (PAPER.md:70-72).  Here the event's wavefunctions live in the warp's private slice of SHARED MEMORY, every
// off-shell current is computed once per combination of the helicities of ITS OWN legs ("helicity recycling",
// me_tasks.cuh) and HBM sees 32 n_ext bytes in and 8 bytes out per event.
//
// Steps: a5 me_phase0 -> a6 P::stage(s) -> a7-a9 P::closings(h) per lane -> a10 warp sum (x2: parity).
#pragma once
#include "generated/epem_mupmum.inc"
#include "generated/gg_ttx.inc"
#include "generated/gg_ttxg.inc"
#include "generated/gg_ttxgg.inc"

namespace madme {

// per-process tables in global memory (read through L1; a few KB, shared by every warp)
template <class P> struct Tables;
#define MADME_DEF_TABLES(P, U)                                                  \
  __device__ const int U##_tasks_d[] = U##_TASK_TABLE;                          \
  __device__ const int U##_combos_d[] = U##_COMBO_TABLE;                        \
  __device__ const int U##_masks_d[] = U##_SUB_MASKS;                           \
  __device__ const int U##_kind_d[] = U##_LEG_KIND;                             \
  __device__ const int U##_massive_d[] = U##_LEG_MASSIVE;                       \
  __device__ const int U##_extoff_d[] = U##_EXT_OFF;                            \
  template <> struct Tables<P> {                                                \
    static __device__ __forceinline__ const int* tasks() { return U##_tasks_d; }     \
    static __device__ __forceinline__ const int* combos() { return U##_combos_d; }   \
    static __device__ __forceinline__ const int* masks() { return U##_masks_d; }     \
    static __device__ __forceinline__ const int* kind() { return U##_kind_d; }       \
    static __device__ __forceinline__ const int* massive() { return U##_massive_d; } \
    static __device__ __forceinline__ const int* ext_off() { return U##_extoff_d; }  \
  };
MADME_DEF_TABLES(epem_mupmum, EPEM_MUPMUM)
MADME_DEF_TABLES(gg_ttx, GG_TTX)
MADME_DEF_TABLES(gg_ttxg, GG_TTXG)
MADME_DEF_TABLES(gg_ttxgg, GG_TTXGG)

// doubles of shared memory per event: momenta [n_ext][4] + the generated scratch layout, 16-byte aligned
template <class P> struct EventSmem { static constexpr int DOUBLES = ((4 * P::N_EXT + P::SMEM_DOUBLES + 1) / 2) * 2; };

template <class P> __device__ __forceinline__ void run_stages(int lane, double* sm, double mass) {
  const int* tab = Tables<P>::tasks();
  const int* ctab = Tables<P>::combos();
#pragma unroll
  for (int s = 0; s < P::N_STAGES; ++s) {
    P::stage(s, lane, sm, tab, ctab, mass);
    __syncwarp();
  }
}

// |M|^2 of the event whose momenta sit in mom_s (shared, [n_ext][4]); every lane returns the helicity-summed,
// colour-summed, averaged value.  hel_out (optional, global [N_HEL]) receives each combination's share.
template <class P>
__device__ __forceinline__ double warp_me2(int lane, double* sm, const double* mom_s, double mass, double scale, double* hel_out) {
  me_phase0(lane, sm, mom_s, P::N_EXT, P::N_SUB, Tables<P>::masks(), Tables<P>::kind(), Tables<P>::massive(),
            Tables<P>::ext_off(), mass);
  __syncwarp();
  run_stages<P>(lane, sm, mass);
  double s = 0.0;
  for (int h = lane; h < P::N_HEL_EVAL; h += 32) {
    const double v = P::closings(sm, h);
    if (hel_out) {  // full index: leg 0 at +1 is bit 0; the parity partner has every helicity flipped
      const int hf = (h << 1) | 1;
      hel_out[hf] = v * scale;
      hel_out[(P::N_HEL - 1) ^ hf] = v * scale;
    }
    s += v;
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  return 2.0 * s * scale;
}

// MAXWARPS bounds the CTA size (register budget); the actual events-per-CTA is blockDim.x / 32 (a run-time knob:
// the threads-per-block scan of PAPER.md:78-84, Fig. 3, is repeated with MADME_WARPS).
template <class P, int MAXWARPS>
__global__ void __launch_bounds__(MAXWARPS * 32) me_eval_kernel(const double* __restrict__ momenta, double* __restrict__ me2,
                                                              double* __restrict__ me2_hel, long long n_ev, double mass,
                                                              double scale) {
  extern __shared__ __align__(16) double smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, warps = blockDim.x >> 5;
  double* mom_s = smem + warp * EventSmem<P>::DOUBLES;
  double* sm = mom_s + 4 * P::N_EXT;
  for (long long ev = static_cast<long long>(blockIdx.x) * warps + warp; ev < n_ev;
       ev += static_cast<long long>(gridDim.x) * warps) {
    if (lane < 4 * P::N_EXT) mom_s[lane] = momenta[ev * (4 * P::N_EXT) + lane];
    __syncwarp();
    const double r = warp_me2<P>(lane, sm, mom_s, mass, scale, me2_hel ? me2_hel + ev * P::N_HEL : nullptr);
    if (lane == 0 && me2) me2[ev] = r;
    __syncwarp();
  }
}

}  // namespace madme
