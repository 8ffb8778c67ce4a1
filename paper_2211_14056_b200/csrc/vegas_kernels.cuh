// vegas_kernels.cuh — the fused integrand kernel (steps a1-a11 up to the per-event weight).
// BASELINE.json:configs[4]: "fused RAMBO + Vegas map + me_eval".
#pragma once
#include "me_kernel.cuh"
#include "vegas_common.cuh"

namespace madme {

// Fused integrand.  A CTA of W warps takes 32 W consecutive events: every thread generates one event (Philox -> Vegas
// map -> RAMBO -> cuts), then the CTA evaluates |M|^2 of the surviving events W at a time (cta_me2: warp w supplies
// its next surviving event, momenta handed over by shuffles) — nothing goes through HBM in between.
// Output per event: f (8 B) and the D bin indices packed one byte each (n_bins <= 255) into idx_out[ev][ceil(D/8)].
template <class P, int W>
__global__ void __launch_bounds__(32 * W) vegas_integrand_kernel(VegasArgs a, double* __restrict__ f_out,
                                                                 unsigned long long* __restrict__ idx_out, int idx_words) {
  constexpr int NF = P::N_EXT - 2;
  constexpr int STRIDE = EventSmem<P>::DOUBLES;
  extern __shared__ __align__(16) double smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double* mom_s = smem + warp * STRIDE;
  const long long n_batches = (a.n_ev + 32 * W - 1) / (32 * W);
  const double e_beam = 0.5 * a.sqrt_s;
  for (long long b = blockIdx.x; b < n_batches; b += gridDim.x) {
    const long long ev = (b * W + warp) * 32 + lane;
    const bool live = ev < a.n_ev;
    double p[NF][4];
    unsigned long long packed[2] = {0ull, 0ull};
    double w = 0.0;
    bool pass = false;
    {
      // events past the end are generated too (valid momenta for the shared evaluation) but neither pass nor store
      double y[VEGAS_MAX_DIM], x[VEGAS_MAX_DIM];
      philox_fill<VEGAS_MAX_DIM>(a.seed, a.iteration, static_cast<uint64_t>(a.first_event + ev), a.n_dim, y);
      double jac = 1.0;
#pragma unroll
      for (int d = 0; d < VEGAS_MAX_DIM; ++d) {
        if (d < a.n_dim) {
          int bin;
          x[d] = vegas_map_1d(a.edges + d * (a.n_bins + 1), a.n_bins, y[d], jac, bin);
          packed[d >> 3] |= static_cast<unsigned long long>(bin) << (8 * (d & 7));
        } else {
          x[d] = 0.5;
        }
      }
      const double wps = rambo_event<NF>(x, a.sqrt_s, a.masses, a.ps_mode, a.w0, p);
      pass = live && passes_cuts<NF>(p, a.gluon_mask, a.ptj_min, a.dr_min);
      w = jac * wps;
    }
    unsigned rest = __ballot_sync(0xffffffffu, pass);
    double me2_mine = 0.0;
    // every slot starts with a valid event (lane 0's), so that a warp that runs out of survivors still feeds
    // finite numbers to the shared current stages
    int src = 0;
    for (;;) {
      const bool more = rest != 0u;
      if (W == 1) { if (!more) break; }
      else if (!__syncthreads_or(more ? 1 : 0)) break;
      if (more) src = __ffs(rest) - 1;
      if (lane < 8) mom_s[lane] = (lane == 0 || lane == 3 || lane == 4) ? e_beam : (lane == 7 ? -e_beam : 0.0);
#pragma unroll
      for (int i = 0; i < NF; ++i)
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
          const double v = __shfl_sync(0xffffffffu, p[i][mu], src);
          if (lane == 8 + 4 * i + mu) mom_s[8 + 4 * i + mu] = v;
        }
      cta_sync<W>();
      const double r = cta_me2<P, W>(smem, a.mass, a.scale, nullptr);
      if (more && lane == src) me2_mine = r;
      rest &= rest - 1u;
      cta_sync<W>();
    }
    if (live) {
      const double f = pass ? w * me2_mine * a.prefactor : 0.0;
      f_out[ev] = f;
      for (int k = 0; k < idx_words; ++k) idx_out[ev * idx_words + k] = packed[k];
    }
  }
}

}  // namespace madme
