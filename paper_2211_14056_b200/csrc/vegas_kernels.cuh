// vegas_kernels.cuh — the fused integrand kernel (steps a1-a11 up to the per-event weight).
// BASELINE.json:configs[4]: "fused RAMBO + Vegas map + me_eval".
#pragma once
#include "me_kernel.cuh"
#include "vegas_common.cuh"

namespace madme {

// Fused integrand.  A CTA of NW warps takes 32 NW consecutive events: every thread generates one event (Philox -> Vegas
// map -> RAMBO -> cuts).  The survivors are COMPACTED across the CTA (ballot + prefix sum) into a small per-CTA staging
// area (final-state momenta, weight, event index: 32 W x (4 n_final + 2) doubles of global memory that never leaves
// L2) so that the CTA then evaluates |M|^2 of exactly the surviving events, W at a time, whatever warp generated them;
// cut events cost no matrix element.  Output per event: f (8 B) and the D bin indices packed one byte each
// (n_bins <= 255) into idx_out[ev][ceil(D/8)].
// One event of the stream: Philox -> Vegas map -> RAMBO -> cuts (steps a1-a4).  Writes the packed bin indices of the
// event; returns whether it passes the cuts, its final-state momenta p, the weight w without |M|^2 and sqrt(s_hat).
// NOT inlined: the prologue keeps 8 momenta, 24 uniforms and 24 mapped coordinates live, and inlined into the kernel it
// made ptxas spill inside the matrix-element part (724 B); as a function it has its own register allocation.
template <int NF>
__device__ __noinline__ bool vegas_generate_one(const VegasArgs& a, long long ev, unsigned long long* __restrict__ idx_out, int idx_words,
                                                double (&p)[NF][4], double& w, double& rs) {
  double y[VEGAS_MAX_DIM], x[VEGAS_MAX_DIM];
  unsigned long long packed[VEGAS_IDX_WORDS] = {};   // one byte per dimension
  bool pass = false;
  w = 0.0;
  rs = a.sqrt_s;
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
  if (a.ps_mode == 2) {
    // hadronic mode (DESIGN.md R-N3): x[0], x[1] are the momentum fractions, the rest drives RAMBO on diet at sqrt(s_hat)
    double msum = 0.0;
#pragma unroll
    for (int i = 0; i < NF; ++i) msum += a.masses[i];
    rs = sqrt(x[0] * x[1]) * a.sqrt_s;
    if (rs > msum) {
      const double wps = rambo_event<NF>(x + 2, rs, a.masses, 1, rambo_volume(NF, rs * rs), p);
      pass = passes_cuts<NF>(p, a.gluon_mask, a.ptj_min, a.dr_min);
      w = jac * toy_density(a.beam_kind[0], x[0]) * toy_density(a.beam_kind[1], x[1]) * wps * (PB_GEV2 / (2.0 * rs * rs));
    }
  } else {
    const double wps = rambo_event<NF>(x, a.sqrt_s, a.masses, a.ps_mode, a.w0, p);
    pass = passes_cuts<NF>(p, a.gluon_mask, a.ptj_min, a.dr_min);
    w = jac * wps * a.prefactor;
  }
  for (int k = 0; k < idx_words; ++k) idx_out[ev * idx_words + k] = packed[k];
  return pass;
}

template <class P>
__global__ void __launch_bounds__(32 * P::N_WARPS, 1) vegas_integrand_kernel(VegasArgs a, double* __restrict__ f_out,
                                                                 unsigned long long* __restrict__ idx_out, int idx_words,
                                                                 double* __restrict__ stage_all) {
  constexpr int NF = P::N_EXT - 2, W = P::W_EVENTS, NW = P::N_WARPS;
  constexpr int STRIDE = EventSmem<P>::DOUBLES;
  constexpr int SLOT = 4 * NF + 4;  // final momenta, weight, event index, beam energy, pad
  extern __shared__ __align__(16) double smem[];
  __shared__ int warp_count[NW];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double* mom_s = smem + warp * STRIDE;
  double* stage = stage_all + static_cast<long long>(blockIdx.x) * (32 * NW) * SLOT;
  const uint32_t tmem = JPark<P>::ON ? tmem_alloc<JPark<P>::COLS>() : 0u;
  const long long n_batches = (a.n_ev + 32 * NW - 1) / (32 * NW);
  for (long long b = blockIdx.x; b < n_batches; b += gridDim.x) {
    const long long ev = (b * NW + warp) * 32 + lane;
    const bool live = ev < a.n_ev;
    {
      double p[NF][4];
      bool pass = false;
      double w = 0.0, rs = a.sqrt_s;
      if (live) {
        pass = vegas_generate_one<NF>(a, ev, idx_out, idx_words, p, w, rs);
        if (!pass) f_out[ev] = 0.0;
      }
      // compaction: position of this survivor among the CTA's survivors, in event order
      const unsigned mask = __ballot_sync(0xffffffffu, pass);
      if (lane == 0) warp_count[warp] = __popc(mask);
      __syncthreads();
      int pos = __popc(mask & ((1u << lane) - 1u));
      for (int k = 0; k < warp; ++k) pos += warp_count[k];
      if (pass) {
        double* s = stage + pos * SLOT;
#pragma unroll
        for (int i = 0; i < NF; ++i)
#pragma unroll
          for (int mu = 0; mu < 4; ++mu) s[4 * i + mu] = p[i][mu];
        s[4 * NF] = w;
        s[4 * NF + 1] = __longlong_as_double(ev);
        s[4 * NF + 2] = 0.5 * rs;
      }
    }
    int n_pass = 0;
#pragma unroll
    for (int k = 0; k < NW; ++k) n_pass += warp_count[k];
    __syncthreads();  // staging writes visible to the CTA
    for (int first = 0; first < n_pass; first += W) {
      const bool valid = (NW == W || warp < W) && first + warp < n_pass;   // warps >= W only help with the items
      const double* s = stage + (valid ? first + warp : 0) * SLOT;  // idle warps re-evaluate slot 0 (finite input, not stored)
      const double e_beam = s[4 * NF + 2];
      if (NW == W || warp < W) {
        if (lane < 8) mom_s[lane] = (lane == 0 || lane == 3 || lane == 4) ? e_beam : (lane == 7 ? -e_beam : 0.0);
        else if (lane < 8 + 4 * NF) mom_s[lane] = s[lane - 8];
      }
      __syncthreads();
      const double r = cta_me2<P>(smem, a.mass, a.scale, nullptr, tmem);
      if (valid && lane == 0) f_out[__double_as_longlong(s[4 * NF + 1])] = s[4 * NF] * r;
      __syncthreads();
    }
    __syncthreads();  // the staging area and warp_count are reused by the next batch
  }
  if (JPark<P>::ON) tmem_free<JPark<P>::COLS>(tmem);
}

}  // namespace madme
