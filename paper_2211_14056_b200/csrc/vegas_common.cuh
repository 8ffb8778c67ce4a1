// vegas_common.cuh — what the fused integrand kernel (vegas_kernels.cuh) and the C ABI (madme.cu) share: the argument
// block, and the deterministic reduction (a11) and grid-refinement (a12) kernels of vegas_iterate.
// Vegas with "the events ... computed in parallel"; BASELINE.json:configs[4]: "weighted accumulation
// and grid refinement on device".  Grid-update details are DESIGN.md readings R-G7.
#pragma once
#include "phase_space.cuh"

namespace madme {

constexpr int VEGAS_MAX_DIM = 4 * PS_MAX_FINAL;
constexpr int VEGAS_IDX_WORDS = (VEGAS_MAX_DIM + 7) / 8;   // bin indices packed one byte per dimension
constexpr double PB_GEV2 = 0.3893793721e9;  // (hbar c)^2 in pb GeV^2

struct VegasArgs {
  const double* edges;  // dev [n_dim][n_bins+1]
  int n_dim, n_bins, ps_mode;
  unsigned long long seed;
  unsigned iteration;
  long long first_event, n_ev;
  double sqrt_s, w0, prefactor;  // prefactor = C / (2 s)
  double masses[PS_MAX_FINAL];
  unsigned gluon_mask;
  int beam_kind[2];  // hadronic mode: the toy density of each beam (0 gluon, 1 quark, 2 antiquark)
  double ptj_min, dr_min, mass, scale;
};

// a11, deterministic: block c owns the contiguous event chunk [c*chunk, (c+1)*chunk); output entry j (j = 0,1,2: sum f,
// sum f^2, pass count; j = 3 + d*n_bins + i: histogram cell (d, i)) is owned by thread j % 512 and receives the chunk's
// events in event order.  partial: [gridDim.x][3 + n_dim*n_bins].  Up to VEGAS_RED_PER_THREAD entries per thread.
constexpr int VEGAS_RED_TILE = 1024;
constexpr int VEGAS_RED_PER_THREAD = 4;
static __global__ void __launch_bounds__(512) vegas_reduce_chunks(const double* __restrict__ f, const unsigned long long* __restrict__ idx,
                                                           int idx_words, int n_dim, int n_bins, long long n_ev, long long chunk,
                                                           double* __restrict__ partial) {
  __shared__ double f_s[VEGAS_RED_TILE];
  __shared__ unsigned long long idx_s[VEGAS_IDX_WORDS * VEGAS_RED_TILE];
  const int n_out = n_dim * n_bins + 3, t = threadIdx.x;
  const long long begin = blockIdx.x * chunk, end = min(n_ev, begin + chunk);
  double acc[VEGAS_RED_PER_THREAD];
  int word[VEGAS_RED_PER_THREAD], shift[VEGAS_RED_PER_THREAD], bin[VEGAS_RED_PER_THREAD];
#pragma unroll
  for (int k = 0; k < VEGAS_RED_PER_THREAD; ++k) {
    acc[k] = 0.0;
    const int j = t + 512 * k, cell = j - 3;
    const int d = cell >= 0 ? cell / n_bins : 0;
    word[k] = d >> 3;
    shift[k] = 8 * (d & 7);
    bin[k] = cell >= 0 ? cell - d * n_bins : -1;
  }
  for (long long base = begin; base < end; base += VEGAS_RED_TILE) {
    const long long left = end - base;
    const int n = left < VEGAS_RED_TILE ? static_cast<int>(left) : VEGAS_RED_TILE;
    for (int e = t; e < n; e += blockDim.x) {
      f_s[e] = f[base + e];
      for (int k = 0; k < idx_words; ++k) idx_s[e * idx_words + k] = idx[(base + e) * idx_words + k];
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < VEGAS_RED_PER_THREAD; ++k) {
      const int j = t + 512 * k;
      if (j >= n_out) continue;
      double a = acc[k];
      if (j == 0) {
        for (int e = 0; e < n; ++e) a += f_s[e];
      } else if (j == 1) {
        for (int e = 0; e < n; ++e) a += f_s[e] * f_s[e];
      } else if (j == 2) {
        for (int e = 0; e < n; ++e) a += (f_s[e] != 0.0) ? 1.0 : 0.0;
      } else {
        for (int e = 0; e < n; ++e) {
          const double v = f_s[e];
          if (static_cast<int>((idx_s[e * idx_words + word[k]] >> shift[k]) & 0xffull) == bin[k]) a += v * v;
        }
      }
      acc[k] = a;
    }
    __syncthreads();
  }
#pragma unroll
  for (int k = 0; k < VEGAS_RED_PER_THREAD; ++k) {
    const int j = t + 512 * k;
    if (j < n_out) partial[static_cast<long long>(blockIdx.x) * n_out + j] = acc[k];
  }
}
// second stage: entry j of sums = partial[0][j] + partial[1][j] + ... in chunk order
static __global__ void vegas_reduce_final(const double* __restrict__ partial, int n_chunks, int n_out, double* __restrict__ sums) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n_out) return;
  double acc = 0.0;
  for (int c = 0; c < n_chunks; ++c) acc += partial[static_cast<long long>(c) * n_out + j];
  sums[j] = acc;
}

// a12: grid refinement, one thread per dimension (n_dim * n_bins = 400 numbers: latency, not throughput).
// smooth (3-point), normalise, damp w = [(r-1)/ln r]^alpha, then walk the cumulative damped weight so that every
// new bin holds the same share, interpolating linearly inside old bins; end points stay exactly 0 and 1.
constexpr int VEGAS_MAX_BINS = 255;
static __global__ void vegas_refine_kernel(double* __restrict__ edges, int n_dim, int n_bins, const double* __restrict__ S, double alpha) {
  const int d = blockIdx.x * blockDim.x + threadIdx.x;
  if (d >= n_dim || n_bins < 2) return;
  double* e = edges + static_cast<long long>(d) * (n_bins + 1);
  const double* Sd = S + static_cast<long long>(d) * n_bins;
  double w[VEGAS_MAX_BINS], ne[VEGAS_MAX_BINS + 1];
  double tot = 0.0;
  for (int i = 0; i < n_bins; ++i) {
    double s;
    if (i == 0) s = (Sd[0] + Sd[1]) / 2.0;
    else if (i == n_bins - 1) s = (Sd[n_bins - 2] + Sd[n_bins - 1]) / 2.0;
    else s = (Sd[i - 1] + Sd[i] + Sd[i + 1]) / 3.0;
    w[i] = s;
    tot += s;
  }
  if (!(tot > 0.0)) return;
  double wtot = 0.0;
  for (int i = 0; i < n_bins; ++i) {
    const double r = w[i] / tot;
    double v;
    if (r <= 0.0) v = 0.0;
    else if (r == 1.0) v = 1.0;
    else v = pow((r - 1.0) / log(r), alpha);
    w[i] = v;
    wtot += v;
  }
  const double target = wtot / n_bins;
  int j = 0;
  double acc = 0.0;
  ne[0] = 0.0;
  ne[n_bins] = 1.0;
  for (int i = 1; i < n_bins; ++i) {
    const double need = i * target;
    while (j < n_bins - 1 && acc + w[j] < need) { acc += w[j]; ++j; }
    const double frac = (w[j] > 0.0) ? (need - acc) / w[j] : 0.0;
    ne[i] = e[j] + frac * (e[j + 1] - e[j]);
  }
  for (int i = 0; i <= n_bins; ++i) e[i] = ne[i];
}

}  // namespace madme
