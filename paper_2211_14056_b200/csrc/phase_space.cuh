// phase_space.cuh — the steps in front of me_eval, as per-thread device functions (one event per thread):
//   a1 Philox4x32-10 uniforms, a2 Vegas grid map, a3 RAMBO (classic / "on diet", massive rescaling), a4 cuts.
// The paper names only "Vegas"; RAMBO, Philox and the cuts come from
// BASELINE.json:north_star / configs and are implemented from their standard definitions, with the readings
// of DESIGN.md §Readings (R-G1..R-G7).  All fp64 except the Philox words (uint32) and bin indices (int).
#pragma once
#include <math.h>
#include <stdint.h>

namespace madme {

constexpr int PS_MAX_FINAL = 6;
constexpr double PS_PI = 3.14159265358979323846;

// ---- a1: Philox4x32-10 (Salmon et al., SC'11) ----------------------------------------------------------
// one round: (c0,c1,c2,c3) <- (hi(M1 c2)^c1^k0, lo(M1 c2), hi(M0 c0)^c3^k1, lo(M0 c0)); Weyl key schedule.
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
  for (int round = 0; round < 10; ++round) {
    const uint32_t lo0 = 0xD2511F53u * c.x, hi0 = __umulhi(0xD2511F53u, c.x);
    const uint32_t lo1 = 0xCD9E8D57u * c.z, hi1 = __umulhi(0xCD9E8D57u, c.z);
    c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
    k.x += 0x9E3779B9u;
    k.y += 0xBB67AE85u;
  }
  return c;
}
// 53 random bits -> the open interval (0,1)
__device__ __forceinline__ double philox_u01(uint32_t hi, uint32_t lo) {
  const unsigned long long bits = ((static_cast<unsigned long long>(hi) << 32) | lo) >> 11;
  return (static_cast<double>(bits) + 0.5) * 0x1p-53;
}
// u[0..n_dim): dimension d <- block j = d/2, word pair d%2 of counter (event lo, event hi, j, iteration)
template <int MAXD>
__device__ __forceinline__ void philox_fill(uint64_t seed, uint32_t iteration, uint64_t event, int n_dim, double* u) {
  const uint2 key = make_uint2(static_cast<uint32_t>(seed), static_cast<uint32_t>(seed >> 32));
#pragma unroll
  for (int j = 0; j < (MAXD + 1) / 2; ++j) {
    if (2 * j < n_dim) {
      const uint4 w = philox4x32_10(
          make_uint4(static_cast<uint32_t>(event), static_cast<uint32_t>(event >> 32), static_cast<uint32_t>(j), iteration), key);
      u[2 * j] = philox_u01(w.x, w.y);
      if (2 * j + 1 < n_dim) u[2 * j + 1] = philox_u01(w.z, w.w);
    }
  }
}

// ---- a2: Vegas map of one coordinate ---------------------------------------------------------------------
// t = y N_b, i = min(floor t, N_b-1), x = e_i + (t-i)(e_{i+1}-e_i), jacobian factor N_b (e_{i+1}-e_i)
__device__ __forceinline__ double vegas_map_1d(const double* __restrict__ e, int n_bins, double y, double& jac, int& bin) {
  const double t = y * n_bins;
  int i = static_cast<int>(floor(t));
  i = max(0, min(i, n_bins - 1));
  const double lo = e[i], w = e[i + 1] - lo;
  jac *= n_bins * w;
  bin = i;
  return lo + (t - i) * w;
}

// ---- a3: RAMBO -------------------------------------------------------------------------------------------
// massless n-body volume W0 = (pi/2)^{n-1} s^{n-2} / [(n-1)!(n-2)!] (2 pi)^{4-3n}
__host__ __device__ inline double rambo_volume(int n, double s) {
  double w = 1.0, fa = 1.0, fb = 1.0;
  for (int i = 0; i < n - 1; ++i) w *= 0.5 * PS_PI;
  for (int i = 0; i < n - 2; ++i) w *= s;
  for (int i = 2; i <= n - 1; ++i) fa *= i;
  for (int i = 2; i <= n - 2; ++i) fb *= i;
  w /= fa * fb;
  // (2 pi)^{4-3n}: 3n-4 divisions
  for (int i = 0; i < 3 * n - 4; ++i) w /= 2.0 * PS_PI;
  return w;
}

// massive legs: xi from sum_i sqrt(m_i^2 + xi^2 E_i^2) = sqrt_s, Newton, exactly 10 steps from
// xi0 = sqrt(1 - (sum m/sqrt_s)^2); returns the weight factor
// (sum|k|/sqrt_s)^{2n-3} prod(|k|/k0) sqrt_s / sum(|k|^2/k0)            (DESIGN.md R-G1)
template <int N>
__device__ __forceinline__ double rambo_massive(double sqrt_s, const double* __restrict__ m, double (&p)[N][4]) {
  double msum = 0.0;
  bool massive = false;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    msum += m[i];
    massive = massive || (m[i] != 0.0);
  }
  if (!massive) return 1.0;
  const double r = msum / sqrt_s;
  double xi = sqrt(1.0 - r * r);
  for (int it = 0; it < 10; ++it) {
    double f = -sqrt_s, df = 0.0;
#pragma unroll
    for (int i = 0; i < N; ++i) {
      const double e2 = p[i][0] * p[i][0];
      const double e = sqrt(m[i] * m[i] + xi * xi * e2);
      f += e;
      df += xi * e2 / e;
    }
    xi -= f / df;
  }
  double sk = 0.0, prod = 1.0, sk2 = 0.0;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    const double e0 = p[i][0];
    const double k0 = sqrt(m[i] * m[i] + xi * xi * e0 * e0);
    const double ka = xi * e0;
    p[i][0] = k0;
    p[i][1] *= xi;
    p[i][2] *= xi;
    p[i][3] *= xi;
    sk += ka;
    prod *= ka / k0;
    sk2 += ka * ka / k0;
  }
  double pw = 1.0;
  const double base = sk / sqrt_s;
#pragma unroll
  for (int i = 0; i < 2 * N - 3; ++i) pw *= base;
  return pw * prod * sqrt_s / sk2;
}

// classic RAMBO: 4 uniforms per particle (cos theta, phi, and two for the energy), then the conformal boost to the rest
// frame of Q = sum q_i and the scaling by x = sqrt_s / M.  The boost is written without cancellations (DESIGN.md
// R-G1b): with q_i = w_i (1, n_i) the invariants q_i.q_j = w_i w_j |n_i - n_j|^2 / 2 are sums of squares, so
//   E_i = (Q.q_i) / M = sum_{j != i} q_i.q_j / M,   M^2 = sum_i Q.q_i,   p_i = x [ q_i - Q (w_i + E_i) / (M + Q0) ]
// keep momentum conservation at the 1e-13 level even when two of the q_i are almost collinear (two-body case).
template <int N>
__device__ __forceinline__ void rambo_classic(const double* __restrict__ r, double sqrt_s, double (&p)[N][4]) {
  double w[N], dir[N][3], Qv[3] = {0.0, 0.0, 0.0}, Q0 = 0.0;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    const double c = 2.0 * r[4 * i] - 1.0, phi = 2.0 * PS_PI * r[4 * i + 1];
    w[i] = -log(r[4 * i + 2] * r[4 * i + 3]);
    const double st = sqrt(1.0 - c * c);
    double sn, cs;
    sincos(phi, &sn, &cs);
    dir[i][0] = st * cs;
    dir[i][1] = st * sn;
    dir[i][2] = c;
    Q0 += w[i];
#pragma unroll
    for (int k = 0; k < 3; ++k) Qv[k] += w[i] * dir[i][k];
  }
  double inv[N], M2 = 0.0;   // inv[i] = Q.q_i
#pragma unroll
  for (int i = 0; i < N; ++i) inv[i] = 0.0;
#pragma unroll
  for (int i = 0; i < N; ++i)
#pragma unroll
    for (int j = i + 1; j < N; ++j) {
      const double dx = dir[i][0] - dir[j][0], dy = dir[i][1] - dir[j][1], dz = dir[i][2] - dir[j][2];
      const double qq = w[i] * w[j] * (0.5 * (dx * dx + dy * dy + dz * dz));
      inv[i] += qq;
      inv[j] += qq;
    }
#pragma unroll
  for (int i = 0; i < N; ++i) M2 += inv[i];
  const double M = sqrt(M2), x = sqrt_s / M, den = 1.0 / (M + Q0);
#pragma unroll
  for (int i = 0; i < N; ++i) {
    const double e = inv[i] / M;
    const double f = (w[i] + e) * den;
    p[i][0] = x * e;
#pragma unroll
    for (int k = 0; k < 3; ++k) p[i][k + 1] = x * (w[i] * dir[i][k] - Qv[k] * f);
  }
}

__device__ __forceinline__ double ipow(double u, int e) {
  double r = 1.0;
  for (int i = 0; i < e; ++i) r *= u;
  return r;
}
// RAMBO "on diet" (Plaetzer 2013): N-2 uniforms for the intermediate masses (root of
// r = (k+1) u^{2k} - k u^{2k+2} by 64 bisection steps), then N-1 isotropic two-body decays with (cos theta, phi)
template <int N>
__device__ __forceinline__ void rambo_diet(const double* __restrict__ r, double sqrt_s, double (&p)[N][4]) {
  double M[N + 1];
  M[1] = sqrt_s;
#pragma unroll
  for (int i = 2; i <= N - 1; ++i) {
    const int k = N - i;
    double lo = 0.0, hi = 1.0;
    for (int it = 0; it < 64; ++it) {
      const double u = 0.5 * (lo + hi);
      const double f = (k + 1) * ipow(u, 2 * k) - k * ipow(u, 2 * k + 2);
      if (f < r[i - 2]) lo = u; else hi = u;
    }
    M[i] = 0.5 * (lo + hi) * M[i - 1];
  }
  M[N] = 0.0;
  double Q[4] = {sqrt_s, 0.0, 0.0, 0.0};
#pragma unroll
  for (int i = 1; i <= N - 1; ++i) {
    const double c = 2.0 * r[N - 2 + 2 * (i - 1)] - 1.0, phi = 2.0 * PS_PI * r[N - 2 + 2 * (i - 1) + 1];
    const double st = sqrt(1.0 - c * c);
    const double pa = (M[i] * M[i] - M[i + 1] * M[i + 1]) / (2.0 * M[i]);
    double sn, cs;
    sincos(phi, &sn, &cs);
    const double a0 = pa, a1 = pa * st * cs, a2 = pa * st * sn, a3 = pa * c;
    const double Qa = Q[1] * a1 + Q[2] * a2 + Q[3] * a3;
    const double e = (Q[0] * a0 + Qa) / M[i];
    const double fac = (Qa / (Q[0] + M[i]) + a0) / M[i];
    p[i - 1][0] = e;
    p[i - 1][1] = a1 + fac * Q[1];
    p[i - 1][2] = a2 + fac * Q[2];
    p[i - 1][3] = a3 + fac * Q[3];
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) Q[mu] -= p[i - 1][mu];
  }
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) p[N - 1][mu] = Q[mu];
}

// one event: final momenta p[N][4] and the weight (w0 = rambo_volume(N, s), computed once on the host)
template <int N>
__device__ __forceinline__ double rambo_event(const double* __restrict__ r, double sqrt_s, const double* __restrict__ m,
                                              int ps_mode, double w0, double (&p)[N][4]) {
  if (ps_mode == 0) rambo_classic<N>(r, sqrt_s, p);
  else rambo_diet<N>(r, sqrt_s, p);
  return w0 * rambo_massive<N>(sqrt_s, m, p);
}

// toy gluon density of the hadronic Vegas mode (DESIGN.md R-N3): a DECLARED toy, g(x) = 3 x^-1.2 (1-x)^5
__device__ __forceinline__ double toy_gluon_density(double x) {
  const double y = 1.0 - x, y2 = y * y;
  return 3.0 * pow(x, -1.2) * (y2 * y2 * y);
}

// the beams of the quark-initiated channels (N1 x N3): declared toys as well.  kind: 0 gluon, 1 quark: 2 x^-0.5 (1-x)^3,
// 2 antiquark: 0.3 x^-1.1 (1-x)^7
__device__ __forceinline__ double toy_density(int kind, double x) {
  if (kind == 0) return toy_gluon_density(x);
  const double y = 1.0 - x, y2 = y * y;
  if (kind == 1) return 2.0 * rsqrt(x) * (y2 * y);
  return 0.3 * pow(x, -1.1) * (y2 * y2 * y2 * y);
}

// ---- a4: cuts (DESIGN.md R-G5) -----------------------------------------------------------------------------
// every final gluon: pT > ptj_min and DeltaR(g, X) = sqrt(dy^2 + dphi^2) > dr_min to every other final parton;
// true rapidity; strict inequalities; a cut value <= 0 is off.  gluon_mask bit i <-> final particle i is a gluon.
template <int N>
__device__ __forceinline__ bool passes_cuts(const double (&p)[N][4], unsigned gluon_mask, double ptj_min, double dr_min) {
  double y[N], ph[N];
#pragma unroll
  for (int i = 0; i < N; ++i) {
    y[i] = 0.5 * log((p[i][0] + p[i][3]) / (p[i][0] - p[i][3]));
    ph[i] = atan2(p[i][2], p[i][1]);
  }
  bool ok = true;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    if (!((gluon_mask >> i) & 1u)) continue;
    if (ptj_min > 0.0 && !(sqrt(p[i][1] * p[i][1] + p[i][2] * p[i][2]) > ptj_min)) ok = false;
    if (dr_min > 0.0) {
#pragma unroll
      for (int j = 0; j < N; ++j) {
        if (j == i) continue;
        double dphi = fabs(ph[i] - ph[j]);
        if (dphi > PS_PI) dphi = 2.0 * PS_PI - dphi;
        const double dy = y[i] - y[j];
        if (!(sqrt(dy * dy + dphi * dphi) > dr_min)) ok = false;
      }
    }
  }
  return ok;
}

}  // namespace madme
