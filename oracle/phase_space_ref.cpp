// ORACLE — TEST INFRASTRUCTURE ONLY (see algebra.hpp header).
//
// phase_space_ref.cpp — the steps either side of me_eval, scalar and sequential:
//   a1  Philox4x32-10 uniforms
//   a3  RAMBO, classic 4n and "on diet" 3n-4 variants, massive legs by xi-rescaling (G1, G2)
//   a4  cuts pT(g) > ptj_min, DeltaR(g, X) > dr_min                    (G5)
// The paper names none of these (it says only "Vegas"); they are required by
// BASELINE.json:north_star / configs and are written from the standard definitions.
#include <cmath>
#include <cstdint>
#include <cstring>
#include "process.hpp"

namespace orc {

// ---- Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), SURVEY §8(c) G4 ---------------------
// counter c[4], key k[2] of uint32; 10 rounds of
//   (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0))
// key bumped by (0x9E3779B9, 0xBB67AE85) between rounds.
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int r = 0; r < 10; ++r) {
    const uint64_t p0 = uint64_t(M0) * c0, p1 = uint64_t(M1) * c2;
    const uint32_t n0 = uint32_t(p1 >> 32) ^ c1 ^ k0, n1 = uint32_t(p1);
    const uint32_t n2 = uint32_t(p0 >> 32) ^ c3 ^ k1, n3 = uint32_t(p0);
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += W0; k1 += W1;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// uniform in the OPEN interval (0,1) from two words: ((x0*2^32 + x1) >> 11 + 1/2) * 2^-53
inline double u01(uint32_t hi, uint32_t lo) {
  const uint64_t x = (uint64_t(hi) << 32 | lo) >> 11;
  return (double(x) + 0.5) * (1.0 / 9007199254740992.0);
}

// key = (seed lo, seed hi); counter = (event lo, event hi, pair index j, iteration);
// dimension d uses j = d/2 and the word pair (d mod 2).
void philox_uniforms(uint64_t seed, uint64_t iteration, uint64_t event, int n_dim, double* u) {
  const uint32_t key[2] = {uint32_t(seed), uint32_t(seed >> 32)};
  for (int j = 0; 2 * j < n_dim; ++j) {
    const uint32_t ctr[4] = {uint32_t(event), uint32_t(event >> 32), uint32_t(j), uint32_t(iteration)};
    uint32_t o[4];
    philox4x32_10(ctr, key, o);
    u[2 * j] = u01(o[0], o[1]);
    if (2 * j + 1 < n_dim) u[2 * j + 1] = u01(o[2], o[3]);
  }
}

// ---- RAMBO ----------------------------------------------------------------------------------
static double factorial(int n) { double f = 1; for (int i = 2; i <= n; ++i) f *= i; return f; }

// W0 = (pi/2)^{n-1} s^{n-2} / [(n-1)!(n-2)!] (2 pi)^{4-3n}: volume of massless n-body phase space
double rambo_w0(int n, double s) {
  const double pi = 3.14159265358979323846;
  return std::pow(pi / 2, n - 1) * std::pow(s, n - 2) / (factorial(n - 1) * factorial(n - 2)) * std::pow(2 * pi, 4 - 3 * n);
}

// massive legs: solve sum_i sqrt(m_i^2 + xi^2 E_i^2) = sqrt_s by Newton, FIXED 10 iterations from
// xi0 = sqrt(1 - (sum m / sqrt_s)^2); then k_i = (sqrt(m^2 + xi^2 E^2), xi p_i) and
// W = W0 (sum|k|/sqrt_s)^{2n-3} prod(|k|/k0) sqrt_s / sum(|k|^2/k0).
static double massive_rescale(int n, double sqrt_s, const double* m, double p[][4]) {
  double msum = 0; bool any = false;
  for (int i = 0; i < n; ++i) { msum += m[i]; any = any || m[i] != 0.0; }
  if (!any) return 1.0;
  double xi = std::sqrt(1.0 - (msum / sqrt_s) * (msum / sqrt_s));
  for (int it = 0; it < 10; ++it) {
    double f = -sqrt_s, df = 0;
    for (int i = 0; i < n; ++i) {
      const double e = std::sqrt(m[i] * m[i] + xi * xi * p[i][0] * p[i][0]);
      f += e; df += xi * p[i][0] * p[i][0] / e;
    }
    xi -= f / df;
  }
  double sk = 0, prod = 1, sk2 = 0;
  for (int i = 0; i < n; ++i) {
    const double e0 = p[i][0];
    const double k0 = std::sqrt(m[i] * m[i] + xi * xi * e0 * e0);
    const double ka = xi * e0;  // |k| = xi |p| = xi E (massless p)
    p[i][0] = k0; p[i][1] *= xi; p[i][2] *= xi; p[i][3] *= xi;
    sk += ka; prod *= ka / k0; sk2 += ka * ka / k0;
  }
  return std::pow(sk / sqrt_s, 2 * n - 3) * prod * sqrt_s / sk2;
}

// classic RAMBO: r[4i+0..3] = (r1,r2,r3,r4) of final particle i:
//   q_i = q0_i (1, n_i), Q = sum q_i, M = sqrt(Q^2), then the boost to the rest frame of Q and the scaling x = sqrt_s / M.
// The boost is evaluated in the cancellation-free form (same map, reading R-G1b; the textbook form
// Q0^2 - |Q|^2 loses conservation to ~1e-9 sqrt_s when two q_i are nearly collinear):
//   q_i.q_j = q0_i q0_j |n_i - n_j|^2 / 2  (>= 0, no cancellation),   Q.q_i = sum_{j != i} q_i.q_j,   M^2 = sum_i Q.q_i,
//   p0_i = x (Q.q_i) / M,      p_i = x [ q_i - Q (q0_i + (Q.q_i)/M) / (M + Q0) ]        (3-vectors),
// which is p0 = x (gamma q0 + b.q), p = x (q + b q0 + a (b.q) b) with b = -Q/M, gamma = Q0/M, a = 1/(1+gamma) rewritten.
static double rambo_classic(const double* r, double sqrt_s, const double* m, int n, double p[][4]) {
  const double pi = 3.14159265358979323846;
  double q0[NMAX_FINAL], nv[NMAX_FINAL][3], Q[4] = {0, 0, 0, 0};
  for (int i = 0; i < n; ++i) {
    const double c = 2 * r[4 * i] - 1, phi = 2 * pi * r[4 * i + 1];
    q0[i] = -std::log(r[4 * i + 2] * r[4 * i + 3]);
    const double st = std::sqrt(1 - c * c);
    nv[i][0] = st * std::cos(phi); nv[i][1] = st * std::sin(phi); nv[i][2] = c;
    Q[0] += q0[i];
    for (int j = 0; j < 3; ++j) Q[j + 1] += q0[i] * nv[i][j];
  }
  double Qq[NMAX_FINAL], M2 = 0;
  for (int i = 0; i < n; ++i) {
    Qq[i] = 0;
    for (int j = 0; j < n; ++j) {
      if (j == i) continue;
      double d2 = 0;
      for (int k = 0; k < 3; ++k) d2 += (nv[i][k] - nv[j][k]) * (nv[i][k] - nv[j][k]);
      Qq[i] += q0[i] * q0[j] * 0.5 * d2;
    }
    M2 += Qq[i];
  }
  const double M = std::sqrt(M2), x = sqrt_s / M;
  for (int i = 0; i < n; ++i) {
    const double e = Qq[i] / M;                 // energy in the rest frame of Q, before the scaling
    const double f = (q0[i] + e) / (M + Q[0]);
    p[i][0] = x * e;
    for (int j = 0; j < 3; ++j) p[i][j + 1] = x * (q0[i] * nv[i][j] - Q[j + 1] * f);
  }
  return rambo_w0(n, sqrt_s * sqrt_s) * massive_rescale(n, sqrt_s, m, p);
}

// RAMBO "on diet" (Plaetzer 2013): r[0..n-3] intermediate masses, then n-1 pairs
// (cos theta, phi).  M_1 = sqrt_s, M_i = u_i M_{i-1} with u_i the root in (0,1) of
//   r = (k+1) u^{2k} - k u^{2k+2},  k = n - i,    i = 2..n-1     (bisection, FIXED 64 steps)
// M_n = 0; then n-1 isotropic two-body decays Q_i -> p_i + Q_{i+1}, boosted with Q_i.
static double upow(double u, int e) { double r = 1; for (int i = 0; i < e; ++i) r *= u; return r; }
static double rambo_diet(const double* r, double sqrt_s, const double* m, int n, double p[][4]) {
  const double pi = 3.14159265358979323846;
  double M[NMAX_FINAL + 1];
  M[1] = sqrt_s;
  for (int i = 2; i <= n - 1; ++i) {
    const int k = n - i;
    double lo = 0, hi = 1;
    for (int it = 0; it < 64; ++it) {
      const double u = 0.5 * (lo + hi);
      const double f = (k + 1) * upow(u, 2 * k) - k * upow(u, 2 * k + 2);
      if (f < r[i - 2]) lo = u; else hi = u;
    }
    M[i] = 0.5 * (lo + hi) * M[i - 1];
  }
  M[n] = 0;
  double Q[4] = {sqrt_s, 0, 0, 0};
  for (int i = 1; i <= n - 1; ++i) {
    const double c = 2 * r[n - 2 + 2 * (i - 1)] - 1, phi = 2 * pi * r[n - 2 + 2 * (i - 1) + 1];
    const double st = std::sqrt(1 - c * c);
    const double pa = (M[i] * M[i] - M[i + 1] * M[i + 1]) / (2 * M[i]);
    const double a[4] = {pa, pa * st * std::cos(phi), pa * st * std::sin(phi), pa * c};  // p_i in the rest frame of Q_i
    // boost from the rest frame of Q_i (mass M_i carried explicitly) to the lab
    const double Qa = Q[1] * a[1] + Q[2] * a[2] + Q[3] * a[3];
    const double e = (Q[0] * a[0] + Qa) / M[i];
    const double fac = (Qa / (Q[0] + M[i]) + a[0]) / M[i];
    p[i - 1][0] = e;
    for (int j = 1; j < 4; ++j) p[i - 1][j] = a[j] + fac * Q[j];
    for (int mu = 0; mu < 4; ++mu) Q[mu] -= p[i - 1][mu];
  }
  for (int mu = 0; mu < 4; ++mu) p[n - 1][mu] = Q[mu];
  return rambo_w0(n, sqrt_s * sqrt_s) * massive_rescale(n, sqrt_s, m, p);
}

// one event: uniforms -> momenta[n+2][4] (incoming legs (sqrt_s/2)(1,0,0,+-1) prepended) and weight
double rambo_event(const double* r, double sqrt_s, const double* m, int n, int ps_mode, double* mom) {
  double p[NMAX_FINAL][4];
  const double w = (ps_mode == 0) ? rambo_classic(r, sqrt_s, m, n, p) : rambo_diet(r, sqrt_s, m, n, p);
  const double e = 0.5 * sqrt_s;
  mom[0] = e; mom[1] = 0; mom[2] = 0; mom[3] = e;
  mom[4] = e; mom[5] = 0; mom[6] = 0; mom[7] = -e;
  for (int i = 0; i < n; ++i) for (int mu = 0; mu < 4; ++mu) mom[8 + 4 * i + mu] = p[i][mu];
  return w;
}

// ---- cuts --------------------------------------------------------------------
// every final gluon: pT > ptj_min; DeltaR(g, X) = sqrt(dy^2 + dphi^2) > dr_min for every other final
// parton X (t, tbar, other gluons); true rapidity y = 1/2 ln((E+pz)/(E-pz)); dphi in (-pi, pi];
// strict inequalities; a cut value <= 0 is disabled.  is_gluon[i] flags final particle i.
int passes_cuts(const double* mom /*[n+2][4]*/, int n, const int* is_gluon, double ptj_min, double dr_min) {
  const double pi = 3.14159265358979323846;
  double y[NMAX_FINAL], ph[NMAX_FINAL];
  for (int i = 0; i < n; ++i) {
    const double* p = mom + 8 + 4 * i;
    y[i] = 0.5 * std::log((p[0] + p[3]) / (p[0] - p[3]));
    ph[i] = std::atan2(p[2], p[1]);
  }
  for (int i = 0; i < n; ++i) {
    if (!is_gluon[i]) continue;
    const double* p = mom + 8 + 4 * i;
    if (ptj_min > 0 && !(std::sqrt(p[1] * p[1] + p[2] * p[2]) > ptj_min)) return 0;
    if (dr_min > 0)
      for (int j = 0; j < n; ++j) {
        if (j == i) continue;
        double dphi = std::fabs(ph[i] - ph[j]);
        if (dphi > pi) dphi = 2 * pi - dphi;
        const double dy = y[i] - y[j];
        if (!(std::sqrt(dy * dy + dphi * dphi) > dr_min)) return 0;
      }
  }
  return 1;
}

}  // namespace orc
