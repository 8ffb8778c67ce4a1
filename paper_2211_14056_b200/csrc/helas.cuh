// helas.cuh — wavefunction / vertex / propagator library of the B200 path, fp64 complex arithmetic.
//
// These are the "spinors", "vertices" and "propagators" of PAPER.md:70 (§2), i.e. the HELAS-style
// routine families BASELINE.json:north_star names (ixxxxx/oxxxxx/vxxxxx, FFV1_{0,1,2}, FFV1P0_3,
// VVV1P0_1, VVVV{1,3,4}P0_1; the closing amplitudes FFV1_0, VVV1_0, VVVV_0 are replaced by dot products), restated from the Feynman rules of
// SURVEY.md §8(c) B/C in the CHIRAL representation with helicity spinors and circular
// polarisations (the oracle uses the Dirac representation with a fixed-axis spin basis, so the
// two sides share neither code nor intermediate values; only the helicity/colour-summed |M|^2 agrees).
//
// All routines here are "bare": couplings (g_s^{n-2} or e^2) and the powers of i carried by
// vertices and propagators are tracked symbolically by the build-time generator
// (paper_2211_14056_b200/gen/) and folded into the {+-1,+-i} colour-flow coefficients, so the
// arithmetic below is pure real/complex FMA work.
//
// Conventions: metric (+,-,-,-); every leg carries its momentum in the
// all-incoming convention k = +p (initial) / -p (final); an off-shell current over the leg set S
// carries K_S = sum_{i in S} k_i, the momentum flowing from the subtree into the next vertex.
//   gamma^mu = [[0, sigma_+^mu], [sigma_-^mu, 0]],  sigma_+- = (1, +-sigma)
//   Vslash = [[0, V0 - s.V], [V0 + s.V, 0]]
// Everything is __host__ __device__ so that tests/ can run the generated programs on the CPU
// (a debugging harness in tests/, never reachable from the product API).
#pragma once
#include <math.h>

#if defined(__CUDACC__)
#define ME_HD __host__ __device__ __forceinline__
#else
#define ME_HD inline
#endif

namespace madme {

struct cplx {
  double re, im;
};
struct wf4 {  // 4 complex components: a spinor (chiral basis) or a 4-vector (upper index)
  cplx c[4];
};
struct vec4 {  // real 4-vector
  double v[4];
};

ME_HD cplx mk(double re, double im) { cplx z; z.re = re; z.im = im; return z; }
ME_HD cplx operator+(cplx a, cplx b) { return mk(a.re + b.re, a.im + b.im); }
ME_HD cplx operator-(cplx a, cplx b) { return mk(a.re - b.re, a.im - b.im); }
ME_HD cplx operator-(cplx a) { return mk(-a.re, -a.im); }
ME_HD cplx operator*(cplx a, cplx b) { return mk(fma(a.re, b.re, -(a.im * b.im)), fma(a.re, b.im, a.im * b.re)); }
ME_HD cplx operator*(double s, cplx a) { return mk(s * a.re, s * a.im); }
ME_HD cplx conj(cplx a) { return mk(a.re, -a.im); }
ME_HD cplx times_i(cplx a) { return mk(-a.im, a.re); }
// acc + a*b
ME_HD cplx cfma(cplx a, cplx b, cplx acc) {
  return mk(fma(a.re, b.re, fma(-a.im, b.im, acc.re)), fma(a.re, b.im, fma(a.im, b.re, acc.im)));
}
// acc - a*b
ME_HD cplx cfms(cplx a, cplx b, cplx acc) {
  return mk(fma(-a.re, b.re, fma(a.im, b.im, acc.re)), fma(-a.re, b.im, fma(-a.im, b.re, acc.im)));
}
// acc + s*a (s real)
ME_HD cplx rfma(double s, cplx a, cplx acc) { return mk(fma(s, a.re, acc.re), fma(s, a.im, acc.im)); }

// Minkowski products
ME_HD double mdot(const vec4& a, const vec4& b) {
  return fma(a.v[0], b.v[0], -fma(a.v[1], b.v[1], fma(a.v[2], b.v[2], a.v[3] * b.v[3])));
}
ME_HD cplx mdot(const vec4& a, const wf4& b) {  // real . complex
  cplx r = a.v[0] * b.c[0];
  r = rfma(-a.v[1], b.c[1], r);
  r = rfma(-a.v[2], b.c[2], r);
  r = rfma(-a.v[3], b.c[3], r);
  return r;
}
ME_HD cplx mdot(const wf4& a, const wf4& b) {  // complex . complex (no conjugation)
  cplx r = a.c[0] * b.c[0];
  r = cfms(a.c[1], b.c[1], r);
  r = cfms(a.c[2], b.c[2], r);
  r = cfms(a.c[3], b.c[3], r);
  return r;
}

// ---------------------------------------------------------------------------------------------
// External wavefunctions (step a5, helicity basis, A3 cancellation-safe forms)
// ---------------------------------------------------------------------------------------------
// Two-component helicity eigenvectors of sigma.p-hat:
//   chi_+ = N (|p|+pz, px+i py),  chi_- = N (-px+i py, |p|+pz),  N = [2|p|(|p|+pz)]^{-1/2}
//   pz = -|p| exactly: chi_+ = (0,1), chi_- = (-1,0);   |p| = 0: chi_+ = (1,0), chi_- = (0,1)
// with |p|+pz := pT^2/(|p|-pz) for pz < 0 (A3).
struct chi2 {
  cplx p[2], m[2];  // chi_+ , chi_-
};
ME_HD chi2 helicity_chi(double px, double py, double pz, double pabs) {
  chi2 x;
  const double pt2 = fma(px, px, py * py);
  if (pabs == 0.0) {
    x.p[0] = mk(1, 0); x.p[1] = mk(0, 0); x.m[0] = mk(0, 0); x.m[1] = mk(1, 0);
  } else if (pt2 == 0.0 && pz < 0.0) {
    x.p[0] = mk(0, 0); x.p[1] = mk(1, 0); x.m[0] = mk(-1, 0); x.m[1] = mk(0, 0);
  } else {
    const double ppz = (pz >= 0.0) ? pabs + pz : pt2 / (pabs - pz);
    const double n = 1.0 / sqrt(2.0 * pabs * ppz);
    x.p[0] = mk(n * ppz, 0); x.p[1] = mk(n * px, n * py);
    x.m[0] = mk(-n * px, n * py); x.m[1] = mk(n * ppz, 0);
  }
  return x;
}

// u(p,lambda) = (w_{-l} chi_l , w_l chi_l),  v(p,lambda) = (-l w_l chi_{-l} , l w_{-l} chi_{-l}),
// w_+- = sqrt(E +- |p|), with sqrt(E-|p|) := m / sqrt(E+|p|) (A3).  p = physical momentum.
// Writes both helicities: out[0] <-> lambda = -1, out[1] <-> lambda = +1.
ME_HD void spinor_u(const double p[4], double mass, wf4 out[2]) {
  const double pabs = sqrt(fma(p[1], p[1], fma(p[2], p[2], p[3] * p[3])));
  const chi2 x = helicity_chi(p[1], p[2], p[3], pabs);
  const double wp = sqrt(p[0] + pabs);
  const double wm = (mass == 0.0) ? 0.0 : mass / wp;
  // lambda = +1: (wm chi_+, wp chi_+)
  out[1].c[0] = wm * x.p[0]; out[1].c[1] = wm * x.p[1]; out[1].c[2] = wp * x.p[0]; out[1].c[3] = wp * x.p[1];
  // lambda = -1: (wp chi_-, wm chi_-)
  out[0].c[0] = wp * x.m[0]; out[0].c[1] = wp * x.m[1]; out[0].c[2] = wm * x.m[0]; out[0].c[3] = wm * x.m[1];
}
ME_HD void spinor_v(const double p[4], double mass, wf4 out[2]) {
  const double pabs = sqrt(fma(p[1], p[1], fma(p[2], p[2], p[3] * p[3])));
  const chi2 x = helicity_chi(p[1], p[2], p[3], pabs);
  const double wp = sqrt(p[0] + pabs);
  const double wm = (mass == 0.0) ? 0.0 : mass / wp;
  // lambda = +1: (-wp chi_-, wm chi_-)
  out[1].c[0] = -wp * x.m[0]; out[1].c[1] = -wp * x.m[1]; out[1].c[2] = wm * x.m[0]; out[1].c[3] = wm * x.m[1];
  // lambda = -1: (wm chi_+, -wp chi_+)
  out[0].c[0] = wm * x.p[0]; out[0].c[1] = wm * x.p[1]; out[0].c[2] = -wp * x.p[0]; out[0].c[3] = -wp * x.p[1];
}
// psi-bar = psi^dagger gamma^0, gamma^0 = [[0,1],[1,0]]: swap the halves and conjugate
ME_HD wf4 dirac_bar(const wf4& s) {
  wf4 r;
  r.c[0] = conj(s.c[2]); r.c[1] = conj(s.c[3]); r.c[2] = conj(s.c[0]); r.c[3] = conj(s.c[1]);
  return r;
}
// eps(p, lambda=+-1) = (-+ e1 - i e2)/sqrt2,  e1 = (0, px pz, py pz, -pT^2)/(|p| pT),  e2 = (0,-py,px,0)/pT
// (pT = 0: e1 = (0,1,0,0), e2 = (0,0,sgn pz,0)).   out[0] <-> lambda=-1, out[1] <-> lambda=+1.
ME_HD void polvec(const double p[4], wf4 out[2]) {
  const double pt2 = fma(p[1], p[1], p[2] * p[2]);
  const double pt = sqrt(pt2);
  const double pabs = sqrt(fma(p[3], p[3], pt2));
  double e1x, e1y, e1z, e2x, e2y;
  if (pt == 0.0) {
    e1x = 1; e1y = 0; e1z = 0; e2x = 0; e2y = (p[3] >= 0.0) ? 1.0 : -1.0;
  } else {
    const double ipt = 1.0 / pt, ipa = 1.0 / pabs;
    e1x = p[1] * p[3] * ipa * ipt; e1y = p[2] * p[3] * ipa * ipt; e1z = -pt * ipa;
    e2x = -p[2] * ipt; e2y = p[1] * ipt;
  }
  const double r2 = 0.70710678118654752440;
  // lambda=+1: (-e1 - i e2)/sqrt2 ; lambda=-1: (+e1 - i e2)/sqrt2
  out[1].c[0] = mk(0, 0); out[1].c[1] = mk(-r2 * e1x, -r2 * e2x); out[1].c[2] = mk(-r2 * e1y, -r2 * e2y); out[1].c[3] = mk(-r2 * e1z, 0);
  out[0].c[0] = mk(0, 0); out[0].c[1] = mk(r2 * e1x, -r2 * e2x); out[0].c[2] = mk(r2 * e1y, -r2 * e2y); out[0].c[3] = mk(r2 * e1z, 0);
}
ME_HD wf4 conj4(const wf4& a) {
  wf4 r;
  for (int i = 0; i < 4; ++i) r.c[i] = conj(a.c[i]);
  return r;
}

// Leg kinds (what stands on the external line), the HELAS names in brackets:
enum LegKind {
  LEG_V_IN = 0,    // incoming vector: eps            [vxxxxx, initial]
  LEG_V_OUT = 1,   // outgoing vector: eps*           [vxxxxx, final]
  LEG_F_OUT = 2,   // outgoing fermion: u-bar, row    [oxxxxx]
  LEG_FB_OUT = 3,  // outgoing antifermion: v, column [ixxxxx]
  LEG_F_IN = 4,    // incoming fermion: u, column     [ixxxxx]
  LEG_FB_IN = 5,   // incoming antifermion: v-bar, row[oxxxxx]
};
// p = PHYSICAL momentum of the leg; out[0], out[1] = helicity -1, +1.
ME_HD void external_wavefunction(int kind, const double p[4], double mass, wf4 out[2]) {
  switch (kind) {
    case LEG_V_IN: polvec(p, out); break;
    case LEG_V_OUT: polvec(p, out); out[0] = conj4(out[0]); out[1] = conj4(out[1]); break;
    case LEG_F_OUT: spinor_u(p, mass, out); out[0] = dirac_bar(out[0]); out[1] = dirac_bar(out[1]); break;
    case LEG_FB_OUT: spinor_v(p, mass, out); break;
    case LEG_F_IN: spinor_u(p, mass, out); break;
    default: spinor_v(p, mass, out); out[0] = dirac_bar(out[0]); out[1] = dirac_bar(out[1]); break;
  }
}

// ---------------------------------------------------------------------------------------------
// Slash products in the chiral representation
// ---------------------------------------------------------------------------------------------
// a = V0+V3, b = V0-V3, c = V1+iV2, d = V1-iV2
//   Vslash psi     = ( b p2 - d p3, -c p2 + a p3,  a p0 + d p1,  c p0 + b p1 )
//   psibar Vslash  = ( a q2 + c q3,  d q2 + b q3,  b q0 - c q1, -d q0 + a q1 )
ME_HD wf4 slash_col(const wf4& V, const wf4& p) {
  const cplx a = V.c[0] + V.c[3], b = V.c[0] - V.c[3];
  const cplx c = V.c[1] + times_i(V.c[2]), d = V.c[1] - times_i(V.c[2]);
  wf4 r;
  r.c[0] = cfms(d, p.c[3], b * p.c[2]);
  r.c[1] = cfms(c, p.c[2], a * p.c[3]);
  r.c[2] = cfma(d, p.c[1], a * p.c[0]);
  r.c[3] = cfma(b, p.c[1], c * p.c[0]);
  return r;
}
ME_HD wf4 slash_row(const wf4& q, const wf4& V) {
  const cplx a = V.c[0] + V.c[3], b = V.c[0] - V.c[3];
  const cplx c = V.c[1] + times_i(V.c[2]), d = V.c[1] - times_i(V.c[2]);
  wf4 r;
  r.c[0] = cfma(c, q.c[3], a * q.c[2]);
  r.c[1] = cfma(b, q.c[3], d * q.c[2]);
  r.c[2] = cfms(c, q.c[1], b * q.c[0]);
  r.c[3] = cfms(d, q.c[0], a * q.c[1]);
  return r;
}
// (s Kslash + m) chi for REAL K, column; then scaled by f.   c = K1+iK2, d = conj(c)
ME_HD wf4 prop_col(const vec4& K, double s, double m, double f, const wf4& x) {
  const double a = s * (K.v[0] + K.v[3]), b = s * (K.v[0] - K.v[3]);
  const cplx c = mk(s * K.v[1], s * K.v[2]), d = mk(s * K.v[1], -s * K.v[2]);
  wf4 r;
  r.c[0] = f * rfma(m, x.c[0], rfma(b, x.c[2], -(d * x.c[3])));
  r.c[1] = f * rfma(m, x.c[1], rfma(a, x.c[3], -(c * x.c[2])));
  r.c[2] = f * rfma(m, x.c[2], rfma(a, x.c[0], d * x.c[1]));
  r.c[3] = f * rfma(m, x.c[3], rfma(b, x.c[1], c * x.c[0]));
  return r;
}
ME_HD wf4 prop_row(const vec4& K, double s, double m, double f, const wf4& q) {
  const double a = s * (K.v[0] + K.v[3]), b = s * (K.v[0] - K.v[3]);
  const cplx c = mk(s * K.v[1], s * K.v[2]), d = mk(s * K.v[1], -s * K.v[2]);
  wf4 r;
  r.c[0] = f * rfma(m, q.c[0], rfma(a, q.c[2], c * q.c[3]));
  r.c[1] = f * rfma(m, q.c[1], rfma(b, q.c[3], d * q.c[2]));
  r.c[2] = f * rfma(m, q.c[2], rfma(b, q.c[0], -(c * q.c[1])));
  r.c[3] = f * rfma(m, q.c[3], rfma(a, q.c[1], -(d * q.c[0])));
  return r;
}

// ---------------------------------------------------------------------------------------------
// Off-shell currents (step a6).  A current over the leg set S is  propagator(K_S) x sum_j i^{k_j} (bare vertex)_j
// over the Feynman subdiagrams j that enter it (me_tasks.cuh::me_run_item): the routines below are the BARE vertices,
// the propagators are prop_row / prop_col above ((-+Kslash_S + m)/(K_S^2 - m^2) on a fermion line) and 1/K_S^2 on a
// vector line.
// ---------------------------------------------------------------------------------------------
// [FFV1_1 / FFV1_2-like]  a spinor absorbs a vector: slash_row(psibar, V), slash_col(V, psi) above.
// [FFV1P0_3-like]  V^mu = psibar gamma^mu psi
//   J0 = q0p2+q1p3+q2p0+q3p1          J1 = (q0p3+q1p2) - (q2p1+q3p0)
//   J2 = -i(q0p3-q1p2) + i(q2p1-q3p0) J3 = (q0p2-q1p3) - (q2p0-q3p1)
ME_HD wf4 ffv_vec_bare(const wf4& q, const wf4& p) {
  const cplx p02 = q.c[0] * p.c[2], p13 = q.c[1] * p.c[3], p20 = q.c[2] * p.c[0], p31 = q.c[3] * p.c[1];
  const cplx p03 = q.c[0] * p.c[3], p12 = q.c[1] * p.c[2], p21 = q.c[2] * p.c[1], p30 = q.c[3] * p.c[0];
  wf4 r;
  r.c[0] = (p02 + p13) + (p20 + p31);
  r.c[1] = (p03 + p12) - (p21 + p30);
  r.c[2] = times_i((p21 - p30) - (p03 - p12));
  r.c[3] = (p02 - p13) - (p20 - p31);
  return r;
}
// [VVV1P0_1-like]  three-gluon vertex with legs (X,K_X), (Y,K_Y), output leg incoming momentum -K_S:
//   V^rho = (X.Y)(K_X-K_Y)^rho + Y^rho ((K_Y+K_S).X) - X^rho ((K_S+K_X).Y)
ME_HD wf4 vvv_vec_bare(const wf4& X, const vec4& KX, const wf4& Y, const vec4& KY) {
  vec4 a, b, d;
  for (int i = 0; i < 4; ++i) {
    a.v[i] = fma(2.0, KY.v[i], KX.v[i]);  // K_Y + K_S
    b.v[i] = fma(2.0, KX.v[i], KY.v[i]);  // K_S + K_X
    d.v[i] = KX.v[i] - KY.v[i];
  }
  const cplx xy = mdot(X, Y), ax = mdot(a, X), by = mdot(b, Y);
  wf4 r;
  for (int i = 0; i < 4; ++i) r.c[i] = cfms(by, X.c[i], cfma(ax, Y.c[i], d.v[i] * xy));
  return r;
}
// [VVVV{1,3,4}P0_1-like]  four-gluon vertex, the three colour (x) Lorentz terms of SURVEY §8(c) C:
//   t1 (f^{xye}f^{zde}): (X.Z) Y - (Y.Z) X
//   t2 (f^{xze}f^{yde}): (X.Y) Z - (Y.Z) X
//   t3 (f^{xde}f^{yze}): (X.Y) Z - (X.Z) Y
ME_HD void vvvv_vec_bare(const wf4& X, const wf4& Y, const wf4& Z, wf4& t1, wf4& t2, wf4& t3) {
  const cplx xy = mdot(X, Y), xz = mdot(X, Z), yz = mdot(Y, Z);
  for (int i = 0; i < 4; ++i) {
    const cplx yzx = yz * X.c[i];
    const cplx xzy = xz * Y.c[i];
    const cplx xyz = xy * Z.c[i];
    t1.c[i] = xzy - yzx;
    t2.c[i] = xyz - yzx;
    t3.c[i] = xyz - xzy;
  }
}

// ---------------------------------------------------------------------------------------------
// Closing amplitudes (step a7): every diagram closes as the contraction of an open current with a propagated one
// (gen/diagrams.py); the vertex-closing forms FFV1_0 / VVV1_0 / VVVV_0 were measured and dropped (profiles/)
// ---------------------------------------------------------------------------------------------
// Propagator-cut closing: J += i^K (U . C), U the open (un-propagated) current over one half of the legs, C the
// propagated current over the other half.  MINK: vector line, Minkowski contraction (+,-,-,-); otherwise a fermion
// line, plain sum over the four spinor components.  Every component is 4 FMAs straight into the flow accumulator.
template <int K> ME_HD void cacc(double& jr, double& ji, cplx a, cplx b) {
  if (K == 0) {        // + a b
    jr = fma(a.re, b.re, fma(-a.im, b.im, jr)); ji = fma(a.re, b.im, fma(a.im, b.re, ji));
  } else if (K == 2) { // - a b
    jr = fma(-a.re, b.re, fma(a.im, b.im, jr)); ji = fma(-a.re, b.im, fma(-a.im, b.re, ji));
  } else if (K == 1) { // + i a b
    jr = fma(-a.re, b.im, fma(-a.im, b.re, jr)); ji = fma(a.re, b.re, fma(-a.im, b.im, ji));
  } else {             // - i a b
    jr = fma(a.re, b.im, fma(a.im, b.re, jr)); ji = fma(-a.re, b.re, fma(a.im, b.im, ji));
  }
}
template <int K, bool MINK> ME_HD void dot_acc(double& jr, double& ji, const wf4& u, const wf4& c) {
  cacc<K>(jr, ji, u.c[0], c.c[0]);
  cacc<MINK ? ((K + 2) & 3) : K>(jr, ji, u.c[1], c.c[1]);
  cacc<MINK ? ((K + 2) & 3) : K>(jr, ji, u.c[2], c.c[2]);
  cacc<MINK ? ((K + 2) & 3) : K>(jr, ji, u.c[3], c.c[3]);
}

// the same contraction as a value (a U . C pair that feeds several colour flows is contracted once) ...
template <bool MINK> ME_HD cplx dot_val(const wf4& u, const wf4& c) {
  cplx t = u.c[0] * c.c[0];
  if (MINK) {
    t = cfms(u.c[1], c.c[1], t); t = cfms(u.c[2], c.c[2], t); t = cfms(u.c[3], c.c[3], t);
  } else {
    t = cfma(u.c[1], c.c[1], t); t = cfma(u.c[2], c.c[2], t); t = cfma(u.c[3], c.c[3], t);
  }
  return t;
}
// ... and J += i^K t
template <int K> ME_HD void jadd(double& jr, double& ji, cplx t) {
  if (K == 0) { jr += t.re; ji += t.im; }
  else if (K == 2) { jr -= t.re; ji -= t.im; }
  else if (K == 1) { jr -= t.im; ji += t.re; }
  else { jr += t.im; ji -= t.re; }
}

}  // namespace madme
