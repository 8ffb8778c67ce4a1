// ORACLE — TEST INFRASTRUCTURE ONLY (see algebra.hpp header).
//
// wavefunctions.hpp — external-leg wavefunctions, step a5 of SURVEY.md §8(a)
// ("spinors" of PAPER.md:70; HELAS ixxxxx/oxxxxx/vxxxxx of BASELINE.json:north_star),
// written as the plain textbook definitions in the Dirac representation:
//
//   u(p,s) = (pslash + m) e_s     / sqrt(E+m),  s = 0,1      (tier 0)
//   v(p,s) = (-pslash + m) e_{s+2} / sqrt(E+m)
//   e_k = unit 4-spinors (fixed-axis spin basis; valid for m = 0 too)
//   gluon/photon: two transverse vectors e1, e2 _|_ p   (linear polarisations, real)
//
// An optional second basis (helicity spinors / circular polarisations) exists ONLY so the
// tests can check that me2 does not depend on the basis (pin table I).
// The helicity-summed |M|^2 needs nothing but completeness:  sum_s u ubar = pslash + m,
// sum_s v vbar = pslash - m, sum_l eps^mu eps*^nu = -g^{mu nu} + gauge terms.
#pragma once
#include "algebra.hpp"

namespace orc {

enum SpinBasis { BASIS_FIXED_AXIS = 0, BASIS_HELICITY = 1 };
enum PolBasis { POL_LINEAR = 0, POL_CIRCULAR = 1 };

// two-component spin vectors chi_s, s = 0,1
inline void chi_basis(const P4& p, int basis, cd chi[2][2]) {
  if (basis == BASIS_FIXED_AXIS) {
    chi[0][0] = 1; chi[0][1] = 0;
    chi[1][0] = 0; chi[1][1] = 1;
    return;
  }
  // helicity eigenvectors of sigma.p-hat: chi_+ ~ (|p|+pz, px+i py), chi_- ~ (-px+i py, |p|+pz)
  const double pt2 = p[1]*p[1] + p[2]*p[2];
  const double pa = std::sqrt(pt2 + p[3]*p[3]);
  if (pa == 0.0) { chi[0][0] = 1; chi[0][1] = 0; chi[1][0] = 0; chi[1][1] = 1; return; }
  if (pt2 == 0.0 && p[3] < 0) { chi[0][0] = 0; chi[0][1] = 1; chi[1][0] = -1; chi[1][1] = 0; return; }
  // |p|+pz without cancellation
  const double ppz = (p[3] >= 0) ? pa + p[3] : pt2 / (pa - p[3]);
  const double N = 1.0 / std::sqrt(2.0 * pa * ppz);
  chi[0][0] = N * ppz;              chi[0][1] = N * cd(p[1], p[2]);
  chi[1][0] = N * cd(-p[1], p[2]);  chi[1][1] = N * ppz;
}

// u(p,s): column spinor of a fermion of mass m
inline Sp u_spinor(const P4& p, double m, int s, int basis) {
  cd chi[2][2]; chi_basis(p, basis, chi);
  Sp e = {{chi[s][0], chi[s][1], 0, 0}};
  M4 A = slash(p) + cd(m) * mident();
  return cd(1.0 / std::sqrt(p[0] + m)) * mul(A, e);
}
// v(p,s): column spinor of an antifermion of mass m
inline Sp v_spinor(const P4& p, double m, int s, int basis) {
  cd chi[2][2]; chi_basis(p, basis, chi);
  Sp e = {{0, 0, chi[s][0], chi[s][1]}};
  M4 A = cd(m) * mident() - slash(p);
  return cd(1.0 / std::sqrt(p[0] + m)) * mul(A, e);
}

// transverse polarisation vectors of a massless vector with momentum p:
//   e1 = (0, px pz, py pz, -pT^2)/(|p| pT),  e2 = (0, -py, px, 0)/pT
//   pT = 0:  e1 = (0,1,0,0), e2 = (0,0,sgn pz,0)
//   circular: eps(lambda=+-1) = (-+ e1 - i e2)/sqrt(2)
// pol = 0,1.  Linear: pol 0 -> e1, pol 1 -> e2.  Circular: pol 0 -> lambda=+1, pol 1 -> lambda=-1.
inline V4 polvec(const P4& p, int pol, int basis) {
  const double pt2 = p[1]*p[1] + p[2]*p[2];
  const double pt = std::sqrt(pt2);
  const double pa = std::sqrt(pt2 + p[3]*p[3]);
  double e1[4], e2[4];
  if (pt == 0.0) {
    e1[0] = 0; e1[1] = 1; e1[2] = 0; e1[3] = 0;
    e2[0] = 0; e2[1] = 0; e2[2] = (p[3] >= 0 ? 1.0 : -1.0); e2[3] = 0;
  } else {
    e1[0] = 0; e1[1] = p[1]*p[3]/(pa*pt); e1[2] = p[2]*p[3]/(pa*pt); e1[3] = -pt/pa;
    e2[0] = 0; e2[1] = -p[2]/pt; e2[2] = p[1]/pt; e2[3] = 0;
  }
  V4 r;
  if (basis == POL_LINEAR) {
    for (int i = 0; i < 4; ++i) r[i] = (pol == 0) ? e1[i] : e2[i];
  } else {
    const double sgn = (pol == 0) ? -1.0 : 1.0;  // lambda=+1: -e1 - i e2 ; lambda=-1: +e1 - i e2
    const double r2 = 1.0 / std::sqrt(2.0);
    for (int i = 0; i < 4; ++i) r[i] = r2 * cd(sgn * e1[i], -e2[i]);
  }
  return r;
}
inline V4 vconj(const V4& a) { return {{std::conj(a[0]), std::conj(a[1]), std::conj(a[2]), std::conj(a[3])}}; }

}  // namespace orc
