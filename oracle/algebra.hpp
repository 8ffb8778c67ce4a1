// ORACLE — TEST INFRASTRUCTURE ONLY.  Not part of the product path.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may build, load or call anything under oracle/.  It shares no code with the
// CUDA path (paper_2211_14056_b200/), and never includes a CUDA header.
//
// algebra.hpp — explicit 4x4 Dirac matrices (Dirac representation), Minkowski
// 4-vectors and SU(3) Gell-Mann tensors, written out as plain definitions.
//
// Cites: SURVEY.md §8(c) A1 (metric diag(+,-,-,-), p=(E,px,py,pz)),
//        §8(c) B "Tier 0 (Dirac representation, fixed-axis spin basis)",
//        §8(c) C (QCD conventions: T^a = lambda^a/2, [T^a,T^b] = i f^{abc} T^c).
//        The paper itself ("vertices, spinors or propagators") gives no
//        formula; everything here is textbook QFT, pinned by tests/test_oracle_*.py.
#pragma once
#include <array>
#include <cmath>
#include <complex>
#include <cstdint>
#include <vector>

namespace orc {

using cd = std::complex<double>;
static const cd I_(0.0, 1.0);

// ---- real Minkowski 4-vector, upper index, (E, px, py, pz) ------------------------------
struct P4 {
  double v[4];
  double& operator[](int i) { return v[i]; }
  double operator[](int i) const { return v[i]; }
};
inline P4 operator+(const P4& a, const P4& b) { return {{a[0]+b[0], a[1]+b[1], a[2]+b[2], a[3]+b[3]}}; }
inline P4 operator-(const P4& a, const P4& b) { return {{a[0]-b[0], a[1]-b[1], a[2]-b[2], a[3]-b[3]}}; }
inline P4 operator*(double s, const P4& a) { return {{s*a[0], s*a[1], s*a[2], s*a[3]}}; }
inline double mdot(const P4& a, const P4& b) { return a[0]*b[0] - a[1]*b[1] - a[2]*b[2] - a[3]*b[3]; }

// ---- complex 4-vector (polarisation / off-shell vector current), upper index ------------
struct V4 {
  cd v[4];
  cd& operator[](int i) { return v[i]; }
  const cd& operator[](int i) const { return v[i]; }
};
inline V4 vzero() { return {{cd(0), cd(0), cd(0), cd(0)}}; }
inline V4 operator+(const V4& a, const V4& b) { return {{a[0]+b[0], a[1]+b[1], a[2]+b[2], a[3]+b[3]}}; }
inline V4 operator-(const V4& a, const V4& b) { return {{a[0]-b[0], a[1]-b[1], a[2]-b[2], a[3]-b[3]}}; }
inline V4 operator*(cd s, const V4& a) { return {{s*a[0], s*a[1], s*a[2], s*a[3]}}; }
inline V4 tocomplex(const P4& p) { return {{cd(p[0]), cd(p[1]), cd(p[2]), cd(p[3])}}; }
// Minkowski product WITHOUT complex conjugation: a.b = a0 b0 - a1 b1 - a2 b2 - a3 b3
inline cd mdot(const V4& a, const V4& b) { return a[0]*b[0] - a[1]*b[1] - a[2]*b[2] - a[3]*b[3]; }
inline cd mdot(const P4& a, const V4& b) { return a[0]*b[0] - a[1]*b[1] - a[2]*b[2] - a[3]*b[3]; }

// ---- Dirac spinors and 4x4 matrices ------------------------------------------------------
struct Sp {  // 4 complex components; used both as column (psi) and as row (psi-bar)
  cd s[4];
  cd& operator[](int i) { return s[i]; }
  const cd& operator[](int i) const { return s[i]; }
};
inline Sp szero() { return {{cd(0), cd(0), cd(0), cd(0)}}; }
inline Sp operator+(const Sp& a, const Sp& b) { return {{a[0]+b[0], a[1]+b[1], a[2]+b[2], a[3]+b[3]}}; }
inline Sp operator*(cd c, const Sp& a) { return {{c*a[0], c*a[1], c*a[2], c*a[3]}}; }

struct M4 {
  cd m[4][4];
};
inline M4 mzero() { M4 r; for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) r.m[i][j] = 0; return r; }
inline M4 mident() { M4 r = mzero(); for (int i = 0; i < 4; ++i) r.m[i][i] = 1; return r; }
inline M4 operator+(const M4& a, const M4& b) { M4 r; for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) r.m[i][j] = a.m[i][j] + b.m[i][j]; return r; }
inline M4 operator-(const M4& a, const M4& b) { M4 r; for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) r.m[i][j] = a.m[i][j] - b.m[i][j]; return r; }
inline M4 operator*(cd c, const M4& a) { M4 r; for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) r.m[i][j] = c * a.m[i][j]; return r; }
inline M4 operator*(const M4& a, const M4& b) {
  M4 r = mzero();
  for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) for (int k = 0; k < 4; ++k) r.m[i][j] += a.m[i][k] * b.m[k][j];
  return r;
}
// matrix * column
inline Sp mul(const M4& a, const Sp& x) {
  Sp r = szero();
  for (int i = 0; i < 4; ++i) for (int k = 0; k < 4; ++k) r[i] += a.m[i][k] * x[k];
  return r;
}
// row * matrix
inline Sp mul(const Sp& x, const M4& a) {
  Sp r = szero();
  for (int j = 0; j < 4; ++j) for (int k = 0; k < 4; ++k) r[j] += x[k] * a.m[k][j];
  return r;
}
// row * column (no conjugation)
inline cd dot(const Sp& row, const Sp& col) { return row[0]*col[0] + row[1]*col[1] + row[2]*col[2] + row[3]*col[3]; }

// gamma^mu in the Dirac representation:
//   gamma^0 = diag(1,1,-1,-1),  gamma^i = [[0, sigma_i], [-sigma_i, 0]]
struct Gammas {
  M4 g[4];
  Gammas() {
    for (int mu = 0; mu < 4; ++mu) g[mu] = mzero();
    g[0].m[0][0] = 1; g[0].m[1][1] = 1; g[0].m[2][2] = -1; g[0].m[3][3] = -1;
    const cd s[3][2][2] = {{{0, 1}, {1, 0}}, {{0, -I_}, {I_, 0}}, {{1, 0}, {0, -1}}};  // Pauli matrices
    for (int i = 0; i < 3; ++i)
      for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) {
          g[i + 1].m[a][b + 2] = s[i][a][b];
          g[i + 1].m[a + 2][b] = -s[i][a][b];
        }
  }
};
inline const Gammas& gammas() { static const Gammas G; return G; }

// slash(V) = gamma^mu V_mu = gamma^0 V^0 - gamma^1 V^1 - gamma^2 V^2 - gamma^3 V^3   (V upper-index)
inline M4 slash(const V4& V) {
  const Gammas& G = gammas();
  return V[0] * G.g[0] - V[1] * G.g[1] - V[2] * G.g[2] - V[3] * G.g[3];
}
inline M4 slash(const P4& p) { return slash(tocomplex(p)); }

// psi-bar = psi^dagger gamma^0
inline Sp bar(const Sp& psi) {
  Sp c = {{std::conj(psi[0]), std::conj(psi[1]), std::conj(psi[2]), std::conj(psi[3])}};
  return mul(c, gammas().g[0]);
}

// ---- SU(3): Gell-Mann matrices, T^a = lambda^a / 2, f^{abc} -------------------------------
struct C3 {
  cd m[3][3];
};
inline C3 c3zero() { C3 r; for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) r.m[i][j] = 0; return r; }
inline C3 c3ident() { C3 r = c3zero(); for (int i = 0; i < 3; ++i) r.m[i][i] = 1; return r; }
inline C3 operator*(const C3& a, const C3& b) {
  C3 r = c3zero();
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) for (int k = 0; k < 3; ++k) r.m[i][j] += a.m[i][k] * b.m[k][j];
  return r;
}
inline C3 operator-(const C3& a, const C3& b) { C3 r; for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) r.m[i][j] = a.m[i][j] - b.m[i][j]; return r; }
inline cd trace(const C3& a) { return a.m[0][0] + a.m[1][1] + a.m[2][2]; }
inline C3 dagger(const C3& a) { C3 r; for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) r.m[i][j] = std::conj(a.m[j][i]); return r; }

struct SU3 {
  C3 T[8];          // T^a = lambda^a / 2
  double f[8][8][8];  // [T^a, T^b] = i f^{abc} T^c  =>  f^{abc} = -2i Tr([T^a,T^b] T^c)
  SU3() {
    C3 l[8];
    for (int a = 0; a < 8; ++a) l[a] = c3zero();
    l[0].m[0][1] = 1; l[0].m[1][0] = 1;
    l[1].m[0][1] = -I_; l[1].m[1][0] = I_;
    l[2].m[0][0] = 1; l[2].m[1][1] = -1;
    l[3].m[0][2] = 1; l[3].m[2][0] = 1;
    l[4].m[0][2] = -I_; l[4].m[2][0] = I_;
    l[5].m[1][2] = 1; l[5].m[2][1] = 1;
    l[6].m[1][2] = -I_; l[6].m[2][1] = I_;
    const double r3 = 1.0 / std::sqrt(3.0);
    l[7].m[0][0] = r3; l[7].m[1][1] = r3; l[7].m[2][2] = -2.0 * r3;
    for (int a = 0; a < 8; ++a)
      for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) T[a].m[i][j] = 0.5 * l[a].m[i][j];
    for (int a = 0; a < 8; ++a)
      for (int b = 0; b < 8; ++b)
        for (int c = 0; c < 8; ++c) {
          cd t = cd(0, -2.0) * trace((T[a] * T[b] - T[b] * T[a]) * T[c]);
          f[a][b][c] = t.real();
        }
  }
};
inline const SU3& su3() { static const SU3 S; return S; }

}  // namespace orc
