// ORACLE — TEST INFRASTRUCTURE ONLY (see algebra.hpp header).
//
// me_tier0.cpp — TIER 0, "the definition" (tier 0; Feynman rules §8(c) C).
//
// The tree amplitude for ONE assignment of helicities and colours to the external legs is
// the sum of all Feynman diagrams.  It is computed here by the colour-dressed off-shell
// recursion stated in SURVEY §8(c) C ("Recursive form used by tier 0"): for every subset S
// of the non-root legs
//     B_S = sum over unordered splits S = A u B       (3-point vertices)
//                            and   S = A u B u C      (4-gluon vertex)
//           of vertex(J_A, J_B[, J_C]),       J_X = propagator(K_X) * B_X,  K_X = sum_{i in X} k_i,
// single legs carrying their wavefunction; amplitude = wavefunction_root . B_{all others}.
// That sums every diagram exactly once without listing them.  Colours are explicit
// Gell-Mann tensors, spinors are explicit 4-component objects, gamma matrices are explicit
// 4x4 matrices; then  me2 = (1/S) sum_{helicities} sum_{colours} |M|^2  by brute force.
//
// Feynman rules, all momenta INCOMING to the vertex:
//   qbar-q-g : i g_s gamma^mu T^a_{ij}
//   ggg      : g_s f^{abc} [ g^{mu nu}(k1-k2)^rho + g^{nu rho}(k2-k3)^mu + g^{rho mu}(k3-k1)^nu ]
//   gggg     : -i g_s^2 [ f^{abe}f^{cde}(g^{mu rho}g^{nu sigma} - g^{mu sigma}g^{nu rho})
//                       + f^{ace}f^{bde}(g^{mu nu}g^{rho sigma} - g^{mu sigma}g^{nu rho})
//                       + f^{ade}f^{bce}(g^{mu nu}g^{rho sigma} - g^{mu rho}g^{nu sigma}) ]
//   fermion propagator i(qslash+m)/(q^2-m^2), q along the fermion arrow;
//   gluon propagator  -i g^{mu nu} delta^{ab} / q^2  (Feynman gauge); no width (§8(c) A2).
//
// Cost: seconds per event for gg->ttbar gg; used on a handful of events to pin tier 1.
#include "me_ref.hpp"

namespace orc {

namespace {

// Type of a current over a leg subset S: a gluon if every fermion line has both or neither of its ends in S, the row
// (psi-bar side) or column (psi side) spinor of line f if exactly one end of exactly one line is in S, nothing (no such
// current exists: two different flavours cannot meet at a vertex) otherwise.  Line 0 = top, line 1 = the light quark.
enum CurType { T_NONE = -1, T_GLUON = 0 };
inline int t_row(int line) { return 1 + 2 * line; }
inline int t_col(int line) { return 2 + 2 * line; }
inline bool is_row(int t) { return t > 0 && (t & 1); }
inline bool is_col(int t) { return t > 0 && !(t & 1); }
inline int line_of(int t) { return (t - 1) / 2; }

// A colour-dressed off-shell current.
//   gluon : c[a][mu], a = 0..7 adjoint colour, mu upper Lorentz index
//   row   : c[j][alpha], j = 0..2 open (anti-quark side) colour index, alpha Dirac index
//   col   : c[i][alpha], i = 0..2 open (quark side) colour index
struct Cur {
  int type = T_GLUON;
  bool set = false;
  cd c[8][4];
  void zero() { for (int a = 0; a < 8; ++a) for (int m = 0; m < 4; ++m) c[a][m] = 0; }
};

inline V4 gl(const Cur& J, int a) { return {{J.c[a][0], J.c[a][1], J.c[a][2], J.c[a][3]}}; }
inline Sp spn(const Cur& J, int i) { return {{J.c[i][0], J.c[i][1], J.c[i][2], J.c[i][3]}}; }

struct Ctx {
  const me_handle_ref* h;
  const Ext* E;
  int n;
  double gs;
  int row_leg[2] = {-1, -1}, col_leg[2] = {-1, -1};  // the psi-bar end and the psi end of each fermion line
  double mline[2] = {0, 0};                          // mass of each line
  std::vector<Cur> J;   // propagated currents, index = subset mask over legs (bit i = leg i)
  std::vector<P4> K;    // K_S
  int type_of(unsigned S) const {
    int t = T_GLUON;
    for (int f = 0; f < 2; ++f) {
      if (row_leg[f] < 0) continue;
      const bool r = S >> row_leg[f] & 1u, c = S >> col_leg[f] & 1u;
      if (r == c) continue;
      if (t != T_GLUON) return T_NONE;
      t = r ? t_row(f) : t_col(f);
    }
    return t;
  }
};

// ggg vertex with legs (A, B, off-shell third leg), all momenta incoming, k3 = -(kA+kB):
//   B^{c rho} += g_s f^{abc} [ (JA.JB)(kA-kB)^rho + JB^rho ((kB-k3).JA) + JA^rho ((k3-kA).JB) ]
void add_ggg(const Ctx& X, const Cur& A, const P4& kA, const Cur& B, const P4& kB, Cur& out) {
  const SU3& G = su3();
  const P4 k3 = (-1.0) * (kA + kB);
  const P4 dAB = kA - kB, dB3 = kB - k3, d3A = k3 - kA;
  for (int a = 0; a < 8; ++a) {
    const V4 ja = gl(A, a);
    if (ja[0] == 0.0 && ja[1] == 0.0 && ja[2] == 0.0 && ja[3] == 0.0) continue;
    for (int b = 0; b < 8; ++b) {
      const V4 jb = gl(B, b);
      if (jb[0] == 0.0 && jb[1] == 0.0 && jb[2] == 0.0 && jb[3] == 0.0) continue;
      const cd ab = mdot(ja, jb), xa = mdot(dB3, ja), xb = mdot(d3A, jb);
      V4 v;
      for (int r = 0; r < 4; ++r) v[r] = ab * dAB[r] + xa * jb[r] + xb * ja[r];
      for (int c = 0; c < 8; ++c) {
        const double f = G.f[a][b][c];
        if (f == 0.0) continue;
        for (int r = 0; r < 4; ++r) out.c[c][r] += X.gs * f * v[r];
      }
    }
  }
}

// gggg vertex with legs (A,B,C, off-shell fourth leg d,sigma):
//   B^{d sigma} += -i g_s^2 [ f^{abe}f^{cde}((JA.JC) JB - (JB.JC) JA)
//                           + f^{ace}f^{bde}((JA.JB) JC - (JB.JC) JA)
//                           + f^{ade}f^{bce}((JA.JB) JC - (JA.JC) JB) ]^sigma
void add_gggg(const Ctx& X, const Cur& A, const Cur& B, const Cur& C, Cur& out) {
  const SU3& G = su3();
  const cd pref = cd(0, -1) * X.gs * X.gs;
  for (int a = 0; a < 8; ++a) {
    const V4 ja = gl(A, a);
    if (ja[0] == 0.0 && ja[1] == 0.0 && ja[2] == 0.0 && ja[3] == 0.0) continue;
    for (int b = 0; b < 8; ++b) {
      const V4 jb = gl(B, b);
      if (jb[0] == 0.0 && jb[1] == 0.0 && jb[2] == 0.0 && jb[3] == 0.0) continue;
      for (int c = 0; c < 8; ++c) {
        const V4 jc = gl(C, c);
        if (jc[0] == 0.0 && jc[1] == 0.0 && jc[2] == 0.0 && jc[3] == 0.0) continue;
        const cd ab = mdot(ja, jb), ac = mdot(ja, jc), bc = mdot(jb, jc);
        for (int d = 0; d < 8; ++d) {
          double c1 = 0, c2 = 0, c3 = 0;
          for (int e = 0; e < 8; ++e) {
            c1 += G.f[a][b][e] * G.f[c][d][e];
            c2 += G.f[a][c][e] * G.f[b][d][e];
            c3 += G.f[a][d][e] * G.f[b][c][e];
          }
          if (c1 == 0.0 && c2 == 0.0 && c3 == 0.0) continue;
          for (int s = 0; s < 4; ++s) {
            const cd t1 = ac * jb[s] - bc * ja[s];
            const cd t2 = ab * jc[s] - bc * ja[s];
            const cd t3 = ab * jc[s] - ac * jb[s];
            out.c[d][s] += pref * (c1 * t1 + c2 * t2 + c3 * t3);
          }
        }
      }
    }
  }
}

// row (ubar ... T..T)_j  absorbs gluon:  B_row[j] += sum_{a,i} R[i] (i g_s gamma^mu G^a_mu) T^a_{ij}
void add_row_g(const Ctx& X, const Cur& R, const Cur& Gc, Cur& out) {
  const SU3& S = su3();
  for (int a = 0; a < 8; ++a) {
    const V4 g = gl(Gc, a);
    if (g[0] == 0.0 && g[1] == 0.0 && g[2] == 0.0 && g[3] == 0.0) continue;
    const M4 V = cd(0, X.gs) * slash(g);
    for (int i = 0; i < 3; ++i) {
      const Sp r = mul(spn(R, i), V);
      for (int j = 0; j < 3; ++j) {
        const cd t = S.T[a].m[i][j];
        if (t == 0.0) continue;
        for (int al = 0; al < 4; ++al) out.c[j][al] += t * r[al];
      }
    }
  }
}
// gluon absorbed by column (T..T v)_i :  B_col[i] += sum_{a,j} T^a_{ij} (i g_s gamma^mu G^a_mu) C[j]
void add_g_col(const Ctx& X, const Cur& Gc, const Cur& C, Cur& out) {
  const SU3& S = su3();
  for (int a = 0; a < 8; ++a) {
    const V4 g = gl(Gc, a);
    if (g[0] == 0.0 && g[1] == 0.0 && g[2] == 0.0 && g[3] == 0.0) continue;
    const M4 V = cd(0, X.gs) * slash(g);
    for (int j = 0; j < 3; ++j) {
      const Sp r = mul(V, spn(C, j));
      for (int i = 0; i < 3; ++i) {
        const cd t = S.T[a].m[i][j];
        if (t == 0.0) continue;
        for (int al = 0; al < 4; ++al) out.c[i][al] += t * r[al];
      }
    }
  }
}
// row x column -> gluon:  B^{a mu} += sum_{ij} R[i] (i g_s gamma^mu) T^a_{ij} C[j]
void add_row_col(const Ctx& X, const Cur& R, const Cur& C, Cur& out) {
  const SU3& S = su3();
  const Gammas& G = gammas();
  for (int i = 0; i < 3; ++i)
    for (int j = 0; j < 3; ++j) {
      V4 v;
      for (int mu = 0; mu < 4; ++mu) v[mu] = cd(0, X.gs) * dot(spn(R, i), mul(G.g[mu], spn(C, j)));
      for (int a = 0; a < 8; ++a) {
        const cd t = S.T[a].m[i][j];
        if (t == 0.0) continue;
        for (int mu = 0; mu < 4; ++mu) out.c[a][mu] += t * v[mu];
      }
    }
}

// un-propagated current B_S: sum over all unordered 2- and 3-way splits
void build_B(Ctx& X, unsigned S, Cur& B) {
  const int tS = X.type_of(S);
  B.type = tS; B.set = true; B.zero();
  if (tS == T_NONE) return;
  const unsigned low = S & (~S + 1u);
  // 2-way splits {A, Bm}; A holds the lowest leg of S so each unordered split appears once
  for (unsigned A = (S - 1) & S; A; A = (A - 1) & S) {
    if (!(A & low)) continue;
    const unsigned Bm = S & ~A;
    const int tA = X.type_of(A), tB = X.type_of(Bm);
    const Cur &JA = X.J[A], &JB = X.J[Bm];
    if (tA == T_NONE || tB == T_NONE) continue;
    if (tS == T_GLUON) {   // g g -> g, or the two ends of ONE line -> g
      if (tA == T_GLUON && tB == T_GLUON) add_ggg(X, JA, X.K[A], JB, X.K[Bm], B);
      else if (is_row(tA) && is_col(tB) && line_of(tA) == line_of(tB)) add_row_col(X, JA, JB, B);
      else if (is_col(tA) && is_row(tB) && line_of(tA) == line_of(tB)) add_row_col(X, JB, JA, B);
    } else if (is_row(tS)) {   // the line's row absorbs a gluon
      if (tA == tS && tB == T_GLUON) add_row_g(X, JA, JB, B);
      else if (tB == tS && tA == T_GLUON) add_row_g(X, JB, JA, B);
    } else {
      if (tA == tS && tB == T_GLUON) add_g_col(X, JB, JA, B);
      else if (tB == tS && tA == T_GLUON) add_g_col(X, JA, JB, B);
    }
  }
  // 3-way splits {A, Bm, C}, all gluon-type (4-gluon vertex)
  if (tS == T_GLUON) {
    for (unsigned A = (S - 1) & S; A; A = (A - 1) & S) {
      if (!(A & low) || X.type_of(A) != T_GLUON) continue;
      const unsigned R = S & ~A;
      const unsigned lowR = R & (~R + 1u);
      for (unsigned Bm = (R - 1) & R; Bm; Bm = (Bm - 1) & R) {
        if (!(Bm & lowR)) continue;
        const unsigned C = R & ~Bm;
        if (X.type_of(Bm) != T_GLUON || X.type_of(C) != T_GLUON) continue;
        add_gggg(X, X.J[A], X.J[Bm], X.J[C], B);
      }
    }
  }
}

// J_S = propagator(K_S) * B_S
void propagate(const Ctx& X, unsigned S, const Cur& B, Cur& J) {
  J = B;
  const P4& K = X.K[S];
  if (B.type == T_NONE) return;
  if (B.type == T_GLUON) {
    const cd pr = cd(0, -1) / mdot(K, K);  // -i / q^2
    for (int a = 0; a < 8; ++a) for (int m = 0; m < 4; ++m) J.c[a][m] = pr * B.c[a][m];
  } else if (is_row(B.type)) {
    // fermion arrow runs INTO this blob: momentum along the arrow is q = -K_S; row * S(q)
    const double mq = X.mline[line_of(B.type)];
    const P4 q = (-1.0) * K;
    const M4 Sq = (cd(0, 1) / (mdot(q, q) - mq * mq)) * (slash(q) + cd(mq) * mident());
    for (int j = 0; j < 3; ++j) { Sp r = mul(spn(B, j), Sq); for (int al = 0; al < 4; ++al) J.c[j][al] = r[al]; }
  } else {
    // fermion arrow runs OUT of this blob: q = +K_S; S(q) * column
    const double mq = X.mline[line_of(B.type)];
    const M4 Sq = (cd(0, 1) / (mdot(K, K) - mq * mq)) * (slash(K) + cd(mq) * mident());
    for (int i = 0; i < 3; ++i) { Sp r = mul(Sq, spn(B, i)); for (int al = 0; al < 4; ++al) J.c[i][al] = r[al]; }
  }
}

}  // namespace

// i*M for one assignment hel[leg] in {0,1}, col[leg] (gluon 0..7, quark 0..2).  Root = leg 0.
// Two fermion lines of different flavour (t and q): every diagram has the same two open lines, so
// there is no relative sign between diagrams from fermion statistics (no exchange diagram exists).
cd tier0_amplitude(const me_handle_ref& h, const Ext& E, const int* hel, const int* col) {
  const Process& P = h.P;
  Ctx X;
  X.h = &h; X.E = &E; X.n = P.n_ext; X.gs = P.gs;
  for (int i = 0; i < P.n_ext; ++i) {
    if (is_row_kind(P.kind[i])) { X.row_leg[P.line[i]] = i; X.mline[P.line[i]] = P.mass[i]; }
    if (is_col_kind(P.kind[i])) X.col_leg[P.line[i]] = i;
  }
  const unsigned full = (1u << P.n_ext) - 1u, rest = full & ~1u;
  X.J.assign(full + 1, Cur());
  X.K.assign(full + 1, P4{{0, 0, 0, 0}});
  for (unsigned S = 1; S <= full; ++S)
    for (int i = 0; i < P.n_ext; ++i)
      if (S >> i & 1u) X.K[S] = X.K[S] + E.k[i];
  // single legs: wavefunction (x) unit colour vector
  for (int i = 1; i < P.n_ext; ++i) {
    Cur& J = X.J[1u << i];
    J.set = true; J.zero();
    if (is_gluon_kind(P.kind[i])) { J.type = T_GLUON; for (int m = 0; m < 4; ++m) J.c[col[i]][m] = E.eps[i][hel[i]][m]; }
    else if (is_row_kind(P.kind[i])) { J.type = t_row(P.line[i]); for (int m = 0; m < 4; ++m) J.c[col[i]][m] = E.sp[i][hel[i]][m]; }
    else { J.type = t_col(P.line[i]); for (int m = 0; m < 4; ++m) J.c[col[i]][m] = E.sp[i][hel[i]][m]; }
  }
  // subsets of the non-root legs in order of size
  for (int sz = 2; sz <= P.n_ext - 1; ++sz)
    for (unsigned S = 2; S <= rest; ++S) {
      if ((S & 1u) || __builtin_popcount(S) != sz) continue;
      Cur B;
      build_B(X, S, B);
      if (S == rest) {
        // close on the root leg with its wavefunction and its colour: a gluon (eps_mu B^{a mu}), the psi end of a
        // line (B is that line's row: B[j] u) or its psi-bar end (B is the column: vbar B[i])
        if (is_gluon_kind(P.kind[0])) return B.type == T_GLUON ? mdot(E.eps[0][hel[0]], gl(B, col[0])) : cd(0);
        if (is_col_kind(P.kind[0])) return B.type == t_row(P.line[0]) ? dot(spn(B, col[0]), E.sp[0][hel[0]]) : cd(0);
        return B.type == t_col(P.line[0]) ? dot(E.sp[0][hel[0]], spn(B, col[0])) : cd(0);
      }
      propagate(X, S, B, X.J[S]);
    }
  return cd(0);
}

// me2 = (1/S) sum_hel sum_col |M|^2    (SURVEY §8(c) E tier 0, F)
double tier0_me2(const me_handle_ref& h, const double* mom) {
  const Process& P = h.P;
  Ext E;
  build_ext(h, mom, E);
  const int n = P.n_ext;
  std::vector<int> ncol(n);
  long long ncomb = 1;
  for (int i = 0; i < n; ++i) { ncol[i] = (P.kind[i] == G_IN || P.kind[i] == G_OUT) ? 8 : 3; ncomb *= ncol[i]; }
  double total = 0;
#pragma omp parallel for reduction(+ : total) schedule(dynamic, 16)
  for (long long ic = 0; ic < ncomb; ++ic) {
    int col[NMAX], hel[NMAX];
    long long t = ic;
    for (int i = 0; i < n; ++i) { col[i] = int(t % ncol[i]); t /= ncol[i]; }
    double s = 0;
    for (int ih = 0; ih < (1 << n); ++ih) {
      for (int i = 0; i < n; ++i) hel[i] = ih >> i & 1;
      s += std::norm(tier0_amplitude(h, E, hel, col));
    }
    total += s;
  }
  return total / P.avg;
}

}  // namespace orc
