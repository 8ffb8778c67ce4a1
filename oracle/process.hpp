// ORACLE — TEST INFRASTRUCTURE ONLY (see algebra.hpp header).
//
// process.hpp — the processes of BASELINE.json:configs[0..3] and the quark-initiated channels of the paper's
// hadronic processes (Table 1) as plain data:
// external legs (kind, mass, fermion line), couplings, averaging factor S of SURVEY.md §8(c) F.
//
// Leg order follows `momenta[n_ev][n_ext][4]` of BASELINE.json:north_star:
//   legs 0,1 incoming (along +z, -z), legs 2.. outgoing
//   gg -> t tbar (g)(g)(g):  g g | t tbar g g g
//   q qbar -> t tbar (g)(g): q qbar | t tbar g g       (q: one massless flavour, different from t)
//   q g -> t tbar q (g)    : q g | t tbar q g
//   qbar g -> t tbar qbar (g): qbar g | t tbar qbar g    (the charge conjugates of the line above)
//   e+ e- -> mu+ mu-      :  e- e+ | mu- mu+
#pragma once
#include <cstring>
#include <string>
#include <vector>
#include "algebra.hpp"

extern "C" {
// mirrors include/madme.h:me_params field by field (the oracle does not include product headers)
typedef struct {
  double alpha_s, alpha_em, m_top, w_top;  // fixed couplings; w_top must be 0
  double ptj_min, dr_min;                  // cuts (<= 0 disables); used by cuts/vegas only
} me_params_ref;
}

namespace orc {

constexpr int NMAX_FINAL = 6;  // max final-state particles

enum LegKind {
  G_IN = 0,   // incoming gluon: eps
  G_OUT = 1,  // outgoing gluon: eps*
  Q_OUT = 2,  // outgoing quark: u-bar (row)
  QB_OUT = 3, // outgoing antiquark: v (column)
  F_IN = 4,   // incoming fermion (e-, q): u (column)
  FB_IN = 5,  // incoming antifermion (e+, qbar): v-bar (row)
};
inline bool is_gluon_kind(int k) { return k == G_IN || k == G_OUT; }
inline bool is_row_kind(int k) { return k == Q_OUT || k == FB_IN; }   // psi-bar ends of a fermion line
inline bool is_col_kind(int k) { return k == QB_OUT || k == F_IN; }   // psi ends

struct Process {
  std::string name;
  bool qed = false;
  int n_ext = 0;
  std::vector<int> kind;
  std::vector<double> mass;
  std::vector<int> line;  // fermion line (flavour) of a fermion leg: 0 = top, 1 = the light quark q; -1 for gluons
  double gs = 0, ee = 0;
  double avg = 1;  // S = spin avg * colour avg * identical-particle factor
  int n_gluon() const { int n = 0; for (int k : kind) n += (k == G_IN || k == G_OUT); return n; }
  int n_lines() const { int n = 0; for (int l : line) n = l + 1 > n ? l + 1 : n; return n; }
};

inline bool make_process(const char* name, const me_params_ref& par, Process& P) {
  P = Process();
  P.name = name;
  const double pi = 3.14159265358979323846;
  P.gs = std::sqrt(4.0 * pi * par.alpha_s);   // g_s = sqrt(4 pi alpha_s)
  P.ee = std::sqrt(4.0 * pi * par.alpha_em);  // e   = sqrt(4 pi alpha)
  if (!std::strcmp(name, "epem_mupmum")) {
    P.qed = true; P.n_ext = 4;
    P.kind = {F_IN, FB_IN, Q_OUT, QB_OUT};
    P.mass = {0, 0, 0, 0};
    P.line = {0, 0, 1, 1};
    P.avg = 4.0;  // spin average 1/4 (BASELINE.json:configs[0])
    return true;
  }
  // quark-initiated channels: averages 1/4 spins x 1/9 (q qbar) or 1/24 (q g) colours x 1/n_id!
  const double mt = par.m_top;
  int extra_q = -1;
  if (!std::strcmp(name, "qqx_ttx")) extra_q = 0;
  else if (!std::strcmp(name, "qqx_ttxg")) extra_q = 1;
  else if (!std::strcmp(name, "qqx_ttxgg")) extra_q = 2;
  if (extra_q >= 0) {
    P.n_ext = 4 + extra_q;
    P.kind = {F_IN, FB_IN, Q_OUT, QB_OUT};
    P.mass = {0, 0, mt, mt};
    P.line = {1, 1, 0, 0};
    double sym = 1;
    for (int i = 0; i < extra_q; ++i) { P.kind.push_back(G_OUT); P.mass.push_back(0); P.line.push_back(-1); sym *= (i + 1); }
    P.avg = 4.0 * 9.0 * sym;
    return true;
  }
  extra_q = -1;
  bool anti = false;
  if (!std::strcmp(name, "qg_ttxq")) extra_q = 0;
  else if (!std::strcmp(name, "qg_ttxqg")) extra_q = 1;
  else if (!std::strcmp(name, "qxg_ttxqx")) { extra_q = 0; anti = true; }
  else if (!std::strcmp(name, "qxg_ttxqxg")) { extra_q = 1; anti = true; }
  if (extra_q >= 0) {
    P.n_ext = 5 + extra_q;
    P.kind = {anti ? FB_IN : F_IN, G_IN, Q_OUT, QB_OUT, anti ? QB_OUT : Q_OUT};
    P.mass = {0, 0, mt, mt, 0};
    P.line = {1, -1, 0, 0, 1};
    for (int i = 0; i < extra_q; ++i) { P.kind.push_back(G_OUT); P.mass.push_back(0); P.line.push_back(-1); }
    P.avg = 4.0 * 24.0;
    return true;
  }
  int extra = -1;
  if (!std::strcmp(name, "gg_ttx")) extra = 0;
  else if (!std::strcmp(name, "gg_ttxg")) extra = 1;
  else if (!std::strcmp(name, "gg_ttxgg")) extra = 2;
  else if (!std::strcmp(name, "gg_ttxggg")) extra = 3;
  if (extra < 0) return false;
  P.n_ext = 4 + extra;
  P.kind = {G_IN, G_IN, Q_OUT, QB_OUT};
  P.mass = {0, 0, par.m_top, par.m_top};
  P.line = {-1, -1, 0, 0};
  double sym = 1;
  for (int i = 0; i < extra; ++i) { P.kind.push_back(G_OUT); P.mass.push_back(0); P.line.push_back(-1); sym *= (i + 1); }
  P.avg = 4.0 * 64.0 * sym;  // 1/4 spins * 1/64 colours * 1/n_id!  (BASELINE.json:configs[1..3])
  return true;
}

}  // namespace orc
