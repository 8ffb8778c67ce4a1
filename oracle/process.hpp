// ORACLE — TEST INFRASTRUCTURE ONLY (see algebra.hpp header).
//
// process.hpp — the processes of BASELINE.json:configs[0..3] as plain data:
// external legs (kind, mass), couplings, averaging factor S of SURVEY.md §8(c) F.
//
// Leg order follows `momenta[n_ev][n_ext][4]` of BASELINE.json:north_star:
//   legs 0,1 incoming (along +z, -z), legs 2.. outgoing
//   gg -> t tbar (g)(g):  g g | t tbar g g
//   e+ e- -> mu+ mu-   :  e- e+ | mu- mu+
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
  F_IN = 4,   // incoming fermion (e-): u (column)          [QED only]
  FB_IN = 5,  // incoming antifermion (e+): v-bar (row)     [QED only]
};

struct Process {
  std::string name;
  bool qed = false;
  int n_ext = 0;
  std::vector<int> kind;
  std::vector<double> mass;
  double gs = 0, ee = 0;
  double avg = 1;  // S = spin avg * colour avg * identical-particle factor
  int n_gluon() const { int n = 0; for (int k : kind) n += (k == G_IN || k == G_OUT); return n; }
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
    P.avg = 4.0;  // spin average 1/4 (BASELINE.json:configs[0])
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
  double sym = 1;
  for (int i = 0; i < extra; ++i) { P.kind.push_back(G_OUT); P.mass.push_back(0); sym *= (i + 1); }
  P.avg = 4.0 * 64.0 * sym;  // 1/4 spins * 1/64 colours * 1/n_id!  (BASELINE.json:configs[1..3])
  return true;
}

}  // namespace orc
