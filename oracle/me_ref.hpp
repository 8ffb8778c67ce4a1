// ORACLE — TEST INFRASTRUCTURE ONLY (see algebra.hpp header).
//
// me_ref.hpp — handle and per-event external-wavefunction table shared by the two
// oracle tiers (tier 0 "definition", tier 1 "diagrammatic scalar").
#pragma once
#include <map>
#include <memory>
#include "process.hpp"
#include "wavefunctions.hpp"

namespace orc {

constexpr int NMAX = 8;  // max external legs

// External wavefunctions of one event, both spin states of every leg (step a5).
struct Ext {
  int n = 0;
  P4 p[NMAX];       // physical momenta as given
  P4 k[NMAX];       // all-incoming convention: k = +p (legs 0,1), -p (final)
  V4 eps[NMAX][2];  // vector legs: eps (incoming) or eps* (outgoing)
  Sp sp[NMAX][2];   // fermion legs: u / v-bar / u-bar / v according to LegKind
};

struct Tier1;   // defined in me_tier1.cpp  (one quark line, colour-flow basis)
struct Tier1G;  // defined in me_tier1g.cpp (any number of lines, diagram basis)

}  // namespace orc

struct me_handle_ref {
  orc::Process P;
  me_params_ref par;
  int spin_basis = orc::BASIS_FIXED_AXIS;
  int pol_basis = orc::POL_LINEAR;
  int ward_leg = -1;  // test hook: replace this gluon's polarisation vector by its momentum
  std::shared_ptr<orc::Tier1> t1;    // processes with one quark line
  std::shared_ptr<orc::Tier1G> t1g;  // processes with two quark lines; built on demand for the others (cross-check)
};

namespace orc {

inline void build_ext(const me_handle_ref& h, const double* mom /*[n_ext][4]*/, Ext& E) {
  const Process& P = h.P;
  E.n = P.n_ext;
  for (int i = 0; i < P.n_ext; ++i) {
    for (int mu = 0; mu < 4; ++mu) E.p[i][mu] = mom[4 * i + mu];
    E.k[i] = (i < 2) ? E.p[i] : (-1.0) * E.p[i];
    for (int s = 0; s < 2; ++s) {
      switch (P.kind[i]) {
        case G_IN:  E.eps[i][s] = polvec(E.p[i], s, h.pol_basis); break;
        case G_OUT: E.eps[i][s] = vconj(polvec(E.p[i], s, h.pol_basis)); break;
        case Q_OUT: E.sp[i][s] = bar(u_spinor(E.p[i], P.mass[i], s, h.spin_basis)); break;   // u-bar, row
        case QB_OUT: E.sp[i][s] = v_spinor(E.p[i], P.mass[i], s, h.spin_basis); break;       // v, column
        case F_IN:  E.sp[i][s] = u_spinor(E.p[i], P.mass[i], s, h.spin_basis); break;        // u, column
        case FB_IN: E.sp[i][s] = bar(v_spinor(E.p[i], P.mass[i], s, h.spin_basis)); break;   // v-bar, row
      }
      if (i == h.ward_leg && (P.kind[i] == G_IN || P.kind[i] == G_OUT)) E.eps[i][s] = tocomplex(E.p[i]);
    }
  }
}

// tier 0 (me_tier0.cpp)
cd tier0_amplitude(const me_handle_ref& h, const Ext& E, const int* hel, const int* col);
double tier0_me2(const me_handle_ref& h, const double* mom);
// tier 1 (me_tier1.cpp)
std::shared_ptr<Tier1> tier1_build(const Process& P);
double tier1_me2(const me_handle_ref& h, const double* mom);
void tier1_flows(const me_handle_ref& h, const Ext& E, const int* hel, cd* J /*[n_flow]*/);
int tier1_n_diagrams(const Tier1& t);
int tier1_n_terms(const Tier1& t);
int tier1_n_4g_diagrams(const Tier1& t);
int tier1_n_flows(const Tier1& t);
const double* tier1_cf(const Tier1& t);          // [n_flow][n_flow], row-major
const int* tier1_flow_perms(const Tier1& t);     // [n_flow][n_gluon] leg indices, lexicographic
// tier 1, diagram basis (me_tier1g.cpp)
std::shared_ptr<Tier1G> tier1g_build(const Process& P);
double tier1g_me2(const me_handle_ref& h, const Tier1G& T, const double* mom);
cd tier1g_amplitude(const me_handle_ref& h, const Tier1G& T, const Ext& E, const int* hel, const int* col);
int tier1g_n_diagrams(const Tier1G& t);
int tier1g_n_terms(const Tier1G& t);
int tier1g_n_4g_diagrams(const Tier1G& t);
// QED literal (me_qed.cpp)
double qed_me2(const me_handle_ref& h, const double* mom);

}  // namespace orc
