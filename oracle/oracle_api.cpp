// ORACLE — TEST INFRASTRUCTURE ONLY (see algebra.hpp / oracle_ref.h headers).
//
// oracle_api.cpp — the extern "C" surface of the oracle: argument checks, loops over events
// (OpenMP over events only, static schedule), and the Vegas integrand of SURVEY.md §8(c) G6.
#define ME_PARAMS_REF_DEFINED
#include "me_ref.hpp"
#include "oracle_ref.h"
#ifdef _OPENMP
#include <omp.h>
#endif

namespace orc {
void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
void philox_uniforms(uint64_t seed, uint64_t iteration, uint64_t event, int n_dim, double* u);
double rambo_event(const double* r, double sqrt_s, const double* m, int n, int ps_mode, double* mom);
int passes_cuts(const double* mom, int n, const int* is_gluon, double ptj_min, double dr_min);
double vegas_map_point(const double* edges, int n_dim, int n_bins, const double* y, double* x, int* idx);
void vegas_refine_dim(double* e, const double* S, int n_bins, double alpha);
}  // namespace orc
using namespace orc;

static int g_threads = 0;  // 0 = OpenMP default

// tier 1 of a QCD process: the flow basis (one quark line) or the diagram basis (two lines)
static double me2_tier1(const me_handle_ref& h, const double* mom) {
  return h.t1 ? tier1_me2(h, mom) : tier1g_me2(h, *h.t1g, mom);
}
// the final-state partons the jet cuts apply to: gluons, and the massless final quark of q g -> t tbar q (g)
static bool is_jet(const Process& P, int leg) {
  return P.kind[leg] == G_OUT || ((P.kind[leg] == Q_OUT || P.kind[leg] == QB_OUT) && P.mass[leg] == 0.0);
}

extern "C" {

void oracle_set_threads_ref(int n) { g_threads = n; }
int oracle_get_threads_ref(void) {
#ifdef _OPENMP
  return g_threads > 0 ? g_threads : omp_get_max_threads();
#else
  return 1;
#endif
}

int me_init_ref(const char* process, const me_params_ref* p, me_handle_ref** out) {
  if (!process || !p || !out) return -1;
  if (p->w_top != 0.0) return -3;  // no width in any propagator
  auto* h = new me_handle_ref();
  h->par = *p;
  if (!make_process(process, *p, h->P)) { delete h; return -2; }
  if (!h->P.qed) {
    if (h->P.n_lines() > 1) h->t1g = tier1g_build(h->P);   // two quark lines: the diagram basis (me_tier1g.cpp)
    else h->t1 = tier1_build(h->P);
  }
  *out = h;
  return 0;
}
void me_free_ref(me_handle_ref* h) { delete h; }
int me_n_external_ref(const me_handle_ref* h) { return h ? h->P.n_ext : -1; }
int me_n_final_ref(const me_handle_ref* h) { return h ? h->P.n_ext - 2 : -1; }

int me_eval_ref(me_handle_ref* h, const double* momenta, double* me2, long long n_ev) {
  if (!h || !momenta || !me2 || n_ev < 0) return -1;
  const int stride = 4 * h->P.n_ext;
  const int nt = oracle_get_threads_ref();
#pragma omp parallel for schedule(static) num_threads(nt)
  for (long long e = 0; e < n_ev; ++e)
    me2[e] = h->P.qed ? qed_me2(*h, momenta + e * stride) : me2_tier1(*h, momenta + e * stride);
  return 0;
}

// tier 1 in the diagram basis for ANY QCD process (the default of the two-line processes; for the one-line ones a
// second, independent organisation of the same diagrams that the tests compare with the flow basis)
int me_eval_diag_ref(me_handle_ref* h, const double* momenta, double* me2, long long n_ev) {
  if (!h || !momenta || !me2 || n_ev < 0 || h->P.qed) return -1;
  if (!h->t1g) h->t1g = tier1g_build(h->P);
  const int stride = 4 * h->P.n_ext;
  const int nt = oracle_get_threads_ref();
#pragma omp parallel for schedule(static) num_threads(nt)
  for (long long e = 0; e < n_ev; ++e) me2[e] = tier1g_me2(*h, *h->t1g, momenta + e * stride);
  return 0;
}
int me_amplitude_diag_ref(me_handle_ref* h, const double* mom, const int* hel, const int* col, double* re_im) {
  if (!h || h->P.qed) return -1;
  if (!h->t1g) h->t1g = tier1g_build(h->P);
  Ext E; build_ext(*h, mom, E);
  const cd a = tier1g_amplitude(*h, *h->t1g, E, hel, col);
  re_im[0] = a.real(); re_im[1] = a.imag();
  return 0;
}

int me_eval_def_ref(me_handle_ref* h, const double* momenta, double* me2, long long n_ev) {
  if (!h || !momenta || !me2 || n_ev < 0) return -1;
  const int stride = 4 * h->P.n_ext;
#ifdef _OPENMP
  omp_set_num_threads(oracle_get_threads_ref());
#endif
  for (long long e = 0; e < n_ev; ++e)  // the colour loop inside is the parallel one
    me2[e] = h->P.qed ? qed_me2(*h, momenta + e * stride) : tier0_me2(*h, momenta + e * stride);
  return 0;
}

int me_set_basis_ref(me_handle_ref* h, int spin_basis, int pol_basis) {
  if (!h) return -1;
  h->spin_basis = spin_basis; h->pol_basis = pol_basis;
  return 0;
}
int me_set_ward_leg_ref(me_handle_ref* h, int leg) { if (!h) return -1; h->ward_leg = leg; return 0; }

int me_info_ref(const me_handle_ref* h, int what) {
  if (!h) return -1;
  if (h->P.qed) return what == 0 || what == 1 || what == 3 ? 1 : 0;
  if (what >= 5 && what <= 7 && !h->t1g) return -1;
  switch (what) {
    case 0: return h->t1 ? tier1_n_diagrams(*h->t1) : tier1g_n_diagrams(*h->t1g);
    case 1: return h->t1 ? tier1_n_terms(*h->t1) : tier1g_n_terms(*h->t1g);
    case 2: return h->t1 ? tier1_n_4g_diagrams(*h->t1) : tier1g_n_4g_diagrams(*h->t1g);
    case 3: return h->t1 ? tier1_n_flows(*h->t1) : 0;   // the diagram basis has no flows
    case 4: return h->P.n_gluon();
    case 5: return tier1g_n_diagrams(*h->t1g);           // the diagram-basis counts, where it has been built
    case 6: return tier1g_n_terms(*h->t1g);
    case 7: return tier1g_n_4g_diagrams(*h->t1g);
  }
  return -1;
}
int me_colour_matrix_ref(const me_handle_ref* h, double* cf) {
  if (!h || !cf || h->P.qed || !h->t1) return -1;
  const int nf = tier1_n_flows(*h->t1);
  for (int i = 0; i < nf * nf; ++i) cf[i] = tier1_cf(*h->t1)[i];
  return 0;
}
int me_flow_perms_ref(const me_handle_ref* h, int* perms) {
  if (!h || !perms || h->P.qed || !h->t1) return -1;
  const int n = tier1_n_flows(*h->t1) * h->P.n_gluon();
  for (int i = 0; i < n; ++i) perms[i] = tier1_flow_perms(*h->t1)[i];
  return 0;
}
int me_amplitude_def_ref(me_handle_ref* h, const double* mom, const int* hel, const int* col, double* re_im) {
  if (!h || h->P.qed) return -1;
  Ext E; build_ext(*h, mom, E);
  const cd a = tier0_amplitude(*h, E, hel, col);
  re_im[0] = a.real(); re_im[1] = a.imag();
  return 0;
}
// The tier-0 amplitude with the external wavefunctions STRIPPED: T[i_0][i_1]...[i_{n-1}] = amplitude with leg l carrying the
// unit wavefunction e_{i_l} (spinor component or Lorentz index), for all-incoming momenta k that need not be physical
// (negative energies allowed: the amplitude is a rational function of k).  The amplitude is multilinear in the
// wavefunctions, so spin sums can be done with completeness relations outside — which is what crossing needs
// (tests/test_oracle_quark_channels.py).  T: [4^n][2], leg 0 slowest.
int me_open_tensor_ref(me_handle_ref* h, const double* k, const int* col, double* T) {
  if (!h || h->P.qed || !k || !col || !T) return -1;
  const int n = h->P.n_ext;
  Ext E;
  E.n = n;
  for (int i = 0; i < n; ++i)
    for (int mu = 0; mu < 4; ++mu) { E.k[i][mu] = k[4 * i + mu]; E.p[i][mu] = (i < 2 ? 1.0 : -1.0) * k[4 * i + mu]; }
  long long total = 1;
  for (int i = 0; i < n; ++i) total *= 4;
  int hel[NMAX] = {0};
  for (long long t = 0; t < total; ++t) {
    long long r = t;
    for (int i = n - 1; i >= 0; --i) {
      const int c = int(r % 4); r /= 4;
      for (int m = 0; m < 4; ++m) { E.eps[i][0][m] = (m == c) ? 1.0 : 0.0; E.sp[i][0][m] = (m == c) ? 1.0 : 0.0; }
    }
    const cd a = tier0_amplitude(*h, E, hel, col);
    T[2 * t] = a.real(); T[2 * t + 1] = a.imag();
  }
  return 0;
}
int me_flows_ref(me_handle_ref* h, const double* mom, const int* hel, double* J) {
  if (!h || h->P.qed || !h->t1) return -1;
  Ext E; build_ext(*h, mom, E);
  std::vector<cd> j(tier1_n_flows(*h->t1));
  tier1_flows(*h, E, hel, j.data());
  for (size_t f = 0; f < j.size(); ++f) { J[2 * f] = j[f].real(); J[2 * f + 1] = j[f].imag(); }
  return 0;
}
int su3_generators_ref(double* T, double* f) {
  const SU3& S = su3();
  for (int a = 0; a < 8; ++a)
    for (int i = 0; i < 3; ++i)
      for (int j = 0; j < 3; ++j) {
        T[((a * 3 + i) * 3 + j) * 2] = S.T[a].m[i][j].real();
        T[((a * 3 + i) * 3 + j) * 2 + 1] = S.T[a].m[i][j].imag();
      }
  for (int a = 0; a < 8; ++a) for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) f[(a * 8 + b) * 8 + c] = S.f[a][b][c];
  return 0;
}
int wavefunction_ref(int kind, const double* p, double mass, int s, int basis, double* out) {
  const P4 P = {{p[0], p[1], p[2], p[3]}};
  cd c[4];
  if (kind == 0) { Sp u = u_spinor(P, mass, s, basis); for (int i = 0; i < 4; ++i) c[i] = u[i]; }
  else if (kind == 1) { Sp v = v_spinor(P, mass, s, basis); for (int i = 0; i < 4; ++i) c[i] = v[i]; }
  else if (kind == 2) { V4 e = polvec(P, s, basis); for (int i = 0; i < 4; ++i) c[i] = e[i]; }
  else return -1;
  for (int i = 0; i < 4; ++i) { out[2 * i] = c[i].real(); out[2 * i + 1] = c[i].imag(); }
  return 0;
}

int philox_raw_ref(const uint32_t* ctr, const uint32_t* key, uint32_t* out) { philox4x32_10(ctr, key, out); return 0; }
int philox_uniform_ref(uint64_t seed, uint64_t iteration, long long first_event, int n_dim, double* rand, long long n_ev) {
  if (!rand || n_ev < 0 || n_dim < 1) return -1;
  for (long long e = 0; e < n_ev; ++e) philox_uniforms(seed, iteration, uint64_t(first_event + e), n_dim, rand + e * n_dim);
  return 0;
}
int rambo_generate_ref(const double* rand, double sqrt_s, const double* masses, int n_final, int ps_mode,
                       double* momenta, double* weights, long long n_ev) {
  if (!rand || !masses || !momenta || !weights || n_ev < 0 || n_final < 2 || n_final > NMAX_FINAL) return -1;
  const int nd = ps_mode == 0 ? 4 * n_final : 3 * n_final - 4;
  for (long long e = 0; e < n_ev; ++e)
    weights[e] = rambo_event(rand + e * nd, sqrt_s, masses, n_final, ps_mode, momenta + e * 4 * (n_final + 2));
  return 0;
}
int cuts_ref(const double* momenta, int n_final, const int* is_gluon, double ptj_min, double dr_min, int* pass, long long n_ev) {
  if (!momenta || !is_gluon || !pass) return -1;
  for (long long e = 0; e < n_ev; ++e) pass[e] = passes_cuts(momenta + e * 4 * (n_final + 2), n_final, is_gluon, ptj_min, dr_min);
  return 0;
}

int vegas_map_ref(const double* edges, int n_dim, int n_bins, const double* y, double* x, double* jac, int* idx, long long n) {
  for (long long e = 0; e < n; ++e) jac[e] = vegas_map_point(edges, n_dim, n_bins, y + e * n_dim, x + e * n_dim, idx + e * n_dim);
  return 0;
}
int vegas_accumulate_ref(const double* f, const int* idx, int n_dim, int n_bins, long long n, double* sums) {
  for (int i = 0; i < 3 + n_dim * n_bins; ++i) sums[i] = 0;
  for (long long e = 0; e < n; ++e) {
    sums[0] += f[e]; sums[1] += f[e] * f[e];
    if (f[e] != 0.0) sums[2] += 1;
    for (int d = 0; d < n_dim; ++d) sums[3 + d * n_bins + idx[e * n_dim + d]] += f[e] * f[e];
  }
  return 0;
}
int vegas_refine_ref(double* edges, int n_dim, int n_bins, const double* S, double alpha) {
  for (int d = 0; d < n_dim; ++d) vegas_refine_dim(edges + size_t(d) * (n_bins + 1), S + size_t(d) * n_bins, n_bins, alpha);
  return 0;
}

// Toy gluon density of the hadronic mode (reading R-N3): g(x) = 3 x^-1.2 (1-x)^5.
// A DECLARED toy parametrisation (no LHAPDF grids in the container); it only has to be the same on both sides.
static double toy_gluon_density(double x) { return 3.0 * std::pow(x, -1.2) * std::pow(1.0 - x, 5); }
// The beams of the quark-initiated channels (SURVEY §8(f) N1 x N3): DECLARED toys as well, a valence-like quark density
// q(x) = 2 x^-0.5 (1-x)^3 and a sea-like antiquark density qbar(x) = 0.3 x^-1.1 (1-x)^7.
static double toy_density(int leg_kind, double x) {
  if (leg_kind == F_IN) return 2.0 * std::pow(x, -0.5) * std::pow(1.0 - x, 3);
  if (leg_kind == FB_IN) return 0.3 * std::pow(x, -1.1) * std::pow(1.0 - x, 7);
  return toy_gluon_density(x);
}

// f(x) = jac_Vegas * W_ps * Theta_cuts * me2 / (2 s) * C,  C = 0.3893793721e9 pb GeV^2
// ps_mode 2 (hadronic, D = 3n-4+2): x_1 = x[0], x_2 = x[1] are the momentum fractions, s_hat = x_1 x_2 s, the remaining
// 3n-4 coordinates drive RAMBO "on diet" at sqrt(s_hat) in the partonic centre-of-mass frame (p_T, rapidity differences
// and azimuths — everything the cuts use — are invariant under the boost along z), and
// f = jac g(x_1) g(x_2) W_ps(s_hat) Theta me2 / (2 s_hat) C; events with sqrt(s_hat) <= sum of the final masses give 0.
int vegas_integrand_ref(me_handle_ref* h, const vegas_grid_ref* g, double sqrt_s, long long first_event, long long n_ev,
                        double* sums, double* f_out) {
  if (!h || !g || !sums || h->P.qed) return -1;
  const int nf = h->P.n_ext - 2, D = g->n_dim, nb = g->n_bins;
  if (g->ps_mode < 0 || g->ps_mode > 2) return -4;
  if (D != (g->ps_mode == 0 ? 4 * nf : g->ps_mode == 1 ? 3 * nf - 4 : 3 * nf - 2)) return -4;
  std::vector<double> masses(nf); std::vector<int> isg(nf);
  for (int i = 0; i < nf; ++i) { masses[i] = h->P.mass[2 + i]; isg[i] = is_jet(h->P, 2 + i); }
  std::vector<double> f(n_ev); std::vector<int> idx(size_t(n_ev) * D);
  const double conv = 0.3893793721e9, flux = 1.0 / (2.0 * sqrt_s * sqrt_s);
  const int nt = oracle_get_threads_ref();
#pragma omp parallel for schedule(static) num_threads(nt)
  for (long long e = 0; e < n_ev; ++e) {
    double y[4 * NMAX_FINAL], x[4 * NMAX_FINAL], mom[4 * NMAX];
    philox_uniforms(g->seed, uint64_t(g->iteration), uint64_t(first_event + e), D, y);
    const double jac = vegas_map_point(g->edges, D, nb, y, x, idx.data() + e * D);
    double val = 0;
    if (g->ps_mode == 2) {
      double msum = 0;
      for (int i = 0; i < nf; ++i) msum += masses[i];
      const double rs_hat = std::sqrt(x[0] * x[1]) * sqrt_s;
      if (rs_hat > msum) {
        const double wps = rambo_event(x + 2, rs_hat, masses.data(), nf, 1, mom);
        if (passes_cuts(mom, nf, isg.data(), h->par.ptj_min, h->par.dr_min))
          val = jac * toy_density(h->P.kind[0], x[0]) * toy_density(h->P.kind[1], x[1]) * wps * me2_tier1(*h, mom) / (2.0 * rs_hat * rs_hat) * conv;
      }
    } else {
      const double wps = rambo_event(x, sqrt_s, masses.data(), nf, g->ps_mode, mom);
      if (passes_cuts(mom, nf, isg.data(), h->par.ptj_min, h->par.dr_min))
        val = jac * wps * me2_tier1(*h, mom) * flux * conv;
    }
    f[e] = val;
  }
  vegas_accumulate_ref(f.data(), idx.data(), D, nb, n_ev, sums);
  if (f_out) for (long long e = 0; e < n_ev; ++e) f_out[e] = f[e];
  return 0;
}

int vegas_iterate_ref(me_handle_ref* h, vegas_grid_ref* g, double sqrt_s, long long n_ev, vegas_result_ref* result) {
  if (!h || !g || !result || n_ev < 2) return -1;
  std::vector<double> sums(3 + g->n_dim * g->n_bins);
  const int rc = vegas_integrand_ref(h, g, sqrt_s, 0, n_ev, sums.data(), nullptr);
  if (rc) return rc;
  const double N = double(n_ev), I = sums[0] / N;
  result->integral = I;
  result->variance = (sums[1] / N - I * I) / (N - 1);
  result->sum_w = sums[0]; result->sum_w2 = sums[1]; result->n_pass = (long long)sums[2];
  vegas_refine_ref(g->edges, g->n_dim, g->n_bins, sums.data() + 3, g->alpha);
  g->iteration += 1;
  return 0;
}

// Unweighted events ("the step behind the path").  Hit-or-miss: event e of the iteration is kept iff
// f_e > 0 and u_e w_max < f_e, with u_e the Philox uniform of counter (event lo, event hi, 0x7fffffff, iteration),
// words 0-1 — a pair index no phase-space dimension reaches (D <= 24 uses pair indices 0..11), so the decision is
// independent of the kinematics.  accepted: global indices in ascending order; counts = (kept, f > w_max).
int vegas_unweight_ref(const double* f, long long n_ev, double w_max, uint64_t seed, uint64_t iteration, long long first_event,
                       long long* accepted, long long* counts) {
  if (!counts || n_ev < 0 || !(w_max > 0) || (n_ev > 0 && (!f || !accepted))) return -1;
  counts[0] = counts[1] = 0;
  const uint32_t key[2] = {uint32_t(seed), uint32_t(seed >> 32)};
  for (long long e = 0; e < n_ev; ++e) {
    if (f[e] > w_max) counts[1] += 1;
    if (!(f[e] > 0)) continue;
    const uint64_t ev = uint64_t(first_event + e);
    const uint32_t ctr[4] = {uint32_t(ev), uint32_t(ev >> 32), 0x7fffffffu, uint32_t(iteration)};
    uint32_t o[4];
    philox4x32_10(ctr, key, o);
    const uint64_t bits = (uint64_t(o[0]) << 32 | o[1]) >> 11;
    const double u = (double(bits) + 0.5) * (1.0 / 9007199254740992.0);
    if (u * w_max < f[e]) accepted[counts[0]++] = first_event + e;
  }
  return 0;
}

// The kinematics of listed events of iteration g->iteration on grid g: momenta [n][n_ext][4] (partonic centre-of-mass
// frame, incoming legs filled in) and weights jac W_ps C/(2 s_hat) (times the toy densities in ps_mode 2) — the
// integrand of vegas_integrand_ref without |M|^2 and without the cuts.
int vegas_generate_ref(me_handle_ref* h, const vegas_grid_ref* g, double sqrt_s, const long long* ids, long long n, double* momenta,
                       double* weights) {
  if (!h || !g || n < 0 || (n > 0 && (!ids || !momenta || !weights)) || h->P.qed) return -1;
  const int nf = h->P.n_ext - 2, D = g->n_dim, nb = g->n_bins;
  if (D != (g->ps_mode == 0 ? 4 * nf : g->ps_mode == 1 ? 3 * nf - 4 : 3 * nf - 2)) return -4;
  std::vector<double> masses(nf);
  double msum = 0;
  for (int i = 0; i < nf; ++i) { masses[i] = h->P.mass[2 + i]; msum += masses[i]; }
  const double conv = 0.3893793721e9;
  std::vector<int> idx(D);
  for (long long k = 0; k < n; ++k) {
    double y[4 * NMAX_FINAL], x[4 * NMAX_FINAL];
    double* mom = momenta + k * 4 * (nf + 2);
    philox_uniforms(g->seed, uint64_t(g->iteration), uint64_t(ids[k]), D, y);
    const double jac = vegas_map_point(g->edges, D, nb, y, x, idx.data());
    if (g->ps_mode == 2) {
      const double rs_hat = std::sqrt(x[0] * x[1]) * sqrt_s;
      if (rs_hat > msum) {
        weights[k] = jac * toy_density(h->P.kind[0], x[0]) * toy_density(h->P.kind[1], x[1]) * rambo_event(x + 2, rs_hat, masses.data(), nf, 1, mom) /
                     (2.0 * rs_hat * rs_hat) * conv;
      } else {
        weights[k] = 0;
        for (int i = 0; i < 4 * (nf + 2); ++i) mom[i] = 0;
        mom[0] = mom[3] = mom[4] = 0.5 * rs_hat; mom[7] = -0.5 * rs_hat;
      }
    } else {
      weights[k] = jac * rambo_event(x, sqrt_s, masses.data(), nf, g->ps_mode, mom) / (2.0 * sqrt_s * sqrt_s) * conv;
    }
  }
  return 0;
}

}  // extern "C"
