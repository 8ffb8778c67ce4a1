// ORACLE — TEST INFRASTRUCTURE ONLY (see algebra.hpp header).
//
// me_qed.cpp — e- e+ -> mu- mu+ at tree level, massless, single s-channel photon
// (BASELINE.json:configs[0]).  One diagram, written out literally with explicit spinors
// and gamma matrices (vertex i e Q gamma^mu, photon propagator
// -i g_{mu nu}/q^2):
//     iM = [vbar(p2) (i e Q gamma^mu) u(p1)] (-i g_{mu nu} / s) [ubar(p3) (i e Q gamma^nu) v(p4)]
//     me2 = (1/4) sum over the 16 spin combinations of |M|^2
// Q = -1 for e and mu; the sign drops out of |M|^2.
// Pinned by the closed form 2 e^4 (t^2+u^2)/s^2 in tests/test_oracle_me.py.
#include "me_ref.hpp"

namespace orc {

double qed_me2(const me_handle_ref& h, const double* mom) {
  const Process& P = h.P;
  Ext E;
  build_ext(h, mom, E);
  const Gammas& G = gammas();
  const P4 q = E.p[0] + E.p[1];
  const double s = mdot(q, q);
  const cd vtx = cd(0, 1) * P.ee * (-1.0);
  double total = 0;
  for (int s1 = 0; s1 < 2; ++s1)
    for (int s2 = 0; s2 < 2; ++s2)
      for (int s3 = 0; s3 < 2; ++s3)
        for (int s4 = 0; s4 < 2; ++s4) {
          V4 Le, Lm;  // upper-index currents
          for (int mu = 0; mu < 4; ++mu) {
            Le[mu] = vtx * dot(E.sp[1][s2], mul(G.g[mu], E.sp[0][s1]));   // vbar(e+) gamma^mu u(e-)
            Lm[mu] = vtx * dot(E.sp[2][s3], mul(G.g[mu], E.sp[3][s4]));   // ubar(mu-) gamma^mu v(mu+)
          }
          const cd M = (cd(0, -1) / s) * mdot(Le, Lm);
          total += std::norm(M);
        }
  return total / P.avg;
}

}  // namespace orc
