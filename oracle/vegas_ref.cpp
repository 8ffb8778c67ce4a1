// ORACLE — TEST INFRASTRUCTURE ONLY (see algebra.hpp header).
//
// vegas_ref.cpp — Vegas (Lepage 1978; refs [7,8] of the paper; the paper
// uses it through VegasFlow, with "the events ... computed in parallel").
// The paper fixes no detail; this follows SURVEY.md §8(c) G7 step by step:
//   (1) map y_d -> x_d through the per-dimension piecewise-linear grid, jac = prod_d N_b dx_{d,i}
//   (3) I = (1/N) sum f,  sigma^2 = [(1/N) sum f^2 - I^2]/(N-1)
//   (4) S_{d,i} = sum over events with bin_d = i of f^2
//   (5) smooth (3-point), normalise, damp w = [(r-1)/ln r]^alpha, re-bin to equal damped weight
// Plain sequential sums in event order.
#include <cmath>
#include <vector>

namespace orc {

// (1) one point.  edges: [n_dim][n_bins+1].  Returns the jacobian; writes x[n_dim], idx[n_dim].
double vegas_map_point(const double* edges, int n_dim, int n_bins, const double* y, double* x, int* idx) {
  double jac = 1;
  for (int d = 0; d < n_dim; ++d) {
    const double* e = edges + size_t(d) * (n_bins + 1);
    const double t = y[d] * n_bins;
    int i = int(std::floor(t));
    if (i > n_bins - 1) i = n_bins - 1;
    if (i < 0) i = 0;
    const double w = e[i + 1] - e[i];
    x[d] = e[i] + (t - i) * w;
    jac *= n_bins * w;
    idx[d] = i;
  }
  return jac;
}

// (5) refine one dimension in place.  S[n_bins] = accumulated f^2 per bin.
void vegas_refine_dim(double* e /*[n_bins+1]*/, const double* S, int n_bins, double alpha) {
  std::vector<double> s(n_bins), w(n_bins), ne(n_bins + 1);
  if (n_bins == 1) return;
  s[0] = (S[0] + S[1]) / 2;
  for (int i = 1; i < n_bins - 1; ++i) s[i] = (S[i - 1] + S[i] + S[i + 1]) / 3;
  s[n_bins - 1] = (S[n_bins - 2] + S[n_bins - 1]) / 2;
  double tot = 0;
  for (int i = 0; i < n_bins; ++i) tot += s[i];
  if (!(tot > 0)) return;  // nothing accumulated: leave the grid alone
  double wtot = 0;
  for (int i = 0; i < n_bins; ++i) {
    const double r = s[i] / tot;
    if (r <= 0) w[i] = 0;
    else if (r == 1.0) w[i] = 1;
    else w[i] = std::pow((r - 1) / std::log(r), alpha);
    wtot += w[i];
  }
  const double target = wtot / n_bins;
  ne[0] = 0; ne[n_bins] = 1;
  int j = 0; double acc = 0;  // acc = damped weight of old bins 0..j-1
  for (int i = 1; i < n_bins; ++i) {
    const double need = i * target;
    while (j < n_bins - 1 && acc + w[j] < need) { acc += w[j]; ++j; }
    const double frac = (w[j] > 0) ? (need - acc) / w[j] : 0.0;
    ne[i] = e[j] + frac * (e[j + 1] - e[j]);
  }
  for (int i = 0; i <= n_bins; ++i) e[i] = ne[i];
}

}  // namespace orc
