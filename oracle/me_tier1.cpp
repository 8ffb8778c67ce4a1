// ORACLE — TEST INFRASTRUCTURE ONLY (see algebra.hpp header).
//
// me_tier1.cpp — TIER 1, "diagrammatic scalar" (SURVEY.md §8(c) tier 1, D, E, F).
// This is the per-event parity reference and the timed CPU baseline.  It follows the
// method of BASELINE.json:north_star step by step:
//   a5  external wavefunctions (both spin states of each leg)            [wavefunctions.hpp]
//   a6  off-shell currents: vertex x propagator, chained over every Feynman diagram
//   a7  one complex amplitude per colour-pure diagram term
//   a8  colour-flow vector  J_sigma += c_{sigma,k} A_k,  c in {+-1, +-i}
//   a9  sum_col |M|^2 = J^dagger CF J,  CF_{sigma tau} = Tr(T^sigma (T^tau)^dagger)
//   a10 sum over helicities, divide by S
//
// Diagram enumeration.  With one quark line every tree diagram is: the
// quark line running from the outgoing t to the outgoing tbar, with gluon subtrees attached
// to it in some order.  So   diagrams  =  ordered partitions of the gluon set into blocks
// x for each block, every rooted gluon tree on that block (internal nodes = ggg vertex with
// 2 children or gggg vertex with 3 children; unordered children => each diagram once).
// A gggg vertex carries three colour (x) Lorentz terms; a "term" is a
// diagram with one of the three picked at every gggg vertex, so that a term is colour-pure.
// Pins: 3 / 16 / 123 diagrams, 1 / 18 of them with a gggg vertex, 3 / 18 / 159 terms.
//
// Colour ("Diagram -> flows").  A gluon subtree whose off-shell line carries
// adjoint index c, contracted with T^c on the quark line, is a polynomial in words over its
// leaves.  Using f^{abc} T^c = -i [T^a, T^b]:
//   leaf a                               -> the word (a)
//   ggg node, legs (X, Y, off-shell c), colour f^{x y c}                  -> -i [X, Y]
//   gggg node, legs (X,Y,Z, off-shell d):
//        term 0  f^{xye} f^{zde}  ->  -[[X,Y],Z]
//        term 1  f^{xze} f^{yde}  ->  -[[X,Z],Y]
//        term 2  f^{xde} f^{yze}  ->  -[[Y,Z],X]
// and the quark line concatenates the polynomials of its attachments from the t end to the
// tbar end.  Each resulting word is a permutation sigma of the gluons = one colour flow.
//
// Kinematic part of a term (Feynman rules of SURVEY §8(c) C, colour stripped):
//   gluon node (X,Y):   J = (-i/K^2) g_s [ (JX.JY)(kX-kY) + JY ((kY-k3).JX) + JX ((k3-kX).JY) ],  k3 = -(kX+kY)
//   gluon node (X,Y,Z): J = (-i/K^2) (-i g_s^2) * { (JX.JZ) JY - (JY.JZ) JX      term 0
//                                                   (JX.JY) JZ - (JY.JZ) JX      term 1
//                                                   (JX.JY) JZ - (JX.JZ) JY      term 2 }
//   quark line: A = ubar (i g_s J1slash) S(q1) (i g_s J2slash) S(q2) ... (i g_s Jmslash) v,
//               S(q) = i (qslash + m)/(q^2 - m^2),  q_k = k_tbar + sum_{l>k} K_l  (along the arrow)
// Generic 4x4 matrix algebra in the Dirac representation; no blocking, no fusion.
#include <algorithm>
#include <set>
#include "me_ref.hpp"

namespace orc {

// ---- polynomials in words over gluon legs ------------------------------------------------
using Word = std::vector<int>;
struct Poly {
  std::map<Word, cd> t;
};
static Poly pmul(const Poly& a, const Poly& b) {
  Poly r;
  for (auto& x : a.t)
    for (auto& y : b.t) {
      Word w = x.first;
      w.insert(w.end(), y.first.begin(), y.first.end());
      r.t[w] += x.second * y.second;
    }
  return r;
}
static Poly padd(const Poly& a, const Poly& b, cd cb) {
  Poly r = a;
  for (auto& y : b.t) r.t[y.first] += cb * y.second;
  return r;
}
static Poly pscale(const Poly& a, cd c) {
  Poly r;
  for (auto& x : a.t) r.t[x.first] = c * x.second;
  return r;
}
static Poly pcomm(const Poly& a, const Poly& b) { return padd(pmul(a, b), pmul(b, a), cd(-1)); }

// ---- colour-pure gluon subtree -----------------------------------------------------------
struct GNode {
  unsigned mask = 0;  // leaf set, bit i = leg i
  int kind = 0;       // 0 leaf, 1 ggg node, 2/3/4 gggg node term 0/1/2
  int ch[3] = {-1, -1, -1};
  int leg = -1;
  int shape = -1;  // id of the underlying diagram shape (gggg term forgotten)
  int n4g = 0;
  Poly colour;
};

struct TrieNode {
  int gnode = -1;
  unsigned mask_after = 0;  // gluon legs absorbed so far, this node included
  std::vector<int> child;
  std::vector<int> terms;  // terms whose attachment sequence ends here
};

struct Tier1 {
  Process P;
  std::vector<int> gl;  // gluon leg indices, ascending
  int leg_t = -1, leg_tb = -1;
  std::vector<GNode> nodes;
  std::map<unsigned, std::vector<int>> trees;  // leaf set -> node ids
  std::map<std::vector<int>, int> shape_ids;
  std::vector<std::vector<int>> terms;  // attachment sequence (node ids) from the t end
  int n_diag = 0, n_diag4g = 0;
  std::vector<TrieNode> trie;  // root = 0, sequences stored from the tbar end
  int n_flow = 0;
  std::vector<int> perms;              // [n_flow][n_g]
  std::vector<std::vector<cd>> W;      // [term][flow]
  std::vector<double> CF;              // [n_flow][n_flow]

  int shape_of(const std::vector<int>& key) {
    auto it = shape_ids.find(key);
    if (it != shape_ids.end()) return it->second;
    int id = int(shape_ids.size());
    shape_ids[key] = id;
    return id;
  }
  const std::vector<int>& trees_of(unsigned S);
  void enum_terms(unsigned rest, std::vector<int>& seq);
  void build();
};

const std::vector<int>& Tier1::trees_of(unsigned S) {
  auto it = trees.find(S);
  if (it != trees.end()) return it->second;
  std::vector<int> out;
  if (__builtin_popcount(S) == 1) {
    GNode g;
    g.mask = S; g.kind = 0; g.leg = __builtin_ctz(S);
    g.shape = shape_of({0, g.leg});
    g.colour.t[Word{g.leg}] = 1;
    nodes.push_back(g);
    out.push_back(int(nodes.size()) - 1);
  } else {
    const unsigned low = S & (~S + 1u);
    for (unsigned A = (S - 1) & S; A; A = (A - 1) & S) {
      if (!(A & low)) continue;
      const unsigned B = S & ~A;
      const std::vector<int> ta = trees_of(A), tb = trees_of(B);
      for (int x : ta)
        for (int y : tb) {
          GNode g;
          g.mask = S; g.kind = 1; g.ch[0] = x; g.ch[1] = y;
          g.shape = shape_of({1, nodes[x].shape, nodes[y].shape});
          g.n4g = nodes[x].n4g + nodes[y].n4g;
          g.colour = pscale(pcomm(nodes[x].colour, nodes[y].colour), cd(0, -1));  // -i [X,Y]
          nodes.push_back(g);
          out.push_back(int(nodes.size()) - 1);
        }
    }
    for (unsigned A = (S - 1) & S; A; A = (A - 1) & S) {
      if (!(A & low)) continue;
      const unsigned R = S & ~A;
      const unsigned lowR = R & (~R + 1u);
      for (unsigned B = (R - 1) & R; B; B = (B - 1) & R) {
        if (!(B & lowR)) continue;
        const unsigned C = R & ~B;
        if (!C) continue;
        const std::vector<int> ta = trees_of(A), tb = trees_of(B), tc = trees_of(C);
        for (int x : ta)
          for (int y : tb)
            for (int z : tc)
              for (int k = 0; k < 3; ++k) {
                GNode g;
                g.mask = S; g.kind = 2 + k; g.ch[0] = x; g.ch[1] = y; g.ch[2] = z;
                g.shape = shape_of({2, nodes[x].shape, nodes[y].shape, nodes[z].shape});
                g.n4g = 1 + nodes[x].n4g + nodes[y].n4g + nodes[z].n4g;
                const Poly &X = nodes[x].colour, &Y = nodes[y].colour, &Z = nodes[z].colour;
                if (k == 0) g.colour = pscale(pcomm(pcomm(X, Y), Z), cd(-1));  // -[[X,Y],Z]
                if (k == 1) g.colour = pscale(pcomm(pcomm(X, Z), Y), cd(-1));  // -[[X,Z],Y]
                if (k == 2) g.colour = pscale(pcomm(pcomm(Y, Z), X), cd(-1));  // -[[Y,Z],X]
                nodes.push_back(g);
                out.push_back(int(nodes.size()) - 1);
              }
      }
    }
  }
  trees[S] = out;
  return trees[S];
}

void Tier1::enum_terms(unsigned rest, std::vector<int>& seq) {
  if (!rest) { terms.push_back(seq); return; }
  for (unsigned A = rest; A; A = (A - 1) & rest) {  // first block (ordered partition: no dedupe)
    const std::vector<int> ta = trees_of(A);
    for (int x : ta) {
      seq.push_back(x);
      enum_terms(rest & ~A, seq);
      seq.pop_back();
    }
  }
}

void Tier1::build() {
  for (int i = 0; i < P.n_ext; ++i) {
    if (P.kind[i] == G_IN || P.kind[i] == G_OUT) gl.push_back(i);
    if (P.kind[i] == Q_OUT) leg_t = i;
    if (P.kind[i] == QB_OUT) leg_tb = i;
  }
  unsigned gmask = 0;
  for (int g : gl) gmask |= 1u << g;
  std::vector<int> seq;
  enum_terms(gmask, seq);
  // diagram count = number of distinct shapes among the terms
  std::set<std::vector<int>> shapes, shapes4g;
  for (auto& t : terms) {
    std::vector<int> key; int n4 = 0;
    for (int x : t) { key.push_back(nodes[x].shape); n4 += nodes[x].n4g; }
    shapes.insert(key);
    if (n4) shapes4g.insert(key);
  }
  n_diag = int(shapes.size());
  n_diag4g = int(shapes4g.size());
  // trie over attachment sequences read from the tbar end
  trie.push_back(TrieNode());
  for (size_t it = 0; it < terms.size(); ++it) {
    int cur = 0;
    for (int pos = int(terms[it].size()) - 1; pos >= 0; --pos) {
      const int g = terms[it][pos];
      int nxt = -1;
      for (int c : trie[cur].child) if (trie[c].gnode == g) nxt = c;
      if (nxt < 0) {
        TrieNode tn;
        tn.gnode = g; tn.mask_after = trie[cur].mask_after | nodes[g].mask;
        trie.push_back(tn);
        nxt = int(trie.size()) - 1;
        trie[cur].child.push_back(nxt);
      }
      cur = nxt;
    }
    trie[cur].terms.push_back(int(it));
  }
  // flows = permutations of the gluon legs in lexicographic order
  std::vector<int> perm = gl;
  std::map<Word, int> flow_of;
  do {
    flow_of[perm] = n_flow++;
    perms.insert(perms.end(), perm.begin(), perm.end());
  } while (std::next_permutation(perm.begin(), perm.end()));
  // term -> flow coefficients: concatenate the attachments' polynomials from the t end
  W.assign(terms.size(), std::vector<cd>(n_flow, cd(0)));
  for (size_t it = 0; it < terms.size(); ++it) {
    Poly p; p.t[Word{}] = 1;
    for (int x : terms[it]) p = pmul(p, nodes[x].colour);
    for (auto& w : p.t) W[it][flow_of.at(w.first)] += w.second;
  }
  // colour matrix from Gell-Mann traces:  CF_{sigma tau} = sum_a Tr(T^sigma (T^tau)^dagger)
  const SU3& S = su3();
  const int ng = int(gl.size());
  CF.assign(size_t(n_flow) * n_flow, 0.0);
  long long ncol = 1;
  for (int i = 0; i < ng; ++i) ncol *= 8;
  std::vector<C3> M(n_flow);
  std::vector<cd> acc(size_t(n_flow) * n_flow, cd(0));
  for (long long ic = 0; ic < ncol; ++ic) {
    int a[NMAX]; long long t = ic;
    for (int i = 0; i < ng; ++i) { a[i] = int(t % 8); t /= 8; }
    for (int f = 0; f < n_flow; ++f) {
      C3 m = c3ident();
      for (int i = 0; i < ng; ++i) {
        const int leg = perms[size_t(f) * ng + i];
        const int slot = int(std::find(gl.begin(), gl.end(), leg) - gl.begin());
        m = m * S.T[a[slot]];
      }
      M[f] = m;
    }
    for (int f = 0; f < n_flow; ++f) {
      const C3 md = M[f];
      for (int g = 0; g < n_flow; ++g) {
        cd tr = 0;  // Tr(M_f M_g^dagger) = sum_ij M_f[i][j] conj(M_g[i][j])
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) tr += md.m[i][j] * std::conj(M[g].m[i][j]);
        acc[size_t(f) * n_flow + g] += tr;
      }
    }
  }
  for (size_t i = 0; i < acc.size(); ++i) CF[i] = acc[i].real();
}

std::shared_ptr<Tier1> tier1_build(const Process& P) {
  auto t = std::make_shared<Tier1>();
  t->P = P;
  t->build();
  return t;
}
int tier1_n_diagrams(const Tier1& t) { return t.n_diag; }
int tier1_n_4g_diagrams(const Tier1& t) { return t.n_diag4g; }
int tier1_n_terms(const Tier1& t) { return int(t.terms.size()); }
int tier1_n_flows(const Tier1& t) { return t.n_flow; }
const double* tier1_cf(const Tier1& t) { return t.CF.data(); }
const int* tier1_flow_perms(const Tier1& t) { return t.perms.data(); }

// ---- evaluation ----------------------------------------------------------------------------
namespace {
struct Eval {
  const Tier1& T;
  const Ext& E;
  const int* hel = nullptr;
  std::vector<P4> K;       // K[mask] = sum of incoming-convention momenta of the legs in mask
  std::vector<V4> val;     // gluon node values for this helicity combination
  std::vector<char> have;
  std::vector<cd> A;       // amplitude of every term
  Eval(const Tier1& t, const Ext& e) : T(t), E(e) {
    const unsigned full = 1u << T.P.n_ext;
    K.assign(full, P4{{0, 0, 0, 0}});
    for (unsigned S = 1; S < full; ++S)
      for (int i = 0; i < T.P.n_ext; ++i)
        if (S >> i & 1u) K[S] = K[S] + E.k[i];
    val.resize(T.nodes.size());
    A.assign(T.terms.size(), cd(0));
  }
  void set_helicities(const int* h) { hel = h; have.assign(T.nodes.size(), 0); }
  const V4& gluon(int id) {
    if (have[id]) return val[id];
    const GNode& g = T.nodes[id];
    const double gs = T.P.gs;
    V4 r;
    if (g.kind == 0) {
      r = E.eps[g.leg][hel[g.leg]];
    } else if (g.kind == 1) {
      const V4 jx = gluon(g.ch[0]), jy = gluon(g.ch[1]);
      const P4 kx = K[T.nodes[g.ch[0]].mask], ky = K[T.nodes[g.ch[1]].mask];
      const P4 k3 = (-1.0) * (kx + ky);
      const P4 dxy = kx - ky, dy3 = ky - k3, d3x = k3 - kx;
      const cd xy = mdot(jx, jy), a = mdot(dy3, jx), b = mdot(d3x, jy);
      const cd pr = cd(0, -1) / mdot(K[g.mask], K[g.mask]);
      for (int m = 0; m < 4; ++m) r[m] = pr * gs * (xy * dxy[m] + a * jy[m] + b * jx[m]);
    } else {
      const V4 jx = gluon(g.ch[0]), jy = gluon(g.ch[1]), jz = gluon(g.ch[2]);
      const cd xy = mdot(jx, jy), xz = mdot(jx, jz), yz = mdot(jy, jz);
      const cd pr = cd(0, -1) / mdot(K[g.mask], K[g.mask]);
      const cd vt = cd(0, -1) * gs * gs;
      for (int m = 0; m < 4; ++m) {
        cd t;
        if (g.kind == 2) t = xz * jy[m] - yz * jx[m];
        else if (g.kind == 3) t = xy * jz[m] - yz * jx[m];
        else t = xy * jz[m] - xz * jy[m];
        r[m] = pr * vt * t;
      }
    }
    val[id] = r; have[id] = 1;
    return val[id];
  }
  // walk the trie from the tbar end; phi = propagated column spinor arriving at this vertex
  void walk(int tn, const Sp& phi) {
    const TrieNode& N = T.trie[tn];
    const double gs = T.P.gs, m = T.P.mass[T.leg_tb];
    const Sp psi = mul(cd(0, gs) * slash(gluon(N.gnode)), phi);  // (i g_s Jslash) phi
    if (!N.terms.empty()) {
      const cd amp = dot(E.sp[T.leg_t][hel[T.leg_t]], psi);  // close with u-bar
      for (int t : N.terms) A[t] = amp;
    }
    if (!N.child.empty()) {
      const P4 q = E.k[T.leg_tb] + K[N.mask_after];
      const M4 Sq = (cd(0, 1) / (mdot(q, q) - m * m)) * (slash(q) + cd(m) * mident());
      const Sp nxt = mul(Sq, psi);
      for (int c : N.child) walk(c, nxt);
    }
  }
  void flows(cd* J) {
    const Sp v = E.sp[T.leg_tb][hel[T.leg_tb]];
    for (int c : T.trie[0].child) walk(c, v);
    for (int f = 0; f < T.n_flow; ++f) J[f] = 0;
    for (size_t t = 0; t < T.terms.size(); ++t)
      for (int f = 0; f < T.n_flow; ++f)
        if (T.W[t][f] != cd(0)) J[f] += T.W[t][f] * A[t];
  }
};
}  // namespace

void tier1_flows(const me_handle_ref& h, const Ext& E, const int* hel, cd* J) {
  Eval ev(*h.t1, E);
  ev.set_helicities(hel);
  ev.flows(J);
}

double tier1_me2(const me_handle_ref& h, const double* mom) {
  const Tier1& T = *h.t1;
  Ext E;
  build_ext(h, mom, E);
  const int n = T.P.n_ext, nf = T.n_flow;
  std::vector<cd> J(nf);
  double total = 0;
  int hel[NMAX];
  Eval ev(T, E);
  for (int ih = 0; ih < (1 << n); ++ih) {
    for (int i = 0; i < n; ++i) hel[i] = ih >> i & 1;
    ev.set_helicities(hel);
    ev.flows(J.data());
    double s = 0;  // J^dagger CF J
    for (int f = 0; f < nf; ++f)
      for (int g = 0; g < nf; ++g) s += (std::conj(J[f]) * T.CF[size_t(f) * nf + g] * J[g]).real();
    total += s;
  }
  return total / T.P.avg;
}

}  // namespace orc
