// ORACLE — TEST INFRASTRUCTURE ONLY (see algebra.hpp header).
//
// me_tier1g.cpp — TIER 1 in the DIAGRAM basis, for any number of fermion lines (SURVEY.md §8(c) tier 1, D; §8(f) N1:
// the quark-initiated channels q qbar -> t tbar (g)(g), q g -> t tbar q (g) of PAPER.md:57-58, Table 1).
//
// me_tier1.cpp organises the diagrams of ONE quark line as attachment sequences and sums colour through the flow
// basis.  With two quark lines that picture does not hold, so this file does what a textbook does:
//   1. list every Feynman diagram as an explicit tree (root = leg 0; a four-gluon vertex gives three colour-pure
//      TERMS);
//   2. per term k: its kinematic value A_k (Feynman rules with the colour factors stripped, generic 4x4 Dirac algebra)
//      and its colour tensor C_k[colours of all external legs] (products of Gell-Mann T^a_{ij} and f^{abc}, contracted
//      along the tree exactly as the propagators delta^{ab}, delta_{ij} say);
//   3. sum over colours of |sum_k C_k A_k|^2 = sum_{kl} A_k conj(A_l) CM_kl with CM_kl = sum_colours C_k conj(C_l),
//      computed once per process by brute force;
//   4. sum over helicities, divide by S.
// No colour-flow basis, no 1/N_c bookkeeping, no recycling.  It also runs the one-line processes (gg -> t tbar + gluons),
// where tests compare it with me_tier1.cpp's flow basis.
//
// Kinematic rules (all momenta incoming, colour stripped; K_X = sum of the incoming momenta of the legs in X):
//   g g -> g*      (X, Y)    : B = g_s [ (JX.JY)(kX-kY) + JY ((kY-k3).JX) + JX ((k3-kX).JY) ], k3 = -(kX+kY);  colour f^{x y c}
//   g g g -> g*    (X, Y, Z) : B = -i g_s^2 { (JX.JZ) JY - (JY.JZ) JX   colour f^{xye} f^{zce}      term 0
//                                             (JX.JY) JZ - (JY.JZ) JX   colour f^{xze} f^{yce}      term 1
//                                             (JX.JY) JZ - (JX.JZ) JY   colour f^{xce} f^{yze}      term 2 }
//   row absorbs g  (R, G)    : B = R (i g_s Gslash);        colour sum_{i,a} R_i G_a T^a_{ij}
//   column absorbs g (G, C)  : B = (i g_s Gslash) C;        colour sum_{j,a} T^a_{ij} G_a C_j
//   row x column -> g* (R, C): B^mu = R (i g_s gamma^mu) C; colour sum_{ij} R_i T^a_{ij} C_j     (same line only)
//   propagators: J = (-i/K^2) B (gluon);  J = B S(-K) (row);  J = S(K) B (column);  S(q) = i (qslash + m)/(q^2 - m^2)
//   amplitude = root wavefunction . B over all other legs (no propagator on the last current).
#include <algorithm>
#include <set>
#include "me_ref.hpp"

namespace orc {

namespace {

enum { TY_NONE = -1, TY_G = 0 };                    // 1 + 2 f: row of line f, 2 + 2 f: column of line f
enum { OP_LEAF = 0, OP_GGG = 1, OP_GGGG0 = 2, OP_GGGG1 = 3, OP_GGGG2 = 4, OP_ROW_G = 5, OP_G_COL = 6, OP_ROW_COL = 7 };

// colour tensor: v[(sum_k col_k stride_k) * open + o], legs ascending, strides in that order; open = dimension of the
// off-shell line's index (8 or 3)
struct CTen {
  std::vector<int> legs, dims;
  int open = 1;
  std::vector<cd> v;
  size_t size() const { size_t n = 1; for (int d : dims) n *= size_t(d); return n; }
};

struct W4 { cd c[4]; };
inline V4 asV(const W4& w) { return {{w.c[0], w.c[1], w.c[2], w.c[3]}}; }
inline Sp asS(const W4& w) { return {{w.c[0], w.c[1], w.c[2], w.c[3]}}; }
inline W4 fromV(const V4& v) { return {{v[0], v[1], v[2], v[3]}}; }
inline W4 fromS(const Sp& s) { return {{s[0], s[1], s[2], s[3]}}; }

struct Node {
  unsigned mask = 0;
  int type = TY_G, op = OP_LEAF, leg = -1;
  int ch[3] = {-1, -1, -1};
  int shape = -1, n4g = 0;
  CTen col;
};

}  // namespace

struct Tier1G {
  Process P;
  std::vector<Node> nodes;
  std::map<unsigned, std::vector<int>> trees;
  std::map<std::vector<int>, int> shape_ids;
  std::vector<int> terms;   // top nodes: trees over all legs but the root whose type closes on the root
  int n_diag = 0, n_diag4g = 0;
  std::vector<cd> CM;       // [n_terms][n_terms]
  std::vector<int> top_legs, top_dims;   // colour index order of the terms' tensors: legs 1.. ascending, then the root
  std::vector<std::vector<cd>> Cfull;    // [term][colour assignment]

  int type_of(unsigned S) const {
    int t = TY_G;
    for (int f = 0; f < P.n_lines(); ++f) {
      int ends = 0, which = 0;
      for (int i = 0; i < P.n_ext; ++i)
        if ((S >> i & 1u) && P.line[i] == f) { ++ends; which = is_row_kind(P.kind[i]) ? 1 + 2 * f : 2 + 2 * f; }
      if (ends == 1) { if (t != TY_G) return TY_NONE; t = which; }
    }
    return t;
  }
  int shape_of(const std::vector<int>& key) {
    auto it = shape_ids.find(key);
    if (it != shape_ids.end()) return it->second;
    const int id = int(shape_ids.size());
    shape_ids[key] = id;
    return id;
  }
  int colour_dim(int leg) const { return is_gluon_kind(P.kind[leg]) ? 8 : 3; }
  int add(Node g) { nodes.push_back(std::move(g)); return int(nodes.size()) - 1; }
  const std::vector<int>& trees_of(unsigned S);
  CTen join(const std::vector<const CTen*>& ch, int open, const std::vector<cd>& vertex) const;
  void build();
};

// out[legs of all children][o] = sum over the children's open indices of vertex[a0][a1](..)[o] prod_k child_k[..][a_k]
// `vertex` is indexed [a0 * d1 (* d2) + a1 ...][o] with d_k = child k's open dimension.
CTen Tier1G::join(const std::vector<const CTen*>& ch, int open, const std::vector<cd>& vertex) const {
  CTen r;
  r.open = open;
  for (const CTen* c : ch) r.legs.insert(r.legs.end(), c->legs.begin(), c->legs.end());
  std::sort(r.legs.begin(), r.legs.end());
  std::vector<size_t> stride_of(P.n_ext, 0);
  size_t st = 1;
  for (int l : r.legs) { r.dims.push_back(colour_dim(l)); stride_of[l] = st; st *= size_t(colour_dim(l)); }
  r.v.assign(st * size_t(open), cd(0));
  // position of every child entry inside the output index
  std::vector<std::vector<size_t>> pos(ch.size());
  for (size_t k = 0; k < ch.size(); ++k) {
    const CTen& c = *ch[k];
    pos[k].resize(c.size());
    for (size_t i = 0; i < c.size(); ++i) {
      size_t t = i, p = 0;
      for (size_t q = 0; q < c.legs.size(); ++q) { p += (t % size_t(c.dims[q])) * stride_of[c.legs[q]]; t /= size_t(c.dims[q]); }
      pos[k][i] = p;
    }
  }
  const size_t nk = ch.size();
  std::vector<size_t> idx(nk, 0);
  while (true) {
    size_t p = 0;
    for (size_t k = 0; k < nk; ++k) p += pos[k][idx[k]];
    // contract the open indices with the vertex
    const int d0 = ch[0]->open, d1 = ch[1]->open, d2 = nk > 2 ? ch[2]->open : 1;
    for (int a = 0; a < d0; ++a) {
      const cd xa = ch[0]->v[idx[0] * size_t(d0) + a];
      if (xa == cd(0)) continue;
      for (int b = 0; b < d1; ++b) {
        const cd xb = xa * ch[1]->v[idx[1] * size_t(d1) + b];
        if (xb == cd(0)) continue;
        for (int c = 0; c < d2; ++c) {
          const cd xc = nk > 2 ? xb * ch[2]->v[idx[2] * size_t(d2) + c] : xb;
          if (xc == cd(0)) continue;
          const size_t vrow = ((size_t(a) * size_t(d1) + size_t(b)) * size_t(d2) + size_t(c)) * size_t(open);
          for (int o = 0; o < open; ++o) r.v[p * size_t(open) + o] += xc * vertex[vrow + o];
        }
      }
    }
    size_t k = 0;
    while (k < nk && ++idx[k] == ch[k]->size()) idx[k++] = 0;
    if (k == nk) break;
  }
  return r;
}

const std::vector<int>& Tier1G::trees_of(unsigned S) {
  auto it = trees.find(S);
  if (it != trees.end()) return it->second;
  std::vector<int> out;
  const int tS = type_of(S);
  const SU3& G = su3();
  if (tS == TY_NONE) {
    // no current
  } else if (__builtin_popcount(S) == 1) {
    Node g;
    g.mask = S; g.type = tS; g.op = OP_LEAF; g.leg = __builtin_ctz(S);
    g.shape = shape_of({OP_LEAF, g.leg});
    const int d = colour_dim(g.leg);
    g.col.legs = {g.leg}; g.col.dims = {d}; g.col.open = d;
    g.col.v.assign(size_t(d) * d, cd(0));
    for (int a = 0; a < d; ++a) g.col.v[size_t(a) * d + a] = 1;   // delta(colour of the leg, open index)
    out.push_back(add(g));
  } else {
    // vertex colour tensors
    std::vector<cd> vf(8 * 8 * 8), vrg(3 * 8 * 3), vgc(8 * 3 * 3), vrc(3 * 3 * 8);
    for (int a = 0; a < 8; ++a) for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) vf[(a * 8 + b) * 8 + c] = G.f[a][b][c];
    for (int i = 0; i < 3; ++i) for (int a = 0; a < 8; ++a) for (int j = 0; j < 3; ++j) {
      vrg[(i * 8 + a) * 3 + j] = G.T[a].m[i][j];   // row_i g_a -> row_j : T^a_{ij}
      vgc[(a * 3 + j) * 3 + i] = G.T[a].m[i][j];   // g_a col_j -> col_i : T^a_{ij}
      vrc[(i * 3 + j) * 8 + a] = G.T[a].m[i][j];   // row_i col_j -> g_a : T^a_{ij}
    }
    const unsigned low = S & (~S + 1u);
    for (unsigned A = (S - 1) & S; A; A = (A - 1) & S) {
      if (!(A & low)) continue;
      const unsigned B = S & ~A;
      const int tA = type_of(A), tB = type_of(B);
      if (tA == TY_NONE || tB == TY_NONE) continue;
      const std::vector<int> ta = trees_of(A), tb = trees_of(B);
      for (int x : ta)
        for (int y : tb) {
          Node g;
          g.mask = S; g.type = tS;
          g.n4g = nodes[x].n4g + nodes[y].n4g;
          bool ok = true;
          const bool rowA = tA > 0 && (tA & 1), colA = tA > 0 && !(tA & 1), rowB = tB > 0 && (tB & 1), colB = tB > 0 && !(tB & 1);
          if (tS == TY_G && tA == TY_G && tB == TY_G) {
            g.op = OP_GGG; g.ch[0] = x; g.ch[1] = y;
            g.col = join({&nodes[x].col, &nodes[y].col}, 8, vf);
          } else if (tS == TY_G && rowA && colB && tA + 1 == tB) {
            g.op = OP_ROW_COL; g.ch[0] = x; g.ch[1] = y;
            g.col = join({&nodes[x].col, &nodes[y].col}, 8, vrc);
          } else if (tS == TY_G && colA && rowB && tB + 1 == tA) {
            g.op = OP_ROW_COL; g.ch[0] = y; g.ch[1] = x;
            g.col = join({&nodes[y].col, &nodes[x].col}, 8, vrc);
          } else if (tS > 0 && (tS & 1) && ((tA == tS && tB == TY_G) || (tB == tS && tA == TY_G))) {
            g.op = OP_ROW_G; g.ch[0] = (tA == tS) ? x : y; g.ch[1] = (tA == tS) ? y : x;
            g.col = join({&nodes[g.ch[0]].col, &nodes[g.ch[1]].col}, 3, vrg);
          } else if (tS > 0 && !(tS & 1) && ((tA == tS && tB == TY_G) || (tB == tS && tA == TY_G))) {
            g.op = OP_G_COL; g.ch[0] = (tA == TY_G) ? x : y; g.ch[1] = (tA == TY_G) ? y : x;
            g.col = join({&nodes[g.ch[0]].col, &nodes[g.ch[1]].col}, 3, vgc);
          } else {
            ok = false;
          }
          if (!ok) continue;
          g.shape = shape_of({g.op, nodes[g.ch[0]].shape, nodes[g.ch[1]].shape});
          if (g.op == OP_GGG) {   // unordered children
            const int s0 = nodes[x].shape, s1 = nodes[y].shape;
            g.shape = shape_of({OP_GGG, std::min(s0, s1), std::max(s0, s1)});
          }
          out.push_back(add(g));
        }
    }
    if (tS == TY_G) {
      // four-gluon vertex: colour of term k over (x, y, z, open c)
      std::vector<cd> vff[3];
      for (int k = 0; k < 3; ++k) vff[k].assign(8 * 8 * 8 * 8, cd(0));
      for (int a = 0; a < 8; ++a) for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) for (int d = 0; d < 8; ++d) {
        double c0 = 0, c1 = 0, c2 = 0;
        for (int e = 0; e < 8; ++e) {
          c0 += G.f[a][b][e] * G.f[c][d][e];
          c1 += G.f[a][c][e] * G.f[b][d][e];
          c2 += G.f[a][d][e] * G.f[b][c][e];
        }
        const size_t i = ((size_t(a) * 8 + b) * 8 + c) * 8 + d;
        vff[0][i] = c0; vff[1][i] = c1; vff[2][i] = c2;
      }
      for (unsigned A = (S - 1) & S; A; A = (A - 1) & S) {
        if (!(A & low) || type_of(A) != TY_G) continue;
        const unsigned R = S & ~A;
        const unsigned lowR = R & (~R + 1u);
        for (unsigned B = (R - 1) & R; B; B = (B - 1) & R) {
          if (!(B & lowR)) continue;
          const unsigned C = R & ~B;
          if (!C || type_of(B) != TY_G || type_of(C) != TY_G) continue;
          const std::vector<int> ta = trees_of(A), tb = trees_of(B), tc = trees_of(C);
          for (int x : ta) for (int y : tb) for (int z : tc)
            for (int k = 0; k < 3; ++k) {
              Node g;
              g.mask = S; g.type = TY_G; g.op = OP_GGGG0 + k;
              g.ch[0] = x; g.ch[1] = y; g.ch[2] = z;
              g.n4g = 1 + nodes[x].n4g + nodes[y].n4g + nodes[z].n4g;
              std::vector<int> sk = {nodes[x].shape, nodes[y].shape, nodes[z].shape};
              std::sort(sk.begin(), sk.end());
              g.shape = shape_of({OP_GGGG0, sk[0], sk[1], sk[2]});
              g.col = join({&nodes[x].col, &nodes[y].col, &nodes[z].col}, 8, vff[k]);
              out.push_back(add(g));
            }
        }
      }
    }
  }
  trees[S] = out;
  return trees[S];
}

void Tier1G::build() {
  const unsigned full = (1u << P.n_ext) - 1u, rest = full & ~1u;
  // the tree over all other legs closes on the root: gluon on gluon, a line's row on its psi end, column on psi-bar end
  int want;
  if (is_gluon_kind(P.kind[0])) want = TY_G;
  else if (is_col_kind(P.kind[0])) want = 1 + 2 * P.line[0];
  else want = 2 + 2 * P.line[0];
  const std::vector<int> top = trees_of(rest);
  std::set<int> shapes, shapes4g;
  for (int t : top) {
    if (nodes[t].type != want) continue;
    terms.push_back(t);
    shapes.insert(nodes[t].shape);
    if (nodes[t].n4g) shapes4g.insert(nodes[t].shape);
  }
  n_diag = int(shapes.size());
  n_diag4g = int(shapes4g.size());
  // colour tensors of the terms over (legs 1.., root): the open index of the top current IS the root's colour
  const size_t nt = terms.size();
  Cfull.resize(nt);
  for (size_t k = 0; k < nt; ++k) Cfull[k] = nodes[terms[k]].col.v;
  if (nt) { top_legs = nodes[terms[0]].col.legs; top_dims = nodes[terms[0]].col.dims; }
  top_legs.push_back(0); top_dims.push_back(colour_dim(0));
  CM.assign(nt * nt, cd(0));
  for (size_t k = 0; k < nt; ++k)
    for (size_t l = 0; l <= k; ++l) {
      cd s = 0;
      const std::vector<cd>&a = Cfull[k], &b = Cfull[l];
      for (size_t i = 0; i < a.size(); ++i) s += a[i] * std::conj(b[i]);
      CM[k * nt + l] = s;
      CM[l * nt + k] = std::conj(s);
    }
}

namespace {
struct EvalG {
  const Tier1G& T;
  const Ext& E;
  const int* hel = nullptr;
  std::vector<P4> K;
  std::vector<W4> val;     // PROPAGATED value of every node for this helicity combination
  std::vector<char> have;
  EvalG(const Tier1G& t, const Ext& e) : T(t), E(e) {
    const unsigned full = 1u << T.P.n_ext;
    K.assign(full, P4{{0, 0, 0, 0}});
    for (unsigned S = 1; S < full; ++S)
      for (int i = 0; i < T.P.n_ext; ++i)
        if (S >> i & 1u) K[S] = K[S] + E.k[i];
    val.resize(T.nodes.size());
  }
  void set_helicities(const int* h) { hel = h; have.assign(T.nodes.size(), 0); }
  double line_mass(int type) const {
    const int f = (type - 1) / 2;
    for (int i = 0; i < T.P.n_ext; ++i) if (T.P.line[i] == f) return T.P.mass[i];
    return 0;
  }
  // the vertex of node g applied to its children's propagated currents: no propagator
  W4 bare(const Node& g) {
    const double gs = T.P.gs;
    if (g.op == OP_LEAF) {
      return is_gluon_kind(T.P.kind[g.leg]) ? fromV(E.eps[g.leg][hel[g.leg]]) : fromS(E.sp[g.leg][hel[g.leg]]);
    } else if (g.op == OP_GGG) {
      const V4 jx = asV(cur(g.ch[0])), jy = asV(cur(g.ch[1]));
      const P4 kx = K[T.nodes[g.ch[0]].mask], ky = K[T.nodes[g.ch[1]].mask];
      const P4 k3 = (-1.0) * (kx + ky);
      const P4 dxy = kx - ky, dy3 = ky - k3, d3x = k3 - kx;
      const cd xy = mdot(jx, jy), a = mdot(dy3, jx), b = mdot(d3x, jy);
      V4 r;
      for (int m = 0; m < 4; ++m) r[m] = gs * (xy * dxy[m] + a * jy[m] + b * jx[m]);
      return fromV(r);
    } else if (g.op >= OP_GGGG0 && g.op <= OP_GGGG2) {
      const V4 jx = asV(cur(g.ch[0])), jy = asV(cur(g.ch[1])), jz = asV(cur(g.ch[2]));
      const cd xy = mdot(jx, jy), xz = mdot(jx, jz), yz = mdot(jy, jz);
      const cd vt = cd(0, -1) * gs * gs;
      V4 r;
      for (int m = 0; m < 4; ++m) {
        cd t;
        if (g.op == OP_GGGG0) t = xz * jy[m] - yz * jx[m];
        else if (g.op == OP_GGGG1) t = xy * jz[m] - yz * jx[m];
        else t = xy * jz[m] - xz * jy[m];
        r[m] = vt * t;
      }
      return fromV(r);
    } else if (g.op == OP_ROW_G) {
      return fromS(mul(asS(cur(g.ch[0])), cd(0, gs) * slash(asV(cur(g.ch[1])))));
    } else if (g.op == OP_G_COL) {
      return fromS(mul(cd(0, gs) * slash(asV(cur(g.ch[0]))), asS(cur(g.ch[1]))));
    } else {
      const Sp r = asS(cur(g.ch[0])), c = asS(cur(g.ch[1]));
      V4 v;
      for (int mu = 0; mu < 4; ++mu) v[mu] = cd(0, gs) * dot(r, mul(gammas().g[mu], c));
      return fromV(v);
    }
  }
  // propagated current of node id
  const W4& cur(int id) {
    if (have[id]) return val[id];
    const Node& g = T.nodes[id];
    W4 b = bare(g);
    if (g.op != OP_LEAF) {
      const P4& k = K[g.mask];
      if (g.type == TY_G) {
        const cd pr = cd(0, -1) / mdot(k, k);
        for (int m = 0; m < 4; ++m) b.c[m] = pr * b.c[m];
      } else if (g.type & 1) {
        const double mq = line_mass(g.type);
        const P4 q = (-1.0) * k;
        const M4 Sq = (cd(0, 1) / (mdot(q, q) - mq * mq)) * (slash(q) + cd(mq) * mident());
        b = fromS(mul(asS(b), Sq));
      } else {
        const double mq = line_mass(g.type);
        const M4 Sq = (cd(0, 1) / (mdot(k, k) - mq * mq)) * (slash(k) + cd(mq) * mident());
        b = fromS(mul(Sq, asS(b)));
      }
    }
    val[id] = b; have[id] = 1;
    return val[id];
  }
  void amplitudes(cd* A) {
    const Process& P = T.P;
    for (size_t k = 0; k < T.terms.size(); ++k) {
      const W4 b = bare(T.nodes[T.terms[k]]);
      if (is_gluon_kind(P.kind[0])) A[k] = mdot(E.eps[0][hel[0]], asV(b));
      else if (is_col_kind(P.kind[0])) A[k] = dot(asS(b), E.sp[0][hel[0]]);
      else A[k] = dot(E.sp[0][hel[0]], asS(b));
    }
  }
};
}  // namespace

std::shared_ptr<Tier1G> tier1g_build(const Process& P) {
  auto t = std::make_shared<Tier1G>();
  t->P = P;
  t->build();
  return t;
}
int tier1g_n_diagrams(const Tier1G& t) { return t.n_diag; }
int tier1g_n_4g_diagrams(const Tier1G& t) { return t.n_diag4g; }
int tier1g_n_terms(const Tier1G& t) { return int(t.terms.size()); }
// rank-revealing data for the tests: the colour matrix between the terms
const cd* tier1g_colour_matrix(const Tier1G& t) { return t.CM.data(); }

double tier1g_me2(const me_handle_ref& h, const Tier1G& T, const double* mom) {
  Ext E;
  build_ext(h, mom, E);
  const int n = T.P.n_ext;
  const size_t nt = T.terms.size();
  std::vector<cd> A(nt);
  double total = 0;
  int hel[NMAX];
  EvalG ev(T, E);
  for (int ih = 0; ih < (1 << n); ++ih) {
    for (int i = 0; i < n; ++i) hel[i] = ih >> i & 1;
    ev.set_helicities(hel);
    ev.amplitudes(A.data());
    double s = 0;  // sum_{kl} A_k CM_kl conj(A_l)
    for (size_t k = 0; k < nt; ++k)
      for (size_t l = 0; l < nt; ++l) s += (A[k] * T.CM[k * nt + l] * std::conj(A[l])).real();
    total += s;
  }
  return total / T.P.avg;
}

// sum_k C_k[col] A_k for one helicity and colour assignment: comparable with tier0_amplitude
cd tier1g_amplitude(const me_handle_ref& h, const Tier1G& T, const Ext& E, const int* hel, const int* col) {
  EvalG ev(T, E);
  ev.set_helicities(hel);
  std::vector<cd> A(T.terms.size());
  ev.amplitudes(A.data());
  size_t idx = 0, st = 1;
  for (size_t q = 0; q + 1 < T.top_legs.size(); ++q) { idx += size_t(col[T.top_legs[q]]) * st; st *= size_t(T.top_dims[q]); }
  const int open = T.top_dims.back();
  cd s = 0;
  for (size_t k = 0; k < T.terms.size(); ++k) s += T.Cfull[k][idx * size_t(open) + size_t(col[0])] * A[k];
  return s;
}

}  // namespace orc
