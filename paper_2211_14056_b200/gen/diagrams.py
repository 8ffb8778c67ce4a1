"""Build-time diagram generator: process -> list of off-shell currents + closing amplitudes + colour flows.

This replaces the MG5_aMC + jinja transpiler layers of the paper (Fig. 2): there is no
MadGraph here, so the Feynman diagrams of a process are enumerated directly and the
colour-flow coefficient table is derived numerically from explicit SU(3) tensors.
It shares no source with oracle/ (which enumerates at run time in C++ with its own data structures).

Model: one fermion line per flavour; vertices {f fbar V, ggg, gggg}; "V" is the gluon for the quark lines (t, and the
massless q of the quark-initiated channels) and the photon for the lepton lines.

A *diagram* is a tree whose leaves are the external legs.  Every diagram is evaluated "closed" at its
centroid vertex: the vertex whose hanging subtrees all have <= n/2 leaves (ties — a propagator
splitting the legs n/2 | n/2 — go to the side that holds leg 0).  The hanging subtrees are the off-shell
currents; structurally identical subtrees are shared between diagrams.  A subtree / diagram containing a
four-gluon vertex splits into three colour-pure terms.

Propagator-cut closings.  A diagram is not evaluated at its centroid vertex: one hanging subtree C of that vertex
that does not hold leg 0 stays a propagated current, the other subtrees of the vertex are merged into the
UN-propagated ("open") current U over the complementary legs (it holds leg 0), and the diagram is the plain
contraction U . C (a 4-component dot product instead of a vertex).  `factorise()` then sums, per colour flow,
the U's and the C's of one leg split into colour-ordered combinations first (every current depends only on the
helicities of its own n/2 legs), so that a flow receives ONE dot product per split — the colour-ordered
recursion is recovered from the Feynman diagrams, not assumed.

Parity.  QCD and QED conserve parity: |M(-h)|^2 = |M(h)|^2 for the colour-summed squared amplitude, so only the
helicity combinations with leg 0 at +1 are evaluated and the sum is doubled (a DECLARED 2x
saving; the flops reported are the ones executed).  Objects holding leg 0 therefore have half the variants.

Powers of i and of the coupling carried by vertices and propagators are NOT applied numerically: every
object carries a symbolic phase in {1, i, -1, -i}, which ends up in the flow coefficient of the term.
Feynman rules, all momenta incoming:
    f fbar V   : i g gamma^mu T^a            ggg : g f^{abc} [...]        gggg : -i g^2 [...]
    fermion propagator  i (qslash + m)/(q^2 - m^2)       vector propagator  -i g^{mu nu}/q^2
"""
import itertools
from collections import namedtuple
from fractions import Fraction

import numpy as np

# ---- legs ---------------------------------------------------------------------------------------------------
# kind ids match csrc/helas.cuh::LegKind
LEG_V_IN, LEG_V_OUT, LEG_F_OUT, LEG_FB_OUT, LEG_F_IN, LEG_FB_IN = range(6)
Leg = namedtuple("Leg", "kind flavour massive")  # flavour: 'g' | 'a' for vectors, 't' | 'e' | 'mu' for fermions

PROCESSES = {
    # name: (legs, coupling-constant name, averaging denominator S of SURVEY §8(c) F)
    "epem_mupmum": ([Leg(LEG_F_IN, "e", False), Leg(LEG_FB_IN, "e", False),
                     Leg(LEG_F_OUT, "mu", False), Leg(LEG_FB_OUT, "mu", False)], "ee", 4),
    "gg_ttx": ([Leg(LEG_V_IN, "g", False), Leg(LEG_V_IN, "g", False),
                Leg(LEG_F_OUT, "t", True), Leg(LEG_FB_OUT, "t", True)], "gs", 4 * 64),
    "gg_ttxg": ([Leg(LEG_V_IN, "g", False), Leg(LEG_V_IN, "g", False), Leg(LEG_F_OUT, "t", True),
                 Leg(LEG_FB_OUT, "t", True), Leg(LEG_V_OUT, "g", False)], "gs", 4 * 64),
    "gg_ttxgg": ([Leg(LEG_V_IN, "g", False), Leg(LEG_V_IN, "g", False), Leg(LEG_F_OUT, "t", True),
                  Leg(LEG_FB_OUT, "t", True), Leg(LEG_V_OUT, "g", False), Leg(LEG_V_OUT, "g", False)],
                 "gs", 4 * 64 * 2),
}
# The quark-initiated channels of the paper's hadronic processes (Table 1: 36 = 16 + 4 x 5 and
# 267 = 123 + 4 x 36 diagrams): a second quark line q (massless, a flavour different from t).
# Averages: 1/4 spins x 1/9 (q qbar) or 1/24 (q g) colours x 1/n! for n identical final gluons.
_G_OUT = Leg(LEG_V_OUT, "g", False)
_QQX = [Leg(LEG_F_IN, "q", False), Leg(LEG_FB_IN, "q", False), Leg(LEG_F_OUT, "t", True), Leg(LEG_FB_OUT, "t", True)]
_QG = [Leg(LEG_F_IN, "q", False), Leg(LEG_V_IN, "g", False), Leg(LEG_F_OUT, "t", True), Leg(LEG_FB_OUT, "t", True),
       Leg(LEG_F_OUT, "q", False)]
PROCESSES["qqx_ttx"] = (_QQX, "gs", 4 * 9)
PROCESSES["qqx_ttxg"] = (_QQX + [_G_OUT], "gs", 4 * 9)
PROCESSES["qg_ttxq"] = (_QG, "gs", 4 * 24)
PROCESSES["qqx_ttxgg"] = (_QQX + [_G_OUT, _G_OUT], "gs", 4 * 9 * 2)
PROCESSES["qg_ttxqg"] = (_QG + [_G_OUT], "gs", 4 * 24)
# the charge conjugates qbar g -> t tbar qbar (g): an incoming and an outgoing ANTIquark of the light flavour
_QXG = [Leg(LEG_FB_IN, "q", False), Leg(LEG_V_IN, "g", False), Leg(LEG_F_OUT, "t", True), Leg(LEG_FB_OUT, "t", True),
        Leg(LEG_FB_OUT, "q", False)]
PROCESSES["qxg_ttxqx"] = (_QXG, "gs", 4 * 24)
PROCESSES["qxg_ttxqxg"] = (_QXG + [_G_OUT], "gs", 4 * 24)
# Processes whose diagrams are ENUMERATED only (Program(name, count_only=True)): none at present.
COUNT_ONLY = {}
# g g -> t tbar g g g (1 240 diagrams, 120 colour flows; the gap to the
# tensorised generator widens with the number of diagrams).  1/4 spins x 1/64 colours x 1/3! identical gluons.
PROCESSES["gg_ttxggg"] = (PROCESSES["gg_ttxgg"][0] + [_G_OUT], "gs", 4 * 64 * 6)
VECTOR_OF = {"t": "g", "q": "g", "e": "a", "mu": "a"}
CUT_ALL = True   # every diagram is the contraction of an open current U with a propagated current C (see _pick_cut)

# ---- SU(3) ---------------------------------------------------------------------------------------------------


def su3():
    """Gell-Mann T^a = lambda^a/2 and f^{abc} from [T^a, T^b] = i f^{abc} T^c."""
    l = np.zeros((8, 3, 3), dtype=complex)
    l[0][0, 1] = l[0][1, 0] = 1
    l[1][0, 1] = -1j
    l[1][1, 0] = 1j
    l[2][0, 0] = 1
    l[2][1, 1] = -1
    l[3][0, 2] = l[3][2, 0] = 1
    l[4][0, 2] = -1j
    l[4][2, 0] = 1j
    l[5][1, 2] = l[5][2, 1] = 1
    l[6][1, 2] = -1j
    l[6][2, 1] = 1j
    l[7] = np.diag([1, 1, -2]) / np.sqrt(3)
    T = l / 2
    f = np.zeros((8, 8, 8))
    for a in range(8):
        for b in range(8):
            comm = T[a] @ T[b] - T[b] @ T[a]
            for c in range(8):
                f[a, b, c] = (-2j * np.trace(comm @ T[c])).real  # Tr(T^c T^d) = delta/2
    return T, f


_T, _F = su3()

# ---- objects ---------------------------------------------------------------------------------------------------
# type: ('V', vflavour) | ('O', flavour) row spinor | ('I', flavour) column spinor
# op  : 'EXT' | 'FFV_ROW' (O,V->O) | 'FFV_COL' (I,V->I) | 'FFV_VEC' (O,I->V) | 'VVV' (V,V->V) | 'VVVV1/2/3' (V,V,V->V)


class Obj:
    __slots__ = ("id", "legs", "type", "op", "args", "phase", "_col", "skel", "has4g", "prop")

    def __init__(self, id, legs, type, op, args, phase, prop=True):
        self.id, self.legs, self.type, self.op, self.args, self.phase = id, tuple(sorted(legs)), type, op, args, phase
        self.prop = prop    # False: the current stops at its vertex (no propagator): the U side of a propagator cut
        self._col = None
        self.skel = None    # structural key: the three colour terms of one 4g subtree share it
        self.has4g = False


class Term:
    """One colour-pure closing amplitude."""
    __slots__ = ("op", "args", "phase", "which", "diagram", "flows")

    def __init__(self, op, args, phase, which, diagram):
        self.op, self.args, self.phase, self.which, self.diagram, self.flows = op, args, phase, which, diagram, None


def _set_partitions(items, k):
    """All unordered partitions of `items` (list) into exactly k non-empty blocks."""
    items = list(items)
    if k == 1:
        yield [items]
        return
    if len(items) < k:
        return
    first, rest = items[0], items[1:]
    # first alone + partition of the rest into k-1
    for p in _set_partitions(rest, k - 1):
        yield [[first]] + p
    # first joins one block of a partition of rest into k
    for p in _set_partitions(rest, k):
        for i in range(len(p)):
            yield p[:i] + [[first] + p[i]] + p[i + 1:]


class Program:
    """The evaluated-closed-at-centroid diagram list of one process."""

    def __init__(self, name, count_only=False, frozen=(0,)):
        """count_only: enumerate the diagrams only (no colour flows, no factorisation).  frozen: legs whose helicity is
        fixed while the others are summed (leg 0: parity; emit.py freezes more legs for processes evaluated in passes)."""
        self.name = name
        self.frozen = tuple(frozen)
        self.legs, self.coupling, self.avg = (COUNT_ONLY[name], "gs", 1) if name in COUNT_ONLY else PROCESSES[name]
        self.n = len(self.legs)
        self.objs = []
        self._memo = {}
        self.terms = []
        self.n_diagrams = 0
        self.n_diagrams_4g = 0
        self._ext = {}
        self._diagrams = {}
        self._unprop = {}
        self.combos = []     # colour-ordered sums of half-split currents (factorise)
        self.dots = []       # (flow, combo/object id of U side, of C side, phase z, 'V'|'F')
        for i, leg in enumerate(self.legs):
            if leg.kind in (LEG_V_IN, LEG_V_OUT):
                t = ("V", leg.flavour)
            elif leg.kind in (LEG_F_OUT, LEG_FB_IN):
                t = ("O", leg.flavour)
            else:
                t = ("I", leg.flavour)
            self._ext[i] = self._new((i,), t, "EXT", (), 1)
        self._close()
        if count_only:
            return
        self._colour()
        self.factorise()

    # -- enumeration ------------------------------------------------------------------------------------------
    def _new(self, legs, type, op, args, phase, prop=True):
        o = Obj(len(self.objs), legs, type, op, args, phase, prop)
        o.skel = (op[:4] if op.startswith("VVVV") else op, tuple(sorted(legs)), tuple(self.objs[a].skel for a in args))
        o.has4g = op.startswith("VVVV") or any(self.objs[a].has4g for a in args)
        self.objs.append(o)
        return o

    def subtrees(self, legs):
        """All distinct subtrees (as off-shell currents, propagator included) with leaf set `legs`."""
        key = tuple(sorted(legs))
        if key in self._memo:
            return self._memo[key]
        if len(key) == 1:
            res = [self._ext[key[0]]]
            self._memo[key] = res
            return res
        res = []
        for parts in _set_partitions(key, 2):
            for A in self.subtrees(parts[0]):
                for B in self.subtrees(parts[1]):
                    res.extend(self._join2(key, A, B))
        for parts in _set_partitions(key, 3):
            for A in self.subtrees(parts[0]):
                for B in self.subtrees(parts[1]):
                    for C in self.subtrees(parts[2]):
                        if A.type == B.type == C.type == ("V", "g"):
                            # vertex -i g^2, propagator -i  -> phase -1
                            ph = A.phase * B.phase * C.phase * (-1)
                            for w in (1, 2, 3):
                                res.append(self._new(key, ("V", "g"), "VVVV%d" % w, (A.id, B.id, C.id), ph))
        self._memo[key] = res
        return res

    def _join2(self, key, A, B):
        out = []
        for X, Y in ((A, B), (B, A)):
            kx, fx = X.type
            ky, fy = Y.type
            if kx == "O" and ky == "V" and VECTOR_OF[fx] == fy:
                # vertex i g, propagator i -> -1
                out.append(self._new(key, X.type, "FFV_ROW", (X.id, Y.id), X.phase * Y.phase * (-1)))
            if kx == "I" and ky == "V" and VECTOR_OF[fx] == fy:
                out.append(self._new(key, X.type, "FFV_COL", (X.id, Y.id), X.phase * Y.phase * (-1)))
            if kx == "O" and ky == "I" and fx == fy:
                # vertex i g, propagator -i -> +1
                out.append(self._new(key, ("V", VECTOR_OF[fx]), "FFV_VEC", (X.id, Y.id), X.phase * Y.phase))
        if A.type == B.type == ("V", "g"):
            # vertex g (real), propagator -i
            out.append(self._new(key, ("V", "g"), "VVV", (A.id, B.id), A.phase * B.phase * (-1j)))
        return out

    def _close(self):
        n = self.n
        allowed = lambda part: 2 * len(part) < n or (2 * len(part) == n and 0 not in part)
        all_legs = list(range(n))
        for parts in _set_partitions(all_legs, 3):
            if not all(allowed(p) for p in parts):
                continue
            for A in self.subtrees(parts[0]):
                for B in self.subtrees(parts[1]):
                    for C in self.subtrees(parts[2]):
                        self._close3(A, B, C)
        for parts in _set_partitions(all_legs, 4):
            if not all(allowed(p) for p in parts):
                continue
            for combo in itertools.product(*[self.subtrees(p) for p in parts]):
                if all(o.type == ("V", "g") for o in combo):
                    cut = self._pick_cut(combo)
                    if cut is not None:
                        self._close_cut(cut, [o for o in combo if o is not cut], True)
                        continue
                    d = self._count_diagram(combo, True)
                    ph = np.prod([o.phase for o in combo]) * (-1j)  # vertex -i g^2
                    for w in (1, 2, 3):
                        self.terms.append(Term("VVVV_AMP", tuple(o.id for o in combo), ph, w, d))

    def _count_diagram(self, combo, closing_4g):
        key = (closing_4g, tuple(sorted(o.skel for o in combo)))
        if key not in self._diagrams:
            self._diagrams[key] = len(self._diagrams)
            self.n_diagrams += 1
            if closing_4g or any(o.has4g for o in combo):
                self.n_diagrams_4g += 1
        return self._diagrams[key]

    # the un-propagated current over the legs of X u Y (u Z): the vertex without the propagator behind it
    def _unprop_current(self, parts):
        key = tuple(sorted(o.id for o in parts))
        if key in self._unprop:
            return self._unprop[key]
        legs = tuple(sorted(l for o in parts for l in o.legs))
        res = []
        if len(parts) == 2:
            A, B = parts
            for X, Y in ((A, B), (B, A)):
                kx, fx = X.type
                ky, fy = Y.type
                if kx == "O" and ky == "V" and VECTOR_OF[fx] == fy:     # vertex i g
                    res.append(self._new(legs, X.type, "FFV_ROW", (X.id, Y.id), X.phase * Y.phase * 1j, prop=False))
                if kx == "I" and ky == "V" and VECTOR_OF[fx] == fy:
                    res.append(self._new(legs, X.type, "FFV_COL", (X.id, Y.id), X.phase * Y.phase * 1j, prop=False))
                if kx == "O" and ky == "I" and fx == fy:
                    res.append(self._new(legs, ("V", VECTOR_OF[fx]), "FFV_VEC", (X.id, Y.id), X.phase * Y.phase * 1j, prop=False))
            if A.type == B.type == ("V", "g"):                          # vertex g (real)
                res.append(self._new(legs, ("V", "g"), "VVV", (A.id, B.id), A.phase * B.phase, prop=False))
        else:
            A, B, C = parts
            if A.type == B.type == C.type == ("V", "g"):                # vertex -i g^2
                ph = A.phase * B.phase * C.phase * (-1j)
                for w in (1, 2, 3):
                    res.append(self._new(legs, ("V", "g"), "VVVV%d" % w, (A.id, B.id, C.id), ph, prop=False))
        self._unprop[key] = res
        return res

    def _close_cut(self, big, others, closing_4g):
        """Diagram = (vertex of `others`, left open) . (propagated current `big` over n/2 legs)."""
        made = False
        for U in self._unprop_current(others):
            ku, fu = U.type
            kc, fc = big.type
            if ku == "V" and kc == "V" and fu == fc:
                kind = "V"
            elif {ku, kc} == {"O", "I"} and fu == fc:
                kind = "F"
            else:
                continue
            if not made:
                d = self._count_diagram(tuple(others) + (big,), closing_4g)
                made = True
            self.terms.append(Term("DOT_" + kind, (U.id, big.id), U.phase * big.phase, 0, d))

    def _pick_cut(self, objs):
        """The hanging subtree that stays a propagated current C when the closing vertex is folded into the open
        current U of the others: never the one holding leg 0 (so that U does, and has half the variants by parity);
        the one with the most legs (U then spans the fewest), ties to the highest leg number (fewest distinct leg
        splits).  CUT_ALL = False restricts this to the n/2 | n/2 splits and closes the rest at the vertex."""
        cands = [o for o in objs if 0 not in o.legs]
        if not CUT_ALL:
            cands = [o for o in cands if 2 * len(o.legs) == self.n]
        if not cands:
            return None
        # among equally large ones, one without a frozen leg: U then holds them all and has the fewest variants
        return max(cands, key=lambda o: (len(o.legs), not any(l in o.legs for l in self.frozen), max(o.legs)))

    def _close3(self, A, B, C):
        objs = (A, B, C)
        cut = self._pick_cut(objs)
        if cut is not None:
            self._close_cut(cut, [o for o in objs if o is not cut], False)
            return
        kinds = [o.type[0] for o in objs]
        if sorted(kinds) == ["I", "O", "V"]:
            O = objs[kinds.index("O")]
            I = objs[kinds.index("I")]
            V = objs[kinds.index("V")]
            if O.type[1] == I.type[1] and VECTOR_OF[O.type[1]] == V.type[1]:
                d = self._count_diagram(objs, False)
                self.terms.append(Term("FFV_AMP", (O.id, V.id, I.id), O.phase * I.phase * V.phase * 1j, 0, d))
        elif all(o.type == ("V", "g") for o in objs):
            d = self._count_diagram(objs, False)
            self.terms.append(Term("VVV_AMP", (A.id, B.id, C.id), A.phase * B.phase * C.phase, 0, d))

    # -- colour ------------------------------------------------------------------------------------------------
    # colour tensor of an object: (array, labels); labels = external coloured legs it contains + 'out'
    def _coloured(self, leg):
        return self.legs[leg].flavour in ("g", "t", "q")

    def _col(self, o):
        if o._col is not None:
            return o._col
        A = [self._col(self.objs[a]) for a in o.args]
        if o.op == "EXT":
            leg = o.legs[0]
            if not self._coloured(leg):
                r = (np.ones(()), [])
            else:
                d = 8 if self.legs[leg].flavour == "g" else 3
                r = (np.eye(d, dtype=complex), [leg, "out"])
        elif not all(self._coloured(l) for l in o.legs):
            r = (np.ones(()), [])
        elif o.op == "FFV_ROW":   # psibar_m (T^c)_{mn} -> open n
            r = self._contract("mcn", _T.transpose(1, 0, 2), A[0], "m", A[1], "c", out="n")
        elif o.op == "FFV_COL":   # (T^c)_{mn} psi_n -> open m
            r = self._contract("mcn", _T.transpose(1, 0, 2), A[0], "n", A[1], "c", out="m")
        elif o.op == "FFV_VEC":   # psibar_m (T^c)_{mn} psi_n -> open c
            r = self._contract("mcn", _T.transpose(1, 0, 2), A[0], "m", A[1], "n", out="c")
        elif o.op == "VVV":       # f^{x y e}
            r = self._contract("xye", _F, A[0], "x", A[1], "y", out="e")
        else:
            ff = {"VVVV1": np.einsum("xye,zde->xyzd", _F, _F), "VVVV2": np.einsum("xze,yde->xyzd", _F, _F),
                  "VVVV3": np.einsum("xde,yze->xyzd", _F, _F)}[o.op]
            r = self._contract("xyzd", ff, A[0], "x", A[1], "y", A[2], "z", out="d")
        o._col = r
        return r

    @staticmethod
    def _contract(vlabels, vertex, *rest, out=None):
        """Contract a vertex tensor with operand tensors over their 'out' axes."""
        ops = list(zip(rest[0::2], rest[1::2]))
        letters = iter("abcdefghijklmnopqrstuvwxyz".upper())
        sub_v = {c: next(letters) for c in vlabels}
        inputs, arrays, keep = [], [], []
        for (arr, labels), vl in ops:
            s = ""
            for lab in labels:
                if lab == "out":
                    s += sub_v[vl]
                else:
                    ch = next(letters)
                    s += ch
                    keep.append((lab, ch))
            inputs.append(s)
            arrays.append(arr)
        keep.sort(key=lambda t: t[0])
        out_s = "".join(ch for _, ch in keep) + (sub_v[out] if out else "")
        expr = "".join(sub_v[c] for c in vlabels) + "," + ",".join(inputs) + "->" + out_s
        res = np.einsum(expr, vertex, *arrays, optimize=True)
        return res, [lab for lab, _ in keep] + (["out"] if out else [])

    def _colour(self):
        col_legs = [i for i in range(self.n) if self._coloured(i)]
        glu = [i for i in col_legs if self.legs[i].flavour == "g"]
        self.gluons = glu
        if not col_legs:
            self.flow_perms = [()]
            self.cf_num = np.array([[1]], dtype=np.int64)
            self.cf_den = 1
            for t in self.terms:
                t.flows = [(0, complex(np.round(t.phase)))]
            return
        # Colour basis.  Every quark line has a psi-bar end (row index: outgoing quark, incoming
        # antiquark) and a psi end (column index).  A basis tensor = one string of T's per line,
        # (T^{a..})_{row end of line k, column end of line pi(k)}, the gluons distributed over the strings in order.
        # One line: the n! permutations.  Two lines: 2 pairings x (n+1)! ordered distributions; the gluon exchanged
        # between the lines gives T^a_{ij} T^a_{kl} = (delta_il delta_kj - delta_ij delta_kl / 3) / 2, so the strings
        # come with 1/2 (crossed pairing) and -1/6 (each line closed on itself): those magnitudes are found below and
        # absorbed into the basis tensors, so that every diagram enters a flow with a pure phase, as with one line.
        flavours = sorted({self.legs[i].flavour for i in col_legs if self.legs[i].flavour != "g"}, key=lambda f: f != "t")
        rows = [[i for i in col_legs if self.legs[i].flavour == f and self.legs[i].kind in (LEG_F_OUT, LEG_FB_IN)][0] for f in flavours]
        cols = [[i for i in col_legs if self.legs[i].flavour == f and self.legs[i].kind in (LEG_FB_OUT, LEG_F_IN)][0] for f in flavours]
        nl = len(flavours)
        assert nl in (1, 2)
        perms, basis = [], []
        gl_letter = {g: "abcdefgh"[k] for k, g in enumerate(glu)}
        for pairing in itertools.permutations(range(nl)):
            for s in itertools.permutations(glu):
                for cutpts in itertools.combinations_with_replacement(range(len(s) + 1), nl - 1):
                    bounds = (0,) + cutpts + (len(s),)
                    strings = [s[bounds[k]:bounds[k + 1]] for k in range(nl)]
                    ops, expr_in, lab = [], [], dict(gl_letter)
                    idx = iter("ijklmnopqrstuvwxyz")
                    for k in range(nl):
                        cur = next(idx)
                        lab[rows[k]] = cur
                        for g in strings[k]:
                            nxt = next(idx)
                            expr_in.append(gl_letter[g] + cur + nxt)
                            ops.append(_T)
                            cur = nxt
                        if strings[k]:
                            lab[cols[pairing[k]]] = cur
                        else:       # empty string: delta(row end, column end)
                            nxt = next(idx)
                            expr_in.append(cur + nxt)
                            ops.append(np.eye(3, dtype=complex))
                            lab[cols[pairing[k]]] = nxt
                    out = "".join(lab[l] for l in col_legs)
                    basis.append(np.einsum(",".join(expr_in) + "->" + out, *ops, optimize=True))
                    perms.append((tuple(pairing), tuple(strings)) if nl > 1 else tuple(s))
        self.flow_perms = perms
        nb = len(basis)
        Bm = np.array([b.ravel() for b in basis])
        del basis
        # A term's flow coefficients solve  sum_f c_f B_f = (its colour tensor): an overdetermined consistent system.
        # Small tensors use every entry; for g g -> t tbar g g g (8^5 x 9 entries, 120 flows, 1 890 terms) a fixed random
        # sample of the entries determines c and a second, disjoint sample checks it.
        size = Bm.shape[1]
        if size > 40000:
            pick = np.random.default_rng(20221114).permutation(size)
            sel, chk = np.sort(pick[:12288]), np.sort(pick[12288:24576])
        else:
            sel = chk = np.arange(size)
        Bs, Bc = Bm[:, sel], Bm[:, chk]
        gram = Bs.conj() @ Bs.T
        assert np.linalg.cond(gram) < 1e8, "the sampled colour basis is not independent"
        cfi0 = np.linalg.inv(gram) @ Bs.conj()
        arrs = []
        for t in self.terms:
            arr, labels = self._term_colour(t)
            assert labels == col_legs, (labels, col_legs)
            flat = arr.ravel()
            c = cfi0 @ flat[sel]
            assert np.allclose(Bc.T @ c, flat[chk], atol=1e-9), "colour factor outside the flow basis"
            arrs.append(c)
        # one magnitude per flow (1 with one line): scale the basis tensor by it
        mag = np.ones(nb)
        for f in range(nb):
            m = sorted({Fraction(abs(c[f])).limit_denominator(1000) for c in arrs if abs(c[f]) > 1e-9})
            assert len(m) <= 1, "a colour flow receives diagrams with different magnitudes: %s" % m
            if m:
                mag[f] = float(m[0])
        self.flow_scale = mag
        Bm = Bm * mag[:, None]
        cf = (Bm.conj() @ Bm.T)
        assert np.allclose(cf.imag, 0)
        cf = cf.real
        den = next(d for d in range(1, 4000) if np.allclose(np.rint(cf * d), cf * d, atol=1e-7))
        if nl == 1:
            assert den == {2: 3, 3: 9, 4: 54, 5: 324}.get(len(glu), den)
        num = np.rint(cf * den)
        self.cf_num = num.astype(np.int64)
        self.cf_den = den
        for t, c in zip(self.terms, arrs):
            c = c / mag * t.phase
            flows = []
            for f in range(nb):
                if abs(c[f]) < 1e-9:
                    continue
                z = complex(round(c[f].real), round(c[f].imag))
                assert abs(z - c[f]) < 1e-9 and abs(z) == 1.0 and (z.real == 0 or z.imag == 0), c[f]
                flows.append((f, z))
            t.flows = flows

    def _term_colour(self, t):
        """Colour tensor of a closing term over the external coloured legs (ascending)."""
        ops = [self._col(self.objs[a]) for a in t.args]
        if t.op == "FFV_AMP":
            return self._contract("mcn", _T.transpose(1, 0, 2), ops[0], "m", ops[1], "c", ops[2], "n")
        if t.op == "VVV_AMP":
            return self._contract("xyz", _F, ops[0], "x", ops[1], "y", ops[2], "z")
        if t.op == "DOT_V":   # gluon propagator: delta^{ab}
            return self._contract("xy", np.eye(8), ops[0], "x", ops[1], "y")
        if t.op == "DOT_F":   # quark propagator: delta_{ij}
            return self._contract("xy", np.eye(3), ops[0], "x", ops[1], "y")
        ff = {1: np.einsum("xye,zwe->xyzw", _F, _F), 2: np.einsum("xze,ywe->xyzw", _F, _F),
              3: np.einsum("xwe,yze->xyzw", _F, _F)}[t.which]
        return self._contract("xyzw", ff, ops[0], "x", ops[1], "y", ops[2], "z", ops[3], "w")

    # -- propagator-cut closings: colour-ordered combinations -------------------------------------------------
    def _combo(self, members):
        """members: [(obj id, coefficient in {+-1, +-i})], first coefficient 1.  A single member is the object itself."""
        if len(members) == 1:
            assert members[0][1] == 1
            return members[0][0]
        key = tuple(members)
        if key not in self._combo_ids:
            first = self.objs[members[0][0]]
            o = self._new(first.legs, first.type, "COMBO", tuple(m[0] for m in members), 1, prop=first.prop)
            self.combo_coefs[o.id] = [m[1] for m in members]
            self.combos.append(o)
            self._combo_ids[key] = o.id
        return self._combo_ids[key]

    def factorise(self):
        """Per leg split and colour flow f: sum_{ij} c^f_ij U_i.C_j = sum_r z_r (sum_i a_i U_i).(sum_j b_j C_j)
        by exact rank-1 peeling of the {0,+-1,+-i} matrix c^f; the sums over i and j are taken once per helicity
        variant of n/2 legs, the dot product once per helicity combination."""
        self._combo_ids, self.combo_coefs = {}, {}
        nf = len(self.flow_perms)
        groups = {}
        for t in self.terms:
            if t.op.startswith("DOT"):
                groups.setdefault(self.objs[t.args[0]].legs, []).append(t)
        unit = lambda z: abs(abs(z) - 1) < 1e-9 and (abs(z.real) < 1e-9 or abs(z.imag) < 1e-9)
        rnd = lambda z: complex(round(z.real), round(z.imag))
        for legs in sorted(groups):
            terms = groups[legs]
            us = sorted({t.args[0] for t in terms})
            cs = sorted({t.args[1] for t in terms})
            kind = terms[0].op[-1]
            M = np.zeros((nf, len(us), len(cs)), dtype=complex)
            for t in terms:
                for f, z in t.flows:
                    M[f, us.index(t.args[0]), cs.index(t.args[1])] += z
            for f in range(nf):
                R = M[f].copy()
                guard = 0
                while np.any(np.abs(R) > 1e-9):
                    guard += 1
                    assert guard <= 16
                    i0, j0 = [int(x) for x in np.argwhere(np.abs(R) > 1e-9)[0]]
                    piv = R[i0, j0]
                    a = R[:, j0] / piv          # a[i0] = 1
                    b = R[i0, :] / piv          # b[j0] = 1
                    R = R - piv * np.outer(a, b)
                    R[np.abs(R) < 1e-9] = 0
                    ma = [(us[i], rnd(a[i])) for i in range(len(us)) if abs(a[i]) > 1e-9]
                    mb = [(cs[j], rnd(b[j])) for j in range(len(cs)) if abs(b[j]) > 1e-9]
                    assert unit(piv) and all(unit(z) for _, z in ma + mb), (piv, ma, mb)
                    # normalise so that the first member has coefficient 1; the phases go to the dot product
                    za, zb = ma[0][1], mb[0][1]
                    ma = [(o, rnd(z / za)) for o, z in ma]
                    mb = [(o, rnd(z / zb)) for o, z in mb]
                    self.dots.append((f, self._combo(ma), self._combo(mb), rnd(piv * za * zb), kind))

    # -- views --------------------------------------------------------------------------------------------------
    def used_objects(self):
        """Objects reachable from the closing terms, in dependency order (ids ascending = creation order is NOT
        dependency-safe for memoised recursion, so sort by leaf count then id)."""
        used = set()

        def visit(i):
            if i in used:
                return
            used.add(i)
            for a in self.objs[i].args:
                visit(a)
        for t in self.terms:
            if not t.op.startswith("DOT"):      # DOT terms are evaluated through self.dots
                for a in t.args:
                    visit(a)
        for _, u, c, _, _ in self.dots:
            visit(u)
            visit(c)
        return sorted((self.objs[i] for i in used), key=lambda o: (len(o.legs), o.op == "COMBO", o.id))

    def summary(self):
        return dict(process=self.name, n_diagrams=self.n_diagrams, n_diagrams_4g=self.n_diagrams_4g,
                    n_terms=len(self.terms), n_flows=len(self.flow_perms),
                    n_currents=sum(1 for o in self.used_objects() if o.op not in ("EXT", "COMBO")),
                    n_combos=sum(1 for o in self.used_objects() if o.op == "COMBO"), n_dots=len(self.dots),
                    n_vertex_closings=sum(1 for t in self.terms if not t.op.startswith("DOT")))
