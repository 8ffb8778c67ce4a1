"""Emit the CUDA source of one process from its Program (gen/diagrams.py).

Output: paper_2211_14056_b200/csrc/generated/<process>.inc — a struct with
  * the scratch layout of one event: a BASE region (subset momenta, external wavefunctions, the currents that
    feed other currents) and one ROUND region that successive rounds reuse,
  * one table of 128-bit task rows (me_tasks.cuh::MeRow) in execution order: the base currents level by level,
    then for every round the open / propagated currents of its leg splits and their colour-ordered combinations,
  * per round, straight-line code `dots(r, sm, h, jr, ji)` for ONE helicity combination (one lane): the
    propagator-cut dot products of the round's leg splits, accumulated straight into the colour-flow vector J
    (steps a7-a8), and `colour(jr, ji)` = J^dagger CF J (step a9).
A round is: tasks -> barrier -> combinations -> barrier -> dots -> barrier; J stays in registers across rounds, so an
event needs BASE + max(ROUND) doubles of shared memory, not the sum over all leg splits.
The file is `__host__ __device__` so tests/ can run it on the CPU for debugging.

Run `python -m paper_2211_14056_b200.gen.emit` to regenerate all processes (done by build()).
"""
import os

from .diagrams import PROCESSES, Program

OPCODE = {"FFV_ROW": 0, "FFV_COL": 1, "FFV_VEC": 2, "VVV": 3, "VVVV1": 4}
OP_COMBO, OP_NOP = 5, 7
HERE = os.path.dirname(os.path.abspath(__file__))
OUT_DIR = os.path.join(os.path.dirname(HERE), "csrc", "generated")
N_ROUNDS = int(os.environ.get("MADME_GEN_ROUNDS", "4"))   # shared-memory footprint knob (see Layout)
GROUP_PAD = int(os.environ.get("MADME_GEN_GROUP_PAD", "4"))   # rows of one op come in multiples of this (a CTA of 8 events maps 4 rows x 8 events on a warp)

# fp64 operation counts of the routines in csrc/helas.cuh as written (FMA = 2, add/mul = 1; complex mul = 1 mul +
# 1 fma per component = 6, complex fma = 8).  (propagated, open) forms.
FLOPS = {
    "FFV_ROW": (8 + 4 * 14 + 2 + 4 * 24 + 8, 8 + 4 * 14),      # slash (4 cadd + 4 (cmul + cfma)) + (Kslash + m) x f
    "FFV_COL": (8 + 4 * 14 + 2 + 4 * 24 + 8, 8 + 4 * 14),
    "FFV_VEC": (8 * 6 + 12 * 2 + 8, 8 * 6 + 12 * 2 + 8),
    "VVV": (12 + 14 * 3 + 4 * 20, 12 + 14 * 3 + 4 * 20),
    "VVVV": (3 * 30 + 6 + 4 * 24, 3 * 30 + 6 + 4 * 24),
    "DOT": 4 * 8, "EXT": 45,
}


def bits_of(legs):
    """Legs that carry a helicity label (leg 0 is fixed at +1 by parity, see diagrams.py)."""
    return [l for l in legs if l != 0]


def variant_index(sub_legs, sup_legs, v):
    """Variant of the sub-object (legs sub_legs) inside variant v of an object over sup_legs."""
    sup = bits_of(sup_legs)
    r = 0
    for k, l in enumerate(bits_of(sub_legs)):
        r |= ((v >> sup.index(l)) & 1) << k
    return r


class Layout:
    """Where every object of one event lives.  A leg split = (legs of the open side U | the rest); all objects that
    only serve one split (its open currents, its top-level propagated currents, the combinations of both sides)
    live in the round region while that split's round is processed."""

    def __init__(self, P, n_rounds):
        self.P = P
        objs = P.used_objects()
        self.objs = objs
        all_legs = tuple(range(P.n))
        subsets = sorted({o.legs for o in objs}, key=lambda s: (len(s), s))
        self.subsets = subsets
        self.sub_index = {s: i for i, s in enumerate(subsets)}
        feeds = set()                      # objects that are inputs of vertex tasks
        for o in objs:
            if o.op != "COMBO":
                feeds.update(o.args)
        self.base = [o for o in objs if o.op == "EXT" or o.id in feeds]
        base_ids = {o.id for o in self.base}
        # split of every other object: U side -> its own legs; C side -> the complement
        u_sets = {P.objs[d[1]].legs for d in P.dots}
        self.split_of = {}
        for o in objs:
            if o.id in base_ids:
                continue
            comp = tuple(l for l in all_legs if l not in o.legs)
            self.split_of[o.id] = o.legs if (0 in o.legs) else comp
            assert self.split_of[o.id] in u_sets, o.legs
        self.splits = sorted(u_sets, key=lambda s: (len(s), s))
        size = {s: 0 for s in self.splits}
        for o in objs:
            if o.id in self.split_of:
                size[self.split_of[o.id]] += 8 * self.nv(o)
        bins = [[0, []] for _ in range(max(1, min(n_rounds, len(self.splits))))]
        for s_, sz in sorted(size.items(), key=lambda kv: -kv[1]):
            b = min(bins, key=lambda x: x[0])
            b[0] += sz
            b[1].append(s_)
        bins = [b for b in bins if b[1]]
        self.rounds = [sorted(b[1], key=lambda s: (len(s), s)) for b in bins]
        self.round_of = {s_: r for r, b in enumerate(self.rounds) for s_ in b}
        # Fixed-stride storage: a GROUP is 4 lines of 128 B (one line per wavefunction component); an object with nv
        # variants owns nv consecutive 16-byte slots (aligned to nv) in each line, so component c of variant v sits at
        # double offset  group*64 + c*16 + (slot+v)*2 : the four component loads of a wavefunction are ONE address plus
        # the immediates 0, 128, 256, 384 bytes, whatever nv is.
        start = 8 * len(subsets)
        start = ((start + 15) // 16) * 16
        self.off = {}

        def allocate(obj_list, first_group_off):
            groups = []          # free slot bitmaps
            for o in sorted(obj_list, key=lambda o: (-self.nv(o), o.id)):
                nv = self.nv(o)
                assert nv <= 8
                for gi, used in enumerate(groups):
                    slot = next((s0 for s0 in range(0, 8, nv) if not any(used[s0:s0 + nv])), None)
                    if slot is not None:
                        break
                else:
                    groups.append([False] * 8)
                    gi, slot, used = len(groups) - 1, 0, groups[-1]
                for k in range(nv):
                    used[slot + k] = True
                self.off[o.id] = first_group_off + gi * 64 + slot * 2
            return first_group_off + len(groups) * 64

        base_end = allocate(self.base, start)
        self.base_doubles = base_end
        tmax = base_end
        for r in range(len(self.rounds)):
            tmax = max(tmax, allocate([o for o in objs if o.id in self.split_of and self.round_of[self.split_of[o.id]] == r], base_end))
        self.smem_doubles = tmax

    def nv(self, o):
        return 1 << len(bits_of(o.legs))

    def round_objs(self, r):
        return [o for o in self.objs if o.id in self.split_of and self.round_of[self.split_of[o.id]] == r]


def emit_process(name, n_rounds=None):
    P = Program(name)
    assert all(t.op.startswith("DOT") for t in P.terms), "every diagram must be a propagator-cut contraction"
    L = Layout(P, N_ROUNDS if n_rounds is None else n_rounds)
    n = P.n
    nf = len(P.flow_perms)
    W = []
    w = W.append
    s = P.summary()
    w("// GENERATED by paper_2211_14056_b200/gen/emit.py — do not edit; regenerate with")
    w("//   python -m paper_2211_14056_b200.gen.emit")
    w("// process %s: %d Feynman diagrams (%d with a 4-gluon vertex), %d colour-pure terms, %d colour flows"
      % (name, s["n_diagrams"], s["n_diagrams_4g"], s["n_terms"], s["n_flows"]))
    w("// (SURVEY.md §8 table; PAPER.md:57-58 Table 1 pins 16 and 123 through 36 = 16+4x5, 267 = 123+4x36)")
    w("// evaluation: %d off-shell currents, %d colour-ordered combinations and %d propagator-cut dot products per"
      % (s["n_currents"], s["n_combos"], s["n_dots"]))
    w("// helicity combination over %d leg splits in %d rounds; %d of %d combinations evaluated (parity, leg 0 at +1)"
      % (len(L.splits), len(L.rounds), 1 << (n - 1), 1 << n))
    w("#pragma once")
    w('#include "../me_tasks.cuh"')
    w("namespace madme {")
    w("struct %s {" % name)
    w("  static constexpr int N_EXT = %d, N_HEL = %d, N_HEL_EVAL = %d, N_FLOW = %d, N_SUB = %d;"
      % (n, 1 << n, 1 << (n - 1), nf, len(L.subsets)))
    w("  static constexpr int N_DIAGRAMS = %d, N_DIAGRAMS_4G = %d, N_TERMS = %d, N_CURRENTS = %d, N_COMBOS = %d, N_DOTS = %d;"
      % (s["n_diagrams"], s["n_diagrams_4g"], s["n_terms"], s["n_currents"], s["n_combos"], s["n_dots"]))
    w("  static constexpr int SMEM_DOUBLES = %d, BASE_DOUBLES = %d;" % (L.smem_doubles, L.base_doubles))
    w("  static constexpr int CF_DEN = %d, AVG_DEN = %d, COUPLING_POWER = %d;  // me2 = g^(2*(n-2)) sum / (CF_DEN*AVG_DEN)"
      % (P.cf_den, P.avg, 2 * (n - 2)))
    w("  static constexpr bool QED = %s;" % ("true" if P.coupling == "ee" else "false"))

    # ---- the task table --------------------------------------------------------------------------------------
    rows = []
    cur_flops = 0
    lg = lambda nv: {1: 0, 2: 1, 4: 2, 8: 3, 16: 4, 32: 5}[nv]
    sub_i = lambda o: L.sub_index[o.legs]

    def pad(mult):
        while len(rows) % mult:
            rows.append((0, 0, OP_NOP << 24, 0))

    def add_tasks(objs):
        nonlocal cur_flops
        for opn, prop in [(a, b) for a in ("FFV_ROW", "FFV_COL", "FFV_VEC", "VVV", "VVVV1") for b in (True, False)]:
            for o in objs:
                if o.op != opn or o.prop != prop:   # open and propagated currents in separate groups: uniform branches
                    continue
                args = [P.objs[a] for a in o.args]
                nv = L.nv(o)
                sibs = []
                if opn == "VVVV1":
                    sibs = [x for x in L.objs if x.op in ("VVVV2", "VVVV3") and x.args == o.args and x.legs == o.legs and x.prop == o.prop]
                    sibs.sort(key=lambda x: x.op)
                    assert len(sibs) == 2
                massive = 1 if (o.type[0] in "OI" and P.legs[[l for l in o.legs if P.legs[l].kind >= 2][0]].massive) else 0
                for v in range(nv):
                    offs = [L.off[a.id] + 2 * variant_index(a.legs, o.legs, v) for a in args] + [0]
                    assert max(offs) < 65536 and L.off[o.id] + 2 * v < 65536
                    x = (L.off[o.id] + 2 * v) | (offs[0] << 16)
                    y = offs[1] | ((offs[2] if len(args) > 2 else 0) << 16)
                    flags = (OPCODE[opn] << 24) | (massive << 27) | ((0 if o.prop else 1) << 28)
                    if sibs:   # four-gluon current: no argument momenta needed; the two sibling outputs take their place
                        z = sub_i(o) | ((L.off[sibs[0].id] + 2 * v) << 8) | flags
                        wv = L.off[sibs[1].id] + 2 * v
                        assert L.off[sibs[0].id] + 2 * v < 65536
                    else:
                        z = sub_i(o) | (sub_i(args[0]) << 8) | (sub_i(args[1]) << 16) | flags
                        wv = 0
                    rows.append((x, y, z, wv))
                    cur_flops += FLOPS["VVVV" if opn == "VVVV1" else opn][0 if o.prop else 1]
            pad(GROUP_PAD)
        pad(32)

    def add_combos(objs):
        nonlocal cur_flops
        for o in objs:
            if o.op != "COMBO":
                continue
            coefs = P.combo_coefs[o.id]
            assert len(coefs) <= 4 and coefs[0] == 1
            nv = L.nv(o)
            for v in range(nv):
                m = [L.off[a] + 2 * v for a in o.args] + [0, 0, 0]
                k = [{1: 0, 1j: 1, -1: 2, -1j: 3}[zc] for zc in coefs] + [0, 0, 0]
                x = (L.off[o.id] + 2 * v) | (m[0] << 16)
                y = m[1] | (m[2] << 16)
                z = m[3] | (OP_COMBO << 24)
                wv = (len(coefs) << 16) | (k[1] << 22) | (k[2] << 24) | (k[3] << 26)
                rows.append((x, y, z, wv))
                cur_flops += 8 * (len(coefs) - 1)
        pad(32)

    base_ends = []
    for lev in sorted({len(o.legs) for o in L.base if o.op != "EXT"}):
        add_tasks([o for o in L.base if len(o.legs) == lev and o.op != "EXT"])
        base_ends.append(len(rows))
    raw_ends, combo_ends = [], []
    for r in range(len(L.rounds)):
        ro = L.round_objs(r)
        add_tasks(ro)
        raw_ends.append(len(rows))
        add_combos(ro)
        combo_ends.append(len(rows))

    def table_fn(fname, vals):
        w("  static ME_HD int %s(int i) {" % fname)
        w("    switch (i) {")
        for i, e in enumerate(vals):
            w("      case %d: return %d;" % (i, e))
        w("      default: return %d;" % (vals[-1] if vals else 0))
        w("    }")
        w("  }")

    # phases: rows up to phase_end(p), barrier, then (if phase_dots(p) >= 0) the dot products of that round, barrier
    ph_end = list(base_ends)
    ph_dots = [-1] * len(base_ends)
    for r in range(len(L.rounds)):
        if raw_ends[r] > (ph_end[-1] if ph_end else 0) and combo_ends[r] > raw_ends[r]:
            ph_end.append(raw_ends[r])
            ph_dots.append(-1)
        ph_end.append(combo_ends[r])
        ph_dots.append(r)
    w("  static constexpr int N_ROWS = %d, N_ROUNDS = %d, N_PHASES = %d;" % (len(rows), len(L.rounds), len(ph_end)))
    w("  // phase p: task rows up to phase_end(p), barrier, then the dot products of round phase_dots(p) (if >= 0), barrier")
    table_fn("phase_end", ph_end)
    table_fn("phase_dots", ph_dots)
    w("#define %s_TASK_TABLE { \\" % name.upper())
    for r4 in rows:
        w("  {%du,%du,%du,%du}, \\" % r4)
    w("  {0u,0u,%du,0u} }" % (OP_NOP << 24))
    w("#define %s_SUB_MASKS { %s }" % (name.upper(), ",".join(str(sum(1 << l for l in sub)) for sub in L.subsets)))
    w("#define %s_LEG_KIND { %s }" % (name.upper(), ",".join(str(leg.kind) for leg in P.legs)))
    w("#define %s_LEG_MASSIVE { %s }" % (name.upper(), ",".join("1" if leg.massive else "0" for leg in P.legs)))
    ext_off = [L.off[o.id] for o in L.objs if o.op == "EXT"]
    assert [o.legs[0] for o in L.objs if o.op == "EXT"] == list(range(n))
    w("#define %s_EXT_OFF { %s }" % (name.upper(), ",".join(str(x) for x in ext_off)))

    # ---- dots, round by round ----------------------------------------------------------------------------------
    def ldw(oid):
        o = P.objs[oid]
        terms = ["%d * b%d" % (2 << k, l) for k, l in enumerate(bits_of(o.legs))]
        return "ld_wf(sm + %s)" % " + ".join([str(L.off[oid])] + terms)

    zcode = {1: 0, 1j: 1, -1: 2, -1j: 3}
    by_split = {}
    for d in P.dots:
        by_split.setdefault(P.objs[d[1]].legs, []).append(d)
    amp_flops = 0
    w("  // a7-a8: the dot products of round r for helicity combination h (leg 0 has helicity +1; bit l-1 of h is the")
    w("  // helicity of leg l, 0 <-> -1, 1 <-> +1), accumulated into the colour-flow vector J = (jr, ji).")
    w("  static ME_HD void dots(int r, const double* __restrict__ sm, int h, double* __restrict__ jr, double* __restrict__ ji) {")
    for l in range(1, n):
        w("    const int b%d = (h >> %d) & 1; (void)b%d;" % (l, l - 1, l))
    w("    switch (r) {")
    for r, split_list in enumerate(L.rounds):
        w("      case %d: {" % r)
        for legs in split_list:
            dots = by_split[legs]
            w("        {  // split %s | rest: %d dot products" % ("".join(str(l) for l in legs), len(dots)))
            for c in sorted({d[2] for d in dots}):
                w("          const wf4 c%d = %s;" % (c, ldw(c)))
            for u in sorted({d[1] for d in dots}):
                w("          { const wf4 u = %s;" % ldw(u))
                for (f, uu, c, z, kind) in dots:
                    if uu == u:
                        w("            dot_acc<%d, %s>(jr[%d], ji[%d], u, c%d);" % (zcode[z], "true" if kind == "V" else "false", f, f, c))
                        amp_flops += FLOPS["DOT"]
                w("          }")
            w("        }")
        w("      } break;")
    w("      default: break;")
    w("    }")
    w("  }")

    # ---- colour contraction grouped by distinct CF numerator (9 distinct values for 4 gluons) ----
    w("  // a9: sum_{f,f'} J_f^* CFnum_{ff'} J_f'  (CF real symmetric, integer numerators over CF_DEN)")
    w("  static ME_HD double colour(const double* __restrict__ jr, const double* __restrict__ ji) {")
    cf = P.cf_num
    vals = sorted({int(cf[f, g]) for f in range(nf) for g in range(f, nf)}, key=lambda v: -abs(v))
    NPART = 2 if nf > 2 else 1
    nm_of = lambda v: "s%s" % (("m%d" % -v) if v < 0 else str(v))
    for v in vals:
        for p in range(NPART):
            w("    double %s_%d = 0.0;" % (nm_of(v), p))
    cnt = {v: 0 for v in vals}
    col_flops = 0
    for f in range(nf):
        for g in range(f, nf):
            v = int(cf[f, g])
            nm = "%s_%d" % (nm_of(v), cnt[v] % NPART)
            cnt[v] += 1
            w("    %s = fma(jr[%d], jr[%d], fma(ji[%d], ji[%d], %s));" % (nm, f, g, f, g, nm))
            col_flops += 4
    diag_vals = {int(cf[f, f]) for f in range(nf)}
    expr = []
    for v in vals:
        tot = " + ".join("%s_%d" % (nm_of(v), p) for p in range(NPART))
        # off-diagonal pairs count twice (CF symmetric); a value on the diagonal must not also be off-diagonal
        on_diag = v in diag_vals
        off_diag = any(int(cf[f, g]) == v for f in range(nf) for g in range(f + 1, nf))
        assert not (on_diag and off_diag), "colour value on and off the diagonal: split the accumulators"
        expr.append("%d.0 * (%s)" % (v if on_diag else 2 * v, tot))
        col_flops += 2
    w("    return " + " + ".join(expr) + ";")
    w("  }")
    ext_flops = FLOPS["EXT"] * 2 * n
    nh = 1 << (n - 1)
    per_event = ext_flops + cur_flops + nh * (amp_flops + col_flops)
    w("  // nominal fp64 flops per event as emitted (FMA = 2): externals %d + currents and combinations %d + %d helicities x"
      % (ext_flops, cur_flops, nh))
    w("  // (dot products %d + colour %d)" % (amp_flops, col_flops))
    w("  static constexpr double FLOPS_PER_EVENT = %d.0;" % per_event)
    w("};")
    w("}  // namespace madme")
    return "\n".join(W) + "\n"


def emit_all(out_dir=OUT_DIR, only=None):
    os.makedirs(out_dir, exist_ok=True)
    paths = []
    for name in PROCESSES:
        if only and name not in only:
            continue
        src = emit_process(name)
        path = os.path.join(out_dir, name + ".inc")
        old = open(path).read() if os.path.exists(path) else None
        if old != src:
            with open(path, "w") as f:
                f.write(src)
        paths.append(path)
    return paths


if __name__ == "__main__":
    for p in emit_all():
        print(p)
