"""Emit the CUDA source of one process from its Program (gen/diagrams.py).

Output: paper_2211_14056_b200/csrc/generated/<process>.inc — a struct with
  * the scratch layout of one event: a BASE region (subset momenta, external wavefunctions, the currents that
    feed other currents) and one ROUND region that successive rounds reuse.  Only objects that somebody READS are
    stored: the feeds and the two operands of every propagator-cut dot product;
  * a table of ITEMS (me_tasks.cuh::MeItem / MeMember).  One item = up to NSLOT colour-ordered currents over one leg
    set (the operands of the dot products of one leg split, or one feed), for VPI helicity variants.  Its MEMBERS
    are the bare vertices of the Feynman subdiagrams that enter those currents; they are evaluated in registers, summed
    with their {+-1, +-i} coefficients into the item's accumulators, the common propagator is applied ONCE to each
    sum and only the sums are stored.  (Round 1 stored every member and summed them in separate combination rows:
    444 of 1 041 rows were load-add-store.)  Items are warp-uniform: the 32 lanes are VPI variants x W events;
  * per round, straight-line code `dots(r, sm, h, jr, ji)` for ONE helicity combination (one lane): the
    propagator-cut dot products of the round's leg splits, accumulated straight into the colour-flow vector J
    (steps a7-a8), and `colour(jr, ji)` = J^dagger CF J (step a9).
A round is: items -> barrier -> dots -> barrier; J is carried across rounds (registers, parked in tensor memory while
the next round's items run), so an event needs BASE + max(ROUND) doubles of shared memory.
The file is `__host__ __device__` so tests/ can run it on the CPU for debugging.

Run `python -m paper_2211_14056_b200.gen.emit` to regenerate all processes (done by build()).
"""
import os

from .diagrams import PROCESSES, Program

HERE = os.path.dirname(os.path.abspath(__file__))
OUT_DIR = os.path.join(os.path.dirname(HERE), "csrc", "generated")
NSLOT_MAX = 4
NSLOT = 4            # accumulators (colour-ordered currents) per item
W_EVENTS = 8         # events per CTA (default geometry)
N_WARPS = int(os.environ.get("MADME_GEN_WARPS", "8"))   # warps per CTA: W_EVENTS own an event in the dot stages, all run items
DYNAMIC = False      # True: items listed longest first for a shared work counter (measured, lost 4 %; the kernel uses the fixed map)
N_ROUNDS = int(os.environ.get("MADME_GEN_ROUNDS", "0"))   # 0: the fewest rounds that fit the budget
# Per-process geometry.  w_events: events per CTA (32 / w_events helicity variants per item); frozen: legs whose helicity
# is fixed during one PASS over the event (leg 0 always: parity; more legs = 2^(len-1) passes, each summing the other
# helicities, so that one lane still holds one helicity combination and J of one pass fits tensor memory); chunk: colour
# flows held in registers at a time by the dot stages (0: all of them), the others wait in tensor memory.
GEOMETRY = {"gg_ttxggg": dict(w_events=4, frozen=(0, 6), chunk=int(os.environ.get("MADME_GEN_CHUNK7", "15")), nslot=4,
                              split_items=os.environ.get("MADME_GEN_SPLIT7", "1") == "1",
                              n_warps=int(os.environ.get("MADME_GEN_WARPS7", "12")))}
if os.environ.get("MADME_GEN_CHUNK6"):      # g g -> t tbar g g with J in tensor memory and more warps than events
    GEOMETRY["gg_ttxgg"] = dict(chunk=int(os.environ["MADME_GEN_CHUNK6"]), n_warps=int(os.environ.get("MADME_GEN_WARPS6", "12")))
if os.environ.get("MADME_GEN_W6"):          # g g -> t tbar g g with fewer events per CTA (two CTAs per SM)
    GEOMETRY["gg_ttxgg"] = dict(w_events=int(os.environ["MADME_GEN_W6"]), n_warps=int(os.environ.get("MADME_GEN_WARPS6", os.environ["MADME_GEN_W6"])))
for _kv in filter(None, os.environ.get("MADME_GEN_WPROC", "").split(",")):      # "process:events_per_cta", measurement hook
    GEOMETRY[_kv.split(":")[0]] = dict(w_events=int(_kv.split(":")[1]), n_warps=int(_kv.split(":")[1]))
if os.environ.get("MADME_GEN_PIPE6"):       # g g -> t tbar g g pipelined over this many double-buffered rounds
    GEOMETRY["gg_ttxgg"] = dict(pipe_rounds=int(os.environ["MADME_GEN_PIPE6"]))
FROZEN = (0,)        # set per process by emit_process
SPLIT_THRESHOLD = float(os.environ.get("MADME_GEN_SPLIT_THR", "1.2"))   # split_for_balance: tasks above this x the mean warp load
LPT_PER_UNIT = int(os.environ.get("MADME_GEN_LPT_UNIT", "120"))   # 0 / 0: 58.6 M, 60 / 120: 59.2 M, 120 / 240: 59.7 M, 200 / 100: 58.5 M events/s (g g -> t tbar g g)
LPT_PER_ITEM = int(os.environ.get("MADME_GEN_LPT_ITEM", "240"))


def geometry(name):
    g = dict(w_events=W_EVENTS, frozen=(0,), chunk=0, n_warps=N_WARPS, nslot=int(os.environ.get("MADME_GEN_NSLOT", "4")), pipe_rounds=0)
    g.update(GEOMETRY.get(name, {}))
    return g


def smem_budget_doubles(w_events):
    """doubles per event so that w_events events fit in the 227 KB a CTA can own"""
    return int(os.environ.get("MADME_GEN_SMEM_DOUBLES", str((232448 // (8 * w_events)) - 32 - 16)))


def voff(v):
    """double offset of helicity variant v inside a stored object: 16-byte slots of one 128-byte line, objects with 16
    variants continue in the next group of four lines"""
    return 2 * (v & 7) + 64 * (v >> 3)

OP_SLASH_ROW, OP_SLASH_COL, OP_FFV_VEC, OP_VVV, OP_VVVV = range(5)
KIND_VEC, KIND_ROW, KIND_COL, KIND_OPEN = range(4)
UNIT_OP = {"FFV_ROW": OP_SLASH_ROW, "FFV_COL": OP_SLASH_COL, "FFV_VEC": OP_FFV_VEC, "VVV": OP_VVV, "VVVV": OP_VVVV}

# fp64 operation counts of the routines in csrc/helas.cuh / me_tasks.cuh as written (FMA = 2, add/mul = 1; complex
# mul = 6, complex fma = 8, real x complex fma = 4)
FLOPS_UNIT = {OP_SLASH_ROW: 64, OP_SLASH_COL: 64, OP_FFV_VEC: 72, OP_VVV: 150, OP_VVVV: 186}
FLOPS_ACC = 16                                  # acc += (+-1 | 0) x: one FMA per real component
FLOPS_FIN = {KIND_VEC: 8, KIND_ROW: 66, KIND_COL: 66, KIND_OPEN: 0}
FLOPS_DOT, FLOPS_EXT = 4 * 8, 45


def bits_of(legs):
    """Legs that carry a helicity label inside one pass (leg 0 is fixed at +1 by parity, see diagrams.py; the other frozen
    legs are fixed by the pass)."""
    return [l for l in legs if l not in FROZEN]


def variant_index(sub_legs, sup_legs, v):
    """Variant of the sub-object (legs sub_legs) inside variant v of an object over sup_legs."""
    sup = bits_of(sup_legs)
    r = 0
    for k, l in enumerate(bits_of(sub_legs)):
        r |= ((v >> sup.index(l)) & 1) << k
    return r


class Unit:
    """One bare vertex evaluation: a Feynman subdiagram's last vertex without its propagator.  A four-gluon vertex
    yields three terms (its three colour x Lorentz structures) from one evaluation."""

    def __init__(self, op, args):
        self.op, self.args = op, args
        self.codes = [[0] * NSLOT_MAX for _ in range(3)]     # [term][slot] -> 0 | 4 + k  (coefficient i^k)
        self.swap = [0, 0, 0]                            # [term] -> b: the term enters as i^b x   (Task.solve_phases)
        self.sign = [[0] * NSLOT_MAX for _ in range(3)]      # [term][slot] -> 0 none | 1 plus | 2 minus


class Task:
    def __init__(self, outputs):
        self.outputs = outputs          # stored objects (ids), <= NSLOT
        self.units = []
        self.out_phase = [0] * len(outputs)   # a_s: the stored current is i^(-a_s) x the true one

    def solve_phases(self, fixed_zero):
        """Write every coefficient i^k (slot s, term m) as i^(a_s) (-1)^(n_sm) i^(b_m) with a_s, b_m in {0, 1}: the
        term is rotated once (b_m), enters the accumulators with a SIGN only, and the phase a_s of a stored current
        is absorbed by the dot products that read it.  fixed_zero: a_s = 0 (the current feeds vertices)."""
        import itertools
        ns = len(self.outputs)
        rows = [(u, k) for u in self.units for k in range(3) if any(u.codes[k])]
        choices = [tuple([0] * ns)] if fixed_zero else itertools.product((0, 1), repeat=ns)
        for a in choices:
            sol = {}
            for u, k in rows:
                bs = {((c & 1) ^ a[sl]) for sl, c in enumerate(u.codes[k]) if c}
                if len(bs) > 1:
                    break
                sol[(id(u), k)] = bs.pop()
            else:
                self.out_phase = list(a)
                for u, k in rows:
                    b = sol[(id(u), k)]
                    u.swap[k] = b
                    for sl, c in enumerate(u.codes[k]):
                        if c:
                            n2 = ((c & 3) - a[sl] - b) % 4
                            assert n2 in (0, 2)
                            u.sign[k][sl] = 1 if n2 == 0 else 2       # 1: +, 2: -
                return True
        return False


class Layout:
    """Where every STORED object of one event lives, and the items that compute them.  A leg split = (legs of the
    open side U | the rest); the operands of a split's dot products live in the round region while that split's
    round is processed."""

    def __init__(self, P, n_rounds, cap=None, pipelined=False):
        """cap: the most doubles the operands of one leg split may take in the round region; a larger split is divided
        into PARTS (its open currents U in groups, each with the dot products they enter) that go to different rounds."""
        self.P = P
        objs = P.used_objects()
        self.objs = objs
        all_legs = tuple(range(P.n))
        feeds = set()                      # objects that are inputs of vertices
        for o in objs:
            if o.op != "COMBO":
                feeds.update(o.args)
        dot_ops = set()
        for (_, u, c, _, _) in P.dots:
            dot_ops.update((u, c))
        self.base = [o for o in objs if o.op == "EXT" or o.id in feeds]
        base_ids = {o.id for o in self.base}
        self.stored = [o for o in objs if o.id in base_ids or o.id in dot_ops]
        subsets = sorted({o.legs for o in objs}, key=lambda s: (len(s), s))
        self.subsets = subsets
        self.sub_index = {s: i for i, s in enumerate(subsets)}
        # split of every stored object outside the base: U side -> its own legs; C side -> the complement
        u_sets = {P.objs[d[1]].legs for d in P.dots}
        self.split_of = {}      # stored object outside the base -> (legs of the U side, part)
        for o in self.stored:
            if o.id in base_ids:
                continue
            comp = tuple(l for l in all_legs if l not in o.legs)
            self.split_of[o.id] = (o.legs if (0 in o.legs) else comp, 0)
            assert self.split_of[o.id][0] in u_sets, o.legs
        size = {(s, 0): 0 for s in sorted(u_sets, key=lambda s: (len(s), s))}
        for o in self.stored:
            if o.id in self.split_of:
                size[self.split_of[o.id]] += 8 * self.nv(o)
        if cap:
            for key in sorted(k for k, v in size.items() if v > cap):
                mine = [o for o in self.stored if self.split_of.get(o.id) == key]
                us = [o for o in mine if o.legs == key[0]]
                # the C side must already be resident (base), so that a part is just a group of U's
                assert len(us) == len(mine), "a split that is too large has C operands outside the base"
                # neighbours share bare vertices: order by the members so that a part keeps them together
                us.sort(key=lambda o: (sorted(self.unit_key(m) for m, _ in self.members_of(o)), o.id))
                part, used = 0, 0
                for o in us:
                    need = 8 * self.nv(o)
                    if used + need > cap:
                        part, used = part + 1, 0
                    used += need
                    self.split_of[o.id] = (key[0], part)
                    size[(key[0], part)] = used
        self.part_of_u = {oid: k[1] for oid, k in self.split_of.items() if P.objs[oid].legs == k[0]}
        self.splits = sorted(size, key=lambda k: (len(k[0]), k))
        bins = [[0, []] for _ in range(max(1, min(n_rounds, len(self.splits))))]
        for s_, sz in sorted(size.items(), key=lambda kv: -kv[1]):
            b = min(bins, key=lambda x: x[0])
            b[0] += sz
            b[1].append(s_)
        bins = [b for b in bins if b[1]]
        self.rounds = [sorted(b[1], key=lambda k: (len(k[0]), k)) for b in bins]
        self.round_of = {s_: r for r, b in enumerate(self.rounds) for s_ in b}
        # Fixed-stride storage: a GROUP is 4 lines of 128 B (one line per wavefunction component); an object with nv
        # variants owns nv consecutive 16-byte slots (aligned to nv) in each line, so component c of variant v sits at
        # double offset  group*64 + c*16 + (slot+v)*2 : the four component loads of a wavefunction are ONE address plus
        # the immediates 0, 128, 256, 384 bytes, whatever nv is.  Objects with more than 8 variants take whole groups.
        start = 8 * len(subsets)
        start = ((start + 15) // 16) * 16
        self.off = {}

        def allocate(obj_list, first_group_off):
            groups = []          # free slot bitmaps
            for o in sorted(obj_list, key=lambda o: (-self.nv(o), o.id)):
                nv = self.nv(o)
                assert nv <= (8 if len(FROZEN) == 1 else 16), "objects with more helicity variants need a wider storage"
                if nv == 16:    # two whole groups, consecutive
                    groups.append([True] * 8)
                    groups.append([True] * 8)
                    self.off[o.id] = first_group_off + (len(groups) - 2) * 64
                    continue
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
        if pipelined:
            # two round regions used in turn: the dot products of round r run while the items of round r + 1 are computed
            size = max(allocate(self.round_objs(r), base_end) for r in range(len(self.rounds))) - base_end
            for r in range(len(self.rounds)):
                allocate(self.round_objs(r), base_end + (r % 2) * size)
            tmax = base_end + 2 * size
        else:
            for r in range(len(self.rounds)):
                tmax = max(tmax, allocate(self.round_objs(r), base_end))
        self.smem_doubles = tmax

    def nv(self, o):
        return 1 << len(bits_of(o.legs))

    def round_objs(self, r):
        return [o for o in self.stored if o.id in self.split_of and self.round_of[self.split_of[o.id]] == r]

    def dot_key(self, d):
        """(legs of the U side, part) of a dot product (flow, u, c, phase, kind)"""
        return (self.P.objs[d[1]].legs, self.part_of_u.get(d[1], 0))

    # ---- tasks -------------------------------------------------------------------------------------------------
    def members_of(self, o):
        """[(member object, coefficient)] of a stored object: a combination's members, or the object itself."""
        P = self.P
        if o.op == "COMBO":
            return [(P.objs[a], c) for a, c in zip(o.args, P.combo_coefs[o.id])]
        return [(o, 1)]

    @staticmethod
    def unit_key(m):
        return ("VVVV" if m.op.startswith("VVVV") else m.op, m.args)

    def make_tasks(self, outputs, fixed_zero=False):
        """Tasks (<= NSLOT outputs each) for stored objects over ONE leg set with one propagator flag."""
        outputs = sorted(outputs, key=lambda o: o.id)
        keys = {o.id: {self.unit_key(m) for m, _ in self.members_of(o)} for o in outputs}
        tasks, left = [], list(outputs)
        while left:
            grp = [left.pop(0)]
            have = set(keys[grp[0].id])
            while left and len(grp) < NSLOT:
                best = max(left, key=lambda o: (len(keys[o.id] & have), -len(keys[o.id] - have), -o.id))
                left.remove(best)
                grp.append(best)
                have |= keys[best.id]
            t = Task(grp)
            units = {}
            for s, o in enumerate(grp):
                for m, coef in self.members_of(o):
                    assert m.legs == o.legs and m.prop == o.prop and m.type == o.type
                    k = self.unit_key(m)
                    if k not in units:
                        units[k] = Unit(UNIT_OP[k[0]], m.args)
                        t.units.append(units[k])
                    term = int(m.op[4]) - 1 if m.op.startswith("VVVV") else 0
                    assert units[k].codes[term][s] == 0
                    units[k].codes[term][s] = 4 + {1: 0, 1j: 1, -1: 2, -1j: 3}[coef]
            if t.solve_phases(fixed_zero):
                tasks.append(t)
            else:       # no common rotation: one current per task always works
                assert len(grp) > 1
                for o in grp:
                    tasks += self.make_tasks([o], fixed_zero)
        return tasks

    def task_flops(self, t):
        o = t.outputs[0]
        kind = self.kind_of(o)
        # every term visits accumulators 0, 1 (and 2, 3 of items with more than two currents)
        nacc = 2 if len(t.outputs) <= 2 else 4
        f = sum(FLOPS_UNIT[u.op] + FLOPS_ACC * nacc * sum(1 for term in u.codes if any(term)) for u in t.units)
        return f + FLOPS_FIN[kind] * len(t.outputs)

    def kind_of(self, o):
        if not o.prop:
            return KIND_OPEN
        return {"V": KIND_VEC, "O": KIND_ROW, "I": KIND_COL}[o.type[0]]


def split_flows(P, nf):
    """Two balanced halves of the colour flows such that few U.C contractions feed flows of both halves (those are
    contracted by both warps of an event).  Pairwise exchange to a local optimum from seeded random starts."""
    import random
    if nf < 2:
        return [0] * nf
    groups = {}
    for (f, u, c, z, k) in P.dots:
        groups.setdefault((u, c), set()).add(f)
    gl = [tuple(sorted(v)) for v in groups.values()]

    def cost(h):
        dup, load = 0, [0, 0]
        for fl in gl:
            sides = {h[f] for f in fl}
            dup += len(sides) > 1
            for x in sides:
                load[x] += 1
        return 16 * dup + abs(load[0] - load[1])
    rng = random.Random(20221114)
    best = None
    for trial in range(24 if nf > 6 else 4):
        h = [0] * ((nf + 1) // 2) + [1] * (nf // 2)
        if trial:
            rng.shuffle(h)
        c = cost(h)
        improved = True
        while improved:
            improved = False
            for a in range(nf):
                for b in range(nf):
                    if h[a] == 0 and h[b] == 1:
                        h[a], h[b] = 1, 0
                        c2 = cost(h)
                        if c2 < c:
                            c, improved = c2, True
                        else:
                            h[a], h[b] = 0, 1
        if best is None or c < best[0]:
            best = (c, list(h))
    return best[1]


def pick_rounds(P, budget):
    if N_ROUNDS:
        return Layout(P, N_ROUNDS)
    L = Layout(P, 1)
    if 4 * P.n + L.smem_doubles <= budget:
        return L
    cap = ((budget - 4 * P.n - L.base_doubles) // 64) * 64 - 64     # whole storage groups, one spare for fragmentation
    assert cap >= 512, "the base region leaves no room for a round"
    for n in range(2, 129):
        L = Layout(P, n, cap)
        if 4 * P.n + L.smem_doubles <= budget or n >= len(L.splits):
            return L
    return L


def emit_process(name, n_rounds=None):
    global FROZEN, NSLOT
    geo = geometry(name)
    FROZEN = tuple(geo["frozen"])
    NSLOT = geo["nslot"]
    try:
        return _emit_process(name, n_rounds, geo)
    finally:
        FROZEN, NSLOT = (0,), 4


def _emit_process(name, n_rounds, geo):
    W_EV, CHUNK, NWARPS = geo["w_events"], geo["chunk"], geo["n_warps"]
    VPI = 32 // W_EV
    DOTS_C_PER_U = NWARPS > W_EV or bool(CHUNK)
    P = Program(name, frozen=FROZEN)
    assert all(t.op.startswith("DOT") for t in P.terms), "every diagram must be a propagator-cut contraction"
    PIPE = geo["pipe_rounds"]
    L = Layout(P, PIPE, pipelined=True) if PIPE else (Layout(P, n_rounds) if n_rounds else pick_rounds(P, smem_budget_doubles(W_EV)))
    assert 4 * P.n + L.smem_doubles <= smem_budget_doubles(W_EV), "the event does not fit the CTA's shared memory"
    n = P.n
    nf = len(P.flow_perms)
    W = []
    w = W.append
    s = P.summary()

    # ---- items ---------------------------------------------------------------------------------------------------
    members = []          # 8-word records
    items = []            # 4-word records, in execution order (stage by stage, interleaved over the W_EVENTS warps)
    stage_end, stage_dots = [], []
    cur_flops = 0
    n_tasks = n_units = 0
    sub_i = lambda legs: L.sub_index[legs]

    def massive_of(o):   # the mass of a fermion current is that of its line (flavour)
        return 1 if (o.type[0] in "OI" and any(leg.massive for leg in P.legs if leg.flavour == o.type[1])) else 0

    out_phase = {}        # stored object id -> a: true current = i^a x stored current

    def makespan(task_list):
        """longest-processing-time-first makespan of the stage's items over the warps, and the task that ends last"""
        pend = sorted(((L.task_flops(t), k) for k, t in enumerate(task_list) for _ in range(0, L.nv(t.outputs[0]), VPI)), reverse=True)
        q = [[0, -1] for _ in range(NWARPS)]
        for c, k in pend:
            b = min(q, key=lambda x: x[0])
            b[0] += c
            b[1] = k if b[1] < 0 or L.task_flops(task_list[k]) > L.task_flops(task_list[b[1]]) else b[1]
        worst = max(q, key=lambda x: x[0])
        return worst[0], worst[1]

    def split_for_balance(task_list, fixed_zero):
        """A stage ends when its longest warp does.  With few large items per stage (g g -> t tbar g g g: 11-16 items over 12
        warps, the largest with 36 bare vertices) the largest item IS the stage: split the largest task of the critical warp
        by outputs (two currents each instead of four; the bare vertices both halves need are evaluated twice) while that
        shortens the stage."""
        start = list(task_list)
        task_list = list(task_list)
        for _ in range(64):
            mean = sum(L.task_flops(t) * ((L.nv(t.outputs[0]) + VPI - 1) // VPI) for t in task_list) / NWARPS
            cands = [k for k, t in enumerate(task_list) if len(t.outputs) >= 2 and L.task_flops(t) > SPLIT_THRESHOLD * mean]
            if not cands:
                break
            k = max(cands, key=lambda k: L.task_flops(task_list[k]))
            t = task_list[k]
            half = (len(t.outputs) + 1) // 2
            parts = L.make_tasks(t.outputs[:half], fixed_zero) + L.make_tasks(t.outputs[half:], fixed_zero)
            if max(L.task_flops(p) for p in parts) > 0.9 * L.task_flops(t):
                break       # the halves share nearly every bare vertex: nothing to gain
            task_list = task_list[:k] + parts + task_list[k + 1:]
        return task_list if makespan(task_list)[0] < 0.97 * makespan(start)[0] else start

    def add_stage(task_list, dots_round):
        """Items of the tasks, balanced over the warps by estimated cost (longest first), then interleaved so that
        warp w runs items w, w + W_EVENTS, ... of the stage."""
        nonlocal cur_flops, n_tasks, n_units
        if geo.get("split_items"):
            task_list = split_for_balance(task_list, dots_round < 0)
        pending = []
        for t in task_list:
            o = t.outputs[0]
            nv = L.nv(o)
            for x, a in zip(t.outputs, t.out_phase):
                out_phase[x.id] = a
            n_tasks += 1
            n_units += len(t.units)
            cur_flops += L.task_flops(t) * nv
            for vbase in range(0, nv, VPI):
                # the balance cost adds the interpreter's overhead per bare vertex and per item (fetch, decode, stores)
                pending.append((L.task_flops(t) + LPT_PER_UNIT * len(t.units) + LPT_PER_ITEM, t, vbase))
        pending.sort(key=lambda x: -x[0])
        if DYNAMIC:     # handed out through a shared counter, longest first
            for cost, t, vbase in pending:
                items.append(encode_item(t, vbase))
        else:
            queues = [[0, []] for _ in range(NWARPS)]
            for cost, t, vbase in pending:
                q = min(queues, key=lambda x: x[0])
                q[0] += cost
                q[1].append((t, vbase))
            depth = max(len(q[1]) for q in queues) if pending else 0
            for k in range(depth):
                for q in queues:
                    if k < len(q[1]):
                        items.append(encode_item(*q[1][k]))
                    else:
                        items.append((0, 0, 0, 0))
        stage_end.append(len(items))
        stage_dots.append(dots_round)

    def encode_item(t, vbase):
        o = t.outputs[0]
        nv = L.nv(o)
        first = len(members)
        for u in t.units:
            args = [P.objs[a] for a in u.args]
            offs, vmaps = [], []
            for a in args:
                assert a.id in L.off, "a vertex argument must be a stored object"
                offs.append(L.off[a.id])
                vm = 0
                for j in range(VPI):
                    if vbase + j < nv:
                        vm |= variant_index(a.legs, o.legs, vbase + j) << (4 * j)
                vmaps.append(vm)
            while len(offs) < 3:
                offs.append(0)
                vmaps.append(0)
            assert max(offs) < 65536
            ks = [sub_i(a.legs) for a in args[:2]]
            code = lambda term: u.swap[term] | (sum(c << (2 * sl) for sl, c in enumerate(u.sign[term])) << 1)
            if VPI == 4:    # four entries per argument, one byte each: the variant's offset in 16-byte slots
                slot = lambda vm: sum((voff((vm >> (4 * j)) & 15) // 2) << (8 * j) for j in range(4))
                members.append((u.op | (ks[0] << 8) | (ks[1] << 16), offs[0] | (offs[1] << 16), offs[2],
                                slot(vmaps[0]), code(0) | (code(1) << 9) | (code(2) << 18), slot(vmaps[1]), slot(vmaps[2]), 0))
            else:           # eight 4-bit entries per argument: a word each (w3, w5, w6)
                assert VPI == 8
                members.append((u.op | (ks[0] << 8) | (ks[1] << 16), offs[0] | (offs[1] << 16), offs[2],
                                vmaps[0], code(0) | (code(1) << 9) | (code(2) << 18), vmaps[1], vmaps[2], 0))
        outs = [L.off[x.id] for x in t.outputs] + [0] * NSLOT_MAX
        assert first < 65536 and len(t.units) < 256 and nv < 256
        w0 = len(t.units) | (len(t.outputs) << 8) | (L.kind_of(o) << 12) | (massive_of(o) << 15) | (nv << 16) | (vbase << 24)
        return (w0, first | (sub_i(o.legs) << 16), outs[0] | (outs[1] << 16), outs[2] | (outs[3] << 16))

    for lev in sorted({len(o.legs) for o in L.base if o.op != "EXT"}):
        tasks = []
        for o in L.base:
            if len(o.legs) == lev and o.op != "EXT":
                tasks += L.make_tasks([o], fixed_zero=True)
        add_stage(tasks, -1)
    for r in range(len(L.rounds)):
        cells = {}
        for o in L.round_objs(r):
            cells.setdefault((o.legs, o.prop), []).append(o)
        tasks = []
        for key in sorted(cells):
            tasks += L.make_tasks(cells[key])
        # pipelined: the stage computes the items of round r and the dot products of round r - 1
        add_stage(tasks, r - 1 if PIPE else r)
    if PIPE:
        add_stage([], len(L.rounds) - 1)

    w("// GENERATED by paper_2211_14056_b200/gen/emit.py — do not edit; regenerate with")
    w("//   python -m paper_2211_14056_b200.gen.emit")
    w("// process %s: %d Feynman diagrams (%d with a 4-gluon vertex), %d colour-pure terms, %d colour flows"
      % (name, s["n_diagrams"], s["n_diagrams_4g"], s["n_terms"], s["n_flows"]))
    w("// (SURVEY.md §8 table; PAPER.md:57-58 Table 1 pins 16 and 123 through 36 = 16+4x5, 267 = 123+4x36)")
    w("// evaluation: %d stored currents computed by %d tasks from %d bare vertices, %d propagator-cut dot products per"
      % (sum(1 for o in L.stored if o.op != "EXT"), n_tasks, n_units, s["n_dots"]))
    w("// helicity combination over %d leg splits in %d rounds; %d of %d combinations evaluated (parity, leg 0 at +1)"
      % (len(L.splits), len(L.rounds), 1 << (n - 1), 1 << n))
    n_pass = 1 << (len(FROZEN) - 1)
    hel_legs = bits_of(range(n))            # bit k of a lane's helicity index h is the helicity of leg hel_legs[k]
    if n_pass > 1:
        w("// in %d passes: legs %s are fixed during a pass, a lane holds one combination of the helicities of legs %s"
          % (n_pass, list(FROZEN[1:]), hel_legs))
    w("#pragma once")
    w('#include "../me_tasks.cuh"')
    w("namespace madme {")
    w("struct %s {" % name)
    w("  static constexpr int N_EXT = %d, N_HEL = %d, N_HEL_EVAL = %d, N_FLOW = %d, N_SUB = %d;"
      % (n, 1 << n, 1 << len(hel_legs), nf, len(L.subsets)))
    w("  // geometry: events per CTA; passes over the event with the helicities of the FROZEN legs fixed (leg 0: +1, the")
    w("  // others by the pass index, bit k-1 of it for the k-th frozen leg); colour flows per register chunk (0: all)")
    w("  static constexpr int W_EVENTS = %d, VPI = %d, N_PASS = %d, CHUNK = %d, N_CHUNK = %d;"
      % (W_EV, VPI, n_pass, CHUNK, (nf + CHUNK - 1) // CHUNK if CHUNK else 1))
    w("  static constexpr bool CHUNKED = %s;" % ("true" if CHUNK else "false"))
    w("  // PIPELINED: stage p computes the items of one round while the dot products of the round before it are taken (two")
    w("  // round regions in turn); half of the warps take the dot products first, half the items")
    w("  static constexpr bool PIPELINED = %s;" % ("true" if PIPE else "false"))
    w("  static constexpr int NSLOT = %d;  // accumulators (colour-ordered currents) per item" % NSLOT)
    w("  static constexpr unsigned FROZEN_MASK = %d;" % sum(1 << l for l in FROZEN))
    w("  // helicity of every leg (bit l) for lane index h of pass p; leg 0 at +1")
    w("  static ME_HD int full_helicity(int h, int p) {")
    w("    return 1 | %s;" % " | ".join(["(((h >> %d) & 1) << %d)" % (k, l) for k, l in enumerate(hel_legs)]
                                        + ["(((p >> %d) & 1) << %d)" % (k, l) for k, l in enumerate(FROZEN[1:])]))
    w("  }")
    w("  // fixed helicities of the frozen legs in pass p, as bits at the leg positions")
    w("  static ME_HD unsigned frozen_helicities(int p) {")
    w("    return 1u%s;" % "".join(" | (((unsigned(p) >> %d) & 1u) << %d)" % (k, l) for k, l in enumerate(FROZEN[1:])))
    w("  }")
    w("  static constexpr int N_DIAGRAMS = %d, N_DIAGRAMS_4G = %d, N_TERMS = %d, N_CURRENTS = %d, N_COMBOS = %d, N_DOTS = %d;"
      % (s["n_diagrams"], s["n_diagrams_4g"], s["n_terms"], s["n_currents"], s["n_combos"], s["n_dots"]))
    w("  static constexpr int SMEM_DOUBLES = %d, BASE_DOUBLES = %d;" % (L.smem_doubles, L.base_doubles))
    w("  static constexpr int CF_DEN = %d, AVG_DEN = %d, COUPLING_POWER = %d;  // me2 = g^(2*(n-2)) sum / (CF_DEN*AVG_DEN)"
      % (P.cf_den, P.avg, 2 * (n - 2)))
    w("  static constexpr bool QED = %s;" % ("true" if P.coupling == "ee" else "false"))
    beam = lambda leg: {0: 0, 4: 1, 5: 2}[leg.kind]      # V_IN gluon, F_IN quark, FB_IN antiquark
    w("  static constexpr int BEAM_KIND_0 = %d, BEAM_KIND_1 = %d;  // toy density of each beam in the hadronic Vegas mode" % (beam(P.legs[0]), beam(P.legs[1])))
    w("  // final-state particle i = leg i + 2: massive (m_top), a jet (massless coloured parton: the cuts apply to it)")
    w("  static constexpr unsigned FINAL_MASSIVE_MASK = %d, JET_MASK = %d;"
      % (sum(1 << (l - 2) for l in range(2, n) if P.legs[l].massive),
         sum(1 << (l - 2) for l in range(2, n) if not P.legs[l].massive and P.legs[l].flavour in ("g", "q"))))

    def table_fn(fname, vals):
        w("  static ME_HD int %s(int i) {" % fname)
        w("    switch (i) {")
        for i, e in enumerate(vals):
            w("      case %d: return %d;" % (i, e))
        w("      default: return %d;" % (vals[-1] if vals else 0))
        w("    }")
        w("  }")

    w("  static constexpr int N_ITEMS = %d, N_MEMBERS = %d, N_ROUNDS = %d, N_STAGES = %d, N_TASKS = %d, N_UNITS = %d;"
      % (len(items), len(members), len(L.rounds), len(stage_end), n_tasks, n_units))
    w("  static constexpr int N_WARPS = %d;" % NWARPS)
    w("  // stage p: items up to stage_end(p) (warp w takes items w, w + %d, ...), barrier, then the dot products of round" % NWARPS)
    w("  // stage_dots(p) (if >= 0), barrier")
    table_fn("stage_end", stage_end)
    table_fn("stage_dots", stage_dots)
    w("#define %s_ITEM_TABLE { \\" % name)
    for r4 in items:
        w("  {%du,%du,%du,%du}, \\" % r4)
    w("  {0u,0u,0u,0u} }")
    w("#define %s_MEMBER_TABLE { \\" % name)
    for r8 in members:
        w("  {{%du,%du,%du,%du,%du,%du,%du,%du}}, \\" % r8)
    w("  {{0u,0u,0u,0u,0u,0u,0u,0u}} }")
    sub_flags = {sub: 0 for sub in L.subsets}     # 1: a propagated current lives on the subset, 2: on the massive line
    for o in L.stored:
        if o.op != "EXT" and o.prop:
            sub_flags[o.legs] |= 1 | (2 * massive_of(o))
    w("#define %s_SUB_MASKS { %s }" % (name, ",".join(str(sum(1 << l for l in sub) | (sub_flags[sub] << 16)) for sub in L.subsets)))
    w("#define %s_LEG_KIND { %s }" % (name, ",".join(str(leg.kind) for leg in P.legs)))
    w("#define %s_LEG_MASSIVE { %s }" % (name, ",".join("1" if leg.massive else "0" for leg in P.legs)))
    ext_off = [L.off[o.id] for o in L.objs if o.op == "EXT"]
    assert [o.legs[0] for o in L.objs if o.op == "EXT"] == list(range(n))
    w("#define %s_EXT_OFF { %s }" % (name, ",".join(str(x) for x in ext_off)))

    # ---- dots, round by round ----------------------------------------------------------------------------------
    def ldw(oid):
        o = P.objs[oid]
        terms = ["%d * b%d" % (voff(1 << k), l) for k, l in enumerate(bits_of(o.legs))]
        return "ld_wf(sm + %s)" % " + ".join([str(L.off[oid])] + terms)

    zcode = {1: 0, 1j: 1, -1: 2, -1j: 3}
    by_split = {}
    for d in P.dots:
        by_split.setdefault(L.dot_key(d), []).append(d)
    def emit_round_body(r, keep, local, ind):
        """the dot products of round r that feed the flows in `keep` (global flow -> index into jr/ji given by `local`);
        returns (flop count, number of contractions)"""
        flops = ncon = 0
        for key in L.rounds[r]:
            dots = [d for d in by_split.get(key, []) if d[0] in keep]
            if not dots:
                continue
            w(ind + "{  // split %s | rest%s: %d dot products" % ("".join(str(l) for l in key[0]), " (part %d)" % key[1] if key[1] else "", len(dots)))
            if not DOTS_C_PER_U:
                for c in sorted({d[2] for d in dots}):
                    w(ind + "  const wf4 c%d = %s;" % (c, ldw(c)))
            for u in sorted({d[1] for d in dots}):
                w(ind + "  { const wf4 u = %s;" % ldw(u))
                by_c = {}
                for (f, uu, c, z, kind) in dots:
                    if uu == u:     # the phases i^a of the stored operands go into the dot product's phase
                        by_c.setdefault((c, kind), []).append((local[f], (zcode[z] + out_phase.get(u, 0) + out_phase.get(c, 0)) % 4))
                for (c, kind), fl in sorted(by_c.items()):
                    mink = "true" if kind == "V" else "false"
                    if DOTS_C_PER_U:     # one C operand live at a time
                        w(ind + "    { const wf4 c%d = %s;" % (c, ldw(c)))
                    ncon += 1
                    if len(fl) == 1:
                        w(ind + "    dot_acc<%d, %s>(jr[%d], ji[%d], u, c%d);" % (fl[0][1], mink, fl[0][0], fl[0][0], c))
                        flops += FLOPS_DOT
                    else:   # one contraction feeds several colour flows: computed once, added with each flow's phase
                        w(ind + "    { const cplx t = dot_val<%s>(u, c%d);" % (mink, c))
                        for f, zc in fl:
                            w(ind + "      jadd<%d>(jr[%d], ji[%d], t);" % (zc, f, f))
                        w(ind + "    }")
                        flops += FLOPS_DOT - 4 + 2 * len(fl)
                    if DOTS_C_PER_U:
                        w(ind + "    }")
                w(ind + "  }")
            w(ind + "}")
        return flops, ncon

    def hel_bits():
        for k, l in enumerate(hel_legs):
            w("    const int b%d = (h >> %d) & 1; (void)b%d;" % (l, k, l))

    def emit_dots(fname, keep, local):
        flops = 0
        w("  static ME_HD void %s(int r, const double* __restrict__ sm, int h, double* __restrict__ jr, double* __restrict__ ji) {" % fname)
        hel_bits()
        w("    switch (r) {")
        for r in range(len(L.rounds)):
            w("      case %d: {" % r)
            flops += emit_round_body(r, keep, local, "        ")[0]
            w("      } break;")
        w("      default: break;")
        w("    }")
        w("  }")
        return flops

    w("  // a7-a8: the dot products of round r for helicity combination h (bit k of h is the helicity of the k-th leg that")
    w("  // is not frozen, 0 <-> -1, 1 <-> +1), accumulated into the colour-flow vector J = (jr, ji).")
    if CHUNK:
        return _emit_chunked(W, w, P, L, nf, CHUNK, n_pass, n, cur_flops, emit_round_body, hel_bits, NWARPS)
    amp_flops = emit_dots("dots", set(range(nf)), {f: f for f in range(nf)})

    # ---- colour contraction grouped by distinct CF numerator (9 distinct values for 4 gluons) ----
    cf = P.cf_num

    def emit_colour(signature, pairs):
        """sum over the listed pairs (name_f, name_g, CF numerator, weight 1 (diagonal) | 2) of w CF (re re + im im);
        name = (array prefix, index).  Returns the flop count."""
        w("  static ME_HD double %s {" % signature)
        if not pairs:
            w("    return 0.0;")
            w("  }")
            return 0
        keys = sorted({(v * wt) for (_, _, v, wt) in pairs}, key=lambda v: -abs(v))
        NPART = 2 if len(pairs) > 8 else 1
        nm_of = lambda v: "s%s" % (("m%d" % -v) if v < 0 else str(v))
        for v in keys:
            for p in range(NPART):
                w("    double %s_%d = 0.0;" % (nm_of(v), p))
        cnt = {v: 0 for v in keys}
        flops = 0
        for (fa, ga, v, wt) in pairs:
            nm = "%s_%d" % (nm_of(v * wt), cnt[v * wt] % NPART)
            cnt[v * wt] += 1
            re = lambda a: ("or_[%d]" if a[0] == "o" else "jr[%d]") % a[1]
            im = lambda a: ("oi[%d]" if a[0] == "o" else "ji[%d]") % a[1]
            w("    %s = fma(%s, %s, fma(%s, %s, %s));" % (nm, re(fa), re(ga), im(fa), im(ga), nm))
            flops += 4
        expr = []
        for v in keys:
            expr.append("%d.0 * (%s)" % (v, " + ".join("%s_%d" % (nm_of(v), p) for p in range(NPART))))
            flops += 2
        w("    return " + " + ".join(expr) + ";")
        w("  }")
        return flops

    w("  // a9: sum_{f,f'} J_f^* CFnum_{ff'} J_f'  (CF real symmetric, integer numerators over CF_DEN)")
    all_pairs = [(("j", f), ("j", g), int(cf[f, g]), 1 if f == g else 2) for f in range(nf) for g in range(f, nf)]
    col_flops = emit_colour("colour(const double* __restrict__ jr, const double* __restrict__ ji)", all_pairs)

    # ---- the same for TWO warps per event: each owns half of the colour flows ------------------------------------
    # (me_kernel.cuh, P::SPLIT_J).  Flows are split so that few U.C contractions feed both halves; warp role A holds
    # flows FLOWS_A, role B flows FLOWS_B.  J^dagger CF J = pairs inside A + pairs inside B + cross pairs; role A takes
    # the cross pairs with the first half of B, role B those of its second half with A (read in two chunks).
    half = split_flows(P, nf)
    fl_a = [f for f in range(nf) if half[f] == 0]
    fl_b = [f for f in range(nf) if half[f] == 1]
    na, nb = len(fl_a), len(fl_b)
    ha, hb = (na + 1) // 2, (nb + 1) // 2
    loc = {f: k for k, f in enumerate(fl_a)}
    loc.update({f: k for k, f in enumerate(fl_b)})
    w("  static constexpr int N_FLOW_A = %d, N_FLOW_B = %d, N_FLOW_HALF = %d, CHUNK_A = %d, CHUNK_B = %d;" % (na, nb, max(na, nb, 1), ha, hb))
    w("  // colour flows of warp role A: %s; of role B: %s" % (fl_a, fl_b))
    flops_a = emit_dots("dots_a", set(fl_a), loc)
    flops_b = emit_dots("dots_b", set(fl_b), loc)
    wt = lambda f, g: 1 if f == g else 2
    own_a = [(("j", loc[f]), ("j", loc[g]), int(cf[f, g]), wt(f, g)) for i, f in enumerate(fl_a) for g in fl_a[i:]]
    own_b = [(("j", loc[f]), ("j", loc[g]), int(cf[f, g]), wt(f, g)) for i, f in enumerate(fl_b) for g in fl_b[i:]]
    # o = the other role's chunk, indexed from the chunk's first flow
    cross_a = [(("j", loc[f]), ("o", loc[g]), int(cf[f, g]), 2) for f in fl_a for g in fl_b[:hb]]
    cross_b0 = [(("j", loc[g]), ("o", loc[f]), int(cf[f, g]), 2) for g in fl_b[hb:] for f in fl_a[:ha]]
    cross_b1 = [(("j", loc[g]), ("o", loc[f] - ha), int(cf[f, g]), 2) for g in fl_b[hb:] for f in fl_a[ha:]]
    two = "const double* __restrict__ jr, const double* __restrict__ ji"
    four = two + ", const double* __restrict__ or_, const double* __restrict__ oi"
    fa_ = emit_colour("colour_own_a(%s)" % two, own_a)
    fb_ = emit_colour("colour_own_b(%s)" % two, own_b)
    fca = emit_colour("colour_cross_a(%s)" % four, cross_a)
    fcb0 = emit_colour("colour_cross_b0(%s)" % four, cross_b0)
    fcb1 = emit_colour("colour_cross_b1(%s)" % four, cross_b1)
    w("  static constexpr bool SPLIT_J = %s;" % ("true" if NWARPS == 2 * W_EV else "false"))
    if NWARPS == 2 * W_EV:
        amp_flops, col_flops = flops_a + flops_b, fa_ + fb_ + fca + fcb0 + fcb1
    ext_flops = FLOPS_EXT * 2 * n
    nh = 1 << len(hel_legs)
    assert n_pass == 1
    per_event = ext_flops + cur_flops + nh * (amp_flops + col_flops)
    w("  // nominal fp64 flops per event as emitted (FMA = 2): externals %d + currents %d + %d helicities x"
      % (ext_flops, cur_flops, nh))
    w("  // (dot products %d + colour %d)" % (amp_flops, col_flops))
    w("  static constexpr double FLOPS_PER_EVENT = %d.0;" % per_event)
    w("};")
    w("}  // namespace madme")
    return "\n".join(W) + "\n"


def _emit_chunked(W, w, P, L, nf, CHUNK, n_pass, n, cur_flops, emit_round_body, hel_bits, NWARPS):
    """The dot and colour stages of a process whose colour-flow vector does not fit the registers of a lane: J lives in
    tensor memory (4 N_FLOW 32-bit columns of the warp's lanes), CHUNK flows at a time are loaded, updated by the dot
    products of the round that feed them, and stored back; J^dagger CF J is summed over pairs of chunks."""
    nc = (nf + CHUNK - 1) // CHUNK
    chunk_of = lambda f: f // CHUNK
    flops = ncon = 0
    has = []
    unit_cost = {}
    w("  // dot products of round r that feed the colour flows of chunk c (flow f = c * CHUNK + index into jr / ji)")
    w("  static ME_HD void dots(int r, int c, const double* __restrict__ sm, int h, double* __restrict__ jr, double* __restrict__ ji) {")
    hel_bits()
    w("    switch (r * N_CHUNK + c) {")
    for r in range(len(L.rounds)):
        for c in range(nc):
            keep = {f for f in range(nf) if chunk_of(f) == c}
            mark = len(W)
            w("      case %d: {  // round %d, flows %d..%d" % (r * nc + c, r, c * CHUNK, min(nf, (c + 1) * CHUNK) - 1))
            fl, k = emit_round_body(r, keep, {f: f - c * CHUNK for f in keep}, "        ")
            if k == 0:
                del W[mark:]
                continue
            w("      } break;")
            flops += fl
            ncon += k
            has.append(r * nc + c)
            unit_cost[(r, c)] = fl
    w("      default: break;")
    w("    }")
    w("  }")
    w("  static ME_HD bool has_dots(int r, int c) {")
    w("    switch (r * N_CHUNK + c) {")
    for k in has:
        w("      case %d:" % k)
    w("        return true;")
    w("      default: return false;")
    w("    }")
    w("  }")
    # which of the WG warps of a tensor-memory sub-partition takes the (event, chunk) unit of round r: longest first
    wg = NWARPS // 4
    owner = {}
    for r in range(len(L.rounds)):
        load = [0] * wg
        for c in sorted((c for (rr, c) in unit_cost if rr == r), key=lambda c: -unit_cost[(r, c)]):
            k = load.index(min(load))
            load[k] += unit_cost[(r, c)]
            owner[(r, c)] = k
    w("  // the warp (index within the %d warps of a tensor-memory sub-partition) that takes chunk c in round r: by cost" % wg)
    w("  static ME_HD int dot_owner(int r, int c) {")
    w("    switch (r * N_CHUNK + c) {")
    for (r, c), k in sorted(owner.items()):
        if k:
            w("      case %d: return %d;" % (r * nc + c, k))
    w("      default: return 0;")
    w("    }")
    w("  }")
    w("  static constexpr int N_CONTRACTIONS = %d;  // per helicity combination (a contraction shared by flows of different chunks counts twice)" % ncon)
    cf = P.cf_num

    def body(pairs):
        """sum of wt CF (re re + im im) over pairs, grouped by value so that few partial sums are live at a time"""
        fl = 0
        by_val = {}
        for (fa, ga, v, wt) in pairs:
            by_val.setdefault(v * wt, []).append((fa, ga))
        re = lambda a: ("or_[%d]" if a[0] == "o" else "jr[%d]") % a[1]
        im = lambda a: ("oi[%d]" if a[0] == "o" else "ji[%d]") % a[1]
        w("        double tot = 0.0;")
        for v in sorted(by_val, key=lambda v: -abs(v)):
            if v == 0:
                continue
            lst = by_val[v]
            w("        { double s0 = 0.0, s1 = 0.0;")
            for k, (fa, ga) in enumerate(lst):
                nm = "s%d" % (k & 1)
                w("          %s = fma(%s, %s, fma(%s, %s, %s));" % (nm, re(fa), re(ga), im(fa), im(ga), nm))
                fl += 4
            w("          tot = fma(%d.0, s0 + s1, tot); }" % v)
            fl += 3
        w("        return tot;")
        return fl

    col_flops = 0
    w("  // a9: sum_{f,f'} J_f^* CFnum_{ff'} J_f' as a sum over chunks (diagonal blocks) and pairs of chunks (x 2)")
    w("  static ME_HD double colour_diag(int c, const double* __restrict__ jr, const double* __restrict__ ji) {")
    w("    switch (c) {")
    for c in range(nc):
        fl_ = [f for f in range(nf) if chunk_of(f) == c]
        w("      case %d: {" % c)
        col_flops += body([(("j", f - c * CHUNK), ("j", g - c * CHUNK), int(cf[f, g]), 1 if f == g else 2) for i, f in enumerate(fl_) for g in fl_[i:]])
        w("      }")
    w("      default: return 0.0;")
    w("    }")
    w("  }")
    w("  // chunk ca in (jr, ji), chunk cb > ca in (or_, oi)")
    w("  static ME_HD double colour_pair(int ca, int cb, const double* __restrict__ jr, const double* __restrict__ ji,")
    w("                                  const double* __restrict__ or_, const double* __restrict__ oi) {")
    w("    switch (ca * N_CHUNK + cb) {")
    for ca in range(nc):
        for cb in range(ca + 1, nc):
            fa_ = [f for f in range(nf) if chunk_of(f) == ca]
            fb_ = [f for f in range(nf) if chunk_of(f) == cb]
            w("      case %d: {" % (ca * nc + cb))
            col_flops += body([(("j", f - ca * CHUNK), ("o", g - cb * CHUNK), int(cf[f, g]), 2) for f in fa_ for g in fb_])
            w("      }")
    w("      default: return 0.0;")
    w("    }")
    w("  }")
    w("  static constexpr bool SPLIT_J = false;")
    w("  static constexpr int N_FLOW_HALF = N_FLOW;")
    ext_flops = FLOPS_EXT * 2 * n
    nh = 1 << len(bits_of(range(n)))
    per_event = n_pass * (ext_flops + cur_flops + nh * (flops + col_flops))
    w("  // nominal fp64 flops per event as emitted (FMA = 2): %d passes x (externals %d + currents %d + %d helicities x"
      % (n_pass, ext_flops, cur_flops, nh))
    w("  // (dot products %d + colour %d))" % (flops, col_flops))
    w("  static constexpr double FLOPS_PER_EVENT = %d.0;" % per_event)
    w("};")
    w("}  // namespace madme")
    return "\n".join(W) + "\n"


def emit_all(out_dir=OUT_DIR, only=None, force=False):
    """Regenerate the programs that are older than the generator's sources (g g -> t tbar g g g alone takes half a minute);
    force, or any MADME_GEN_* override in the environment, regenerates everything."""
    os.makedirs(out_dir, exist_ok=True)
    paths = []
    newest = max(os.path.getmtime(os.path.join(HERE, f)) for f in ("emit.py", "diagrams.py"))
    # the MADME_GEN_* overrides the existing files were generated with
    stamp_path = os.path.join(out_dir, ".overrides")
    stamp = repr(sorted((k, v) for k, v in os.environ.items() if k.startswith("MADME_GEN_")))
    if (open(stamp_path).read() if os.path.exists(stamp_path) else "[]") != stamp:
        force = True
    with open(stamp_path, "w") as f:
        f.write(stamp)
    for name in PROCESSES:
        if only and name not in only:
            continue
        path = os.path.join(out_dir, name + ".inc")
        if not force and os.path.exists(path) and os.path.getmtime(path) >= newest:
            paths.append(path)
            continue
        src = emit_process(name)
        old = open(path).read() if os.path.exists(path) else None
        if old != src:
            with open(path, "w") as f:
                f.write(src)
        else:
            os.utime(path)
        paths.append(path)
    return paths


if __name__ == "__main__":
    import sys
    for p in emit_all(force="--force" in sys.argv):
        print(p)
