"""Workload table: the five configurations of BASELINE.json:configs as plain data.

This module holds NO arithmetic of the method.  It is the one place that both the tests
(oracle side) and bench.py / the product binding read the configuration from: process name,
sqrt(s), final-state masses, seed, event count, phase-space mode, cuts.
"""
from collections import namedtuple

# is_gluon: the final-state partons the jet cuts (p_T > ptj_min, Delta R > dr_min) apply to: the massless ones
Workload = namedtuple("Workload", "name process sqrt_s masses is_gluon seed n_events ps_mode n_dim cuts")

M_TOP = 173.0
PARAMS = dict(alpha_s=0.118, alpha_em=1.0 / 132.507, m_top=M_TOP, w_top=0.0, ptj_min=20.0, dr_min=0.4)

WORKLOADS = [
    # configs[0]: e+ e- -> mu+ mu-, sqrt(s) = 100 GeV, 2^14 events, seed 0, classic RAMBO (8 uniforms)
    Workload("config0", "epem_mupmum", 100.0, (0.0, 0.0), (0, 0), 0, 1 << 14, 0, 8, False),
    # configs[1]: g g -> t tbar, sqrt(s) = 1 TeV, 2^20 events, seed 1
    Workload("config1", "gg_ttx", 1000.0, (M_TOP, M_TOP), (0, 0), 1, 1 << 20, 0, 8, False),
    # configs[2]: g g -> t tbar g, 2^20 events, seed 2, cuts -> weight 0
    Workload("config2", "gg_ttxg", 1000.0, (M_TOP, M_TOP, 0.0), (0, 0, 1), 2, 1 << 20, 0, 12, True),
    # configs[3]: g g -> t tbar g g, 2^24 events, seed 3 — the headline workload
    Workload("config3", "gg_ttxgg", 1000.0, (M_TOP, M_TOP, 0.0, 0.0), (0, 0, 1, 1), 3, 1 << 24, 0, 16, True),
    # configs[4]: Vegas over config 3, D = 3n-4 = 8 (reading R-G3), 50 bins, 5 x 2^24 events, seed 4
    Workload("config4", "gg_ttxgg", 1000.0, (M_TOP, M_TOP, 0.0, 0.0), (0, 0, 1, 1), 4, 1 << 24, 1, 8, True),
    # the literal "10-dimensional" reading of configs[4] — hadronic, momentum fractions x1, x2 in front of
    # the 8 RAMBO-on-diet dimensions, a DECLARED toy gluon density (no PDF grids in the container), sqrt(S) = 13 TeV
    Workload("config4_hadronic", "gg_ttxgg", 13000.0, (M_TOP, M_TOP, 0.0, 0.0), (0, 0, 1, 1), 4, 1 << 24, 2, 10, True),
    # the quark-initiated channels of the paper's hadronic processes p p -> t tbar g (36 = 16 + 4 x 5
    # diagrams) and p p -> t tbar g g (267 = 123 + 4 x 36), PAPER.md:57-58 (Table 1), as partonic events at fixed sqrt(s)
    # like configs 1-3; the final light quark of q g -> t tbar q (g) is a jet like the gluons (cuts apply to it)
    Workload("qqx_ttx", "qqx_ttx", 1000.0, (M_TOP, M_TOP), (0, 0), 11, 1 << 20, 0, 8, False),
    Workload("qqx_ttxg", "qqx_ttxg", 1000.0, (M_TOP, M_TOP, 0.0), (0, 0, 1), 12, 1 << 20, 0, 12, True),
    Workload("qg_ttxq", "qg_ttxq", 1000.0, (M_TOP, M_TOP, 0.0), (0, 0, 1), 13, 1 << 20, 0, 12, True),
    Workload("qqx_ttxgg", "qqx_ttxgg", 1000.0, (M_TOP, M_TOP, 0.0, 0.0), (0, 0, 1, 1), 14, 1 << 22, 0, 16, True),
    Workload("qg_ttxqg", "qg_ttxqg", 1000.0, (M_TOP, M_TOP, 0.0, 0.0), (0, 0, 1, 1), 15, 1 << 22, 0, 16, True),
    # the antiquark-initiated mirror of q g -> t tbar q g (the other reading of the "4 x 36" of PAPER.md:58: q qbar, q g, qbar g)
    Workload("qxg_ttxqxg", "qxg_ttxqxg", 1000.0, (M_TOP, M_TOP, 0.0, 0.0), (0, 0, 1, 1), 16, 1 << 22, 0, 16, True),
    Workload("qxg_ttxqx", "qxg_ttxqx", 1000.0, (M_TOP, M_TOP, 0.0), (0, 0, 1), 17, 1 << 20, 0, 12, True),
    # g g -> t tbar g g g (2 -> 5; 1 240 diagrams, 120 colour flows) — the paper's point is that the
    # gap to the tensorised generator widens with the diagram count; events shaped like config 3
    Workload("gg_ttxggg", "gg_ttxggg", 1000.0, (M_TOP, M_TOP, 0.0, 0.0, 0.0), (0, 0, 1, 1, 1), 21, 1 << 20, 0, 20, True),
]
BY_NAME = {w.name: w for w in WORKLOADS}
VEGAS_BINS = 50
VEGAS_ITERATIONS = 5
VEGAS_ALPHA = 1.5
