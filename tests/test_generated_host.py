"""The build-time generator (gen/) and the vertex library (csrc/helas.cuh), checked WITHOUT a GPU: the generated
programs are compiled with g++ (tests/host/host_harness.cpp emulates the 32 lanes sequentially) and compared with
the oracle.  The harness is test-only; libmadme.so has no CPU path."""
import ctypes as C
import os
import subprocess

import numpy as np
import pytest

from oracle import ref
from paper_2211_14056_b200.gen import diagrams, emit
from paper_2211_14056_b200.workloads import BY_NAME, PARAMS

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def host():
    emit.emit_all()
    so = os.path.join(HERE, "host", "libhost_harness.so")
    src = os.path.join(HERE, "host", "host_harness.cpp")
    subprocess.check_call(["g++", "-std=c++17", "-O1", "-shared", "-fPIC", "-o", so, src])
    lib = C.CDLL(so)
    lib.host_me_eval.argtypes = [C.c_char_p, C.c_void_p, C.c_void_p, C.c_longlong, C.c_double, C.c_double, C.c_void_p, C.c_int]
    return lib


def _momenta(cfg, n):
    w = BY_NAME[cfg]
    r = ref.philox_uniform(w.seed, 0, 0, w.n_dim, n)
    return ref.rambo_generate(r, w.sqrt_s, w.masses, w.ps_mode)[0]


@pytest.mark.parametrize("name,nd,n4,nt,nf", [("gg_ttx", 3, 0, 3, 2), ("gg_ttxg", 16, 1, 18, 6), ("gg_ttxgg", 123, 18, 159, 24)])
def test_generator_counts(name, nd, n4, nt, nf):
    """PAPER.md:57-58 (36 = 16 + 4x5, 267 = 123 + 4x36) and tests/golden/diagram_counts.txt."""
    s = diagrams.Program(name).summary()
    assert (s["n_diagrams"], s["n_diagrams_4g"], s["n_terms"], s["n_flows"]) == (nd, n4, nt, nf)


def test_diagram_counts_of_the_hadronic_processes():
    """PAPER.md:57-58 (Table 1) prints 36 diagrams for p p -> t tbar g and 267 for p p -> t tbar g g.  The generator's own
    enumeration of every partonic channel reproduces both totals: 36 = 16 (gg) + 4 x 5 (q qbar, qbar q, q g, g q) and
    267 = 123 + 4 x 36 (tests/golden/diagram_counts_quark_channels.txt: diagrams, with a four-gluon vertex, terms).
    g g -> t tbar g g g: 1 240 diagrams, 295 with a four-gluon vertex — 10 of those with two (three
    external gluons on one, two on the other), hence 945 + 3 x 285 + 9 x 10 = 1 890 colour-pure terms (SURVEY's 1 830
    counts one vertex each)."""
    n = lambda name: diagrams.Program(name, count_only=True)
    counts = {}
    for line in open(os.path.join(HERE, "golden", "diagram_counts_quark_channels.txt")):
        if line.startswith("#") or not line.strip():
            continue
        proc, nd, n4, nt = [x.strip() for x in line.split("|")]
        s = diagrams.Program(proc).summary()
        assert (s["n_diagrams"], s["n_diagrams_4g"], s["n_terms"]) == (int(nd), int(n4), int(nt))
        counts[proc] = s["n_diagrams"]
    assert counts == {"qqx_ttx": 1, "qqx_ttxg": 5, "qqx_ttxgg": 36, "qg_ttxq": 5, "qg_ttxqg": 36}
    gg = {k: diagrams.Program(k).summary()["n_diagrams"] for k in ("gg_ttxg", "gg_ttxgg")}
    assert gg["gg_ttxg"] + 2 * counts["qqx_ttxg"] + 2 * counts["qg_ttxq"] == 36
    assert gg["gg_ttxgg"] + 2 * counts["qqx_ttxgg"] + 2 * counts["qg_ttxqg"] == 267
    big = n("gg_ttxggg")
    assert (big.n_diagrams, big.n_diagrams_4g, len(big.terms)) == (1240, 295, 1890)
    assert len(big.terms) == (1240 - 295) + 3 * 285 + 9 * 10


def test_gg_ttxggg_generated_program_matches_oracle(host):
    """the chunked form (two passes over the helicity of the last gluon, 120 flows in chunks of 20, splits
    divided into parts over 9 rounds) on the CPU harness against the oracle's tier 1."""
    w = BY_NAME["gg_ttxggg"]
    mom = _momenta("gg_ttxggg", 6)
    out = np.empty(6)
    hel = np.zeros((6, 128))
    g = np.sqrt(4 * np.pi * PARAMS["alpha_s"])
    assert host.host_me_eval(b"gg_ttxggg", mom.ctypes.data, out.ctypes.data, 6, PARAMS["m_top"], g, hel.ctypes.data, 0) == 0
    expect = ref.MatrixElementRef("gg_ttxggg").eval(mom)
    assert np.max(np.abs(out / expect - 1)) < 1e-11
    assert np.max(np.abs(2 * hel.sum(1) / expect - 1)) < 1e-11      # the harness stores each evaluated combination once


def test_generator_colour_matrix_golden():
    rows = {}
    for line in open(os.path.join(HERE, "golden", "colour_matrix_rows.txt")):
        if line.startswith("#") or not line.strip():
            continue
        n, den, row, _ = [x.strip() for x in line.split("|")]
        rows[int(n)] = (int(den), [int(x) for x in row.split()])
    for name, n in (("gg_ttx", 2), ("gg_ttxg", 3), ("gg_ttxgg", 4)):
        P = diagrams.Program(name)
        assert P.cf_den == rows[n][0]
        assert list(P.cf_num[0]) == rows[n][1]


@pytest.mark.parametrize("split", [0, 1])
@pytest.mark.parametrize("cfg,n", [("config0", 64), ("config1", 64), ("config2", 32), ("config3", 12), ("qqx_ttx", 64),
                                   ("qqx_ttxg", 32), ("qg_ttxq", 32), ("qqx_ttxgg", 16), ("qg_ttxqg", 16), ("qxg_ttxqx", 32),
                                   ("qxg_ttxqxg", 16)])
def test_generated_program_matches_oracle(host, cfg, n, split):
    """split = 1: the form with two warps per event, each holding half of the colour flows (me_kernel.cuh, SPLIT_J)."""
    w = BY_NAME[cfg]
    mom = _momenta(cfg, n)
    out = np.empty(n)
    qed = w.process == "epem_mupmum"
    g = np.sqrt(4 * np.pi * (PARAMS["alpha_em"] if qed else PARAMS["alpha_s"]))
    assert host.host_me_eval(w.process.encode(), mom.ctypes.data, out.ctypes.data, n, 0.0 if qed else PARAMS["m_top"], g, None, split) == 0
    expect = ref.MatrixElementRef(w.process).eval(mom)
    assert np.max(np.abs(out / expect - 1)) < 1e-11
