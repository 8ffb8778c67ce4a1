"""Pins for the oracle's g g -> t tbar g g g (the gap widens with the number of
diagrams).  Tier 1 (oracle/me_tier1.cpp: attachment sequences + 120 colour flows) is pinned by the diagram counts, by the
tier-0 amplitude (the definition) per colour and helicity assignment, by the Ward identity, and by Lorentz and Bose
invariance.  A full tier-0 colour sum (8^5 x 9 colours x 128 helicities) is out of reach of a CPU test; the flow
decomposition against single tier-0 amplitudes plus the colour matrix from explicit Gell-Mann traces stands in for it.
CPU only (-m "not gpu")."""
import numpy as np
import pytest

from oracle import ref
from paper_2211_14056_b200.workloads import BY_NAME
from tests.helpers import random_lorentz, transform


def events(n, first=0):
    w = BY_NAME["gg_ttxggg"]
    u = ref.philox_uniform(w.seed, 0, first, w.n_dim, n)
    return ref.rambo_generate(u, w.sqrt_s, w.masses, w.ps_mode)[0]


@pytest.fixture(scope="module")
def me():
    return ref.MatrixElementRef("gg_ttxggg")


def test_counts(me):
    """1 240 diagrams, 295 with a four-gluon vertex, 120 = 5! flows.  Colour-pure terms:
    945 diagrams without a four-gluon vertex + 3 x 285 with one + 9 x 10 with two = 1 890 (SURVEY's 1 830 counts one
    vertex per diagram; the ten diagrams with two four-gluon vertices — three external gluons on one, two on the other,
    5!/(3! 2!) = 10 — carry 9 terms each)."""
    i = me.info()
    assert (i["n_diag"], i["n_diag_4g"], i["n_flow"], i["n_gluon"]) == (1240, 295, 120, 5)
    assert i["n_terms"] == 945 + 3 * 285 + 9 * 10 == 1890


def test_colour_matrix_properties(me):
    """CF_{sigma tau} = Tr(T^sigma (T^tau)^dagger) for 5 gluons: symmetric, integer over 4 x 3^4 = 324 (powers of 1/2 from
    Tr(T^a T^b) = delta/2 and of 1/3 from the Fierz identity), diagonal N_c C_F^5, every row a permutation of the first,
    full rank 120."""
    cf = me.colour_matrix()
    assert np.allclose(cf, cf.T)
    assert np.max(np.abs(cf * 324 - np.round(cf * 324))) < 1e-7
    assert np.max(np.abs(cf * 162 - np.round(cf * 162))) > 0.4      # 162 is not enough
    assert np.allclose(np.diag(cf), 3 * (4.0 / 3) ** 5)
    first = np.sort(np.round(cf[0] * 324))
    for r in cf:
        assert np.array_equal(np.sort(np.round(r * 324)), first)
    assert np.linalg.matrix_rank(cf) == 120


def test_flow_decomposition_vs_definition(me):
    """sum_sigma (T^sigma)_{ij} J_sigma == the tier-0 amplitude for random colour and helicity assignments."""
    T, _ = ref.su3_generators()
    perms = me.flow_perms()
    gl = sorted(perms[0])
    mom = events(2)
    rng = np.random.default_rng(31)
    draw = lambda: (rng.integers(0, 2, 7), [int(rng.integers(0, 8)) if i in gl else int(rng.integers(0, 3)) for i in range(7)])
    checked = tries = 0
    while checked < 8 and tries < 200:
        tries += 1
        hel, col = draw()
        J = me.flows(mom[tries % 2], hel)
        a1 = 0
        for s, perm in enumerate(perms):
            M = np.eye(3, dtype=complex)
            for leg in perm:
                M = M @ T[col[leg]]
            a1 += M[col[2], col[3]] * J[s]
        scale = np.max(np.abs(J))
        if abs(a1) < 1e-3 * scale:
            continue
        a0 = me.amplitude_def(mom[tries % 2], hel, col)
        assert abs(a0 - a1) < 1e-12 * scale
        checked += 1
    assert checked == 8


def test_ward_identity(me):
    mom = events(2)
    base = me.eval(mom)
    for leg in (0, 1, 4, 6):
        me.set_ward_leg(leg)
        try:
            w = me.eval(mom)
        finally:
            me.set_ward_leg(-1)
        assert np.max(w / (base * mom[:, leg, 0] ** 2)) < 1e-20


def test_lorentz_and_bose_invariance(me):
    mom = events(2, first=2)
    base = me.eval(mom)
    L = random_lorentz(np.random.default_rng(8))
    assert np.max(np.abs(me.eval(transform(mom, L)) / base - 1)) < 1e-10
    sw = mom.copy()
    sw[:, [4, 6]] = sw[:, [6, 4]]
    assert np.max(np.abs(me.eval(sw) / base - 1)) < 1e-11
    sw = mom.copy()
    sw[:, [0, 1]] = sw[:, [1, 0]]
    assert np.max(np.abs(me.eval(sw) / base - 1)) < 1e-11
