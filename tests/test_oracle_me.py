"""Pins for the matrix-element oracle (oracle/): things the paper's physics and the mathematics fix,
independent of the oracle's own code.  SURVEY.md §8(c) I lists them; each test cites its row.
CPU only (-m "not gpu").
"""
import itertools
import os

import numpy as np
import pytest

from oracle import ref
from paper_2211_14056_b200.workloads import BY_NAME, PARAMS
from tests.helpers import closed_form_epem_mupmum, closed_form_gg_ttx, mdot, random_lorentz, transform

GOLD = os.path.join(os.path.dirname(__file__), "golden")
QCD = ["gg_ttx", "gg_ttxg", "gg_ttxgg"]


def events(cfg, n, first=0):
    w = BY_NAME[cfg]
    u = ref.philox_uniform(w.seed, 0, first, w.n_dim, n)
    mom, wt = ref.rambo_generate(u, w.sqrt_s, w.masses, w.ps_mode)
    return mom


@pytest.fixture(scope="module")
def me():
    return {p: ref.MatrixElementRef(p) for p in ["epem_mupmum"] + QCD}


# ---- closed forms (exact, every event) ---------------------------------------------------------------
def test_config0_closed_form_full(me):
    """BASELINE.json:configs[0]: all 2^14 events against 2 e^4 (t^2+u^2)/s^2."""
    mom = events("config0", 1 << 14)
    got = me["epem_mupmum"].eval(mom)
    want = closed_form_epem_mupmum(mom, PARAMS["alpha_em"])
    # classic RAMBO momenta are on shell / conserving only to ~1e-11 when the generated directions are nearly
    # parallel (cancellation in Q^2); the closed form is then itself uncertain at that level.
    assert np.max(np.abs(got / want - 1)) < 1e-10
    assert np.median(np.abs(got / want - 1)) < 1e-14


def two_body(sqrt_s, m, n, seed):
    """Exactly on-shell, exactly conserving 2->2 kinematics built by hand (not by RAMBO)."""
    rng = np.random.default_rng(seed)
    c, phi = rng.uniform(-1, 1, n), rng.uniform(0, 2 * np.pi, n)
    c[:4] = [1 - 1e-9, -1 + 1e-9, 0.0, 1 - 1e-4]   # forward / backward / central
    e = sqrt_s / 2
    pa = np.sqrt(e * e - m * m)
    st = np.sqrt(1 - c * c)
    mom = np.zeros((n, 4, 4))
    mom[:, 0] = [e, 0, 0, e]
    mom[:, 1] = [e, 0, 0, -e]
    mom[:, 2, 0] = mom[:, 3, 0] = e
    mom[:, 2, 1:] = np.stack([pa * st * np.cos(phi), pa * st * np.sin(phi), pa * c], -1)
    mom[:, 3, 1:] = -mom[:, 2, 1:]
    return mom, c


def test_closed_forms_exact_kinematics(me):
    """Same two closed forms on hand-built on-shell momenta (incl. cos(theta) = +-(1-1e-9)), written in the
    scattering angle so that the expected value has no cancellation: tolerance 1e-12."""
    mom, c = two_body(100.0, 0.0, 256, 1)
    e2 = 4 * np.pi * PARAMS["alpha_em"]
    want = e2 ** 2 * (1 + c * c)                       # 2 e^4 (t^2+u^2)/s^2 with t,u = -s(1 -+ c)/2
    assert np.max(np.abs(me["epem_mupmum"].eval(mom) / want - 1)) < 1e-12
    m = PARAMS["m_top"]
    mom, c = two_body(1000.0, m, 256, 2)
    beta = np.sqrt(1 - 4 * m * m / 1e6)
    t1, t2, rho = (1 - beta * c) / 2, (1 + beta * c) / 2, 4 * m * m / 1e6
    gs2 = 4 * np.pi * PARAMS["alpha_s"]
    want = gs2 ** 2 * (1 / (6 * t1 * t2) - 3.0 / 8) * (t1 ** 2 + t2 ** 2 + rho - rho ** 2 / (4 * t1 * t2))
    assert np.max(np.abs(me["gg_ttx"].eval(mom) / want - 1)) < 1e-12
    me["gg_ttx"].set_basis(1, 1)
    try:
        assert np.max(np.abs(me["gg_ttx"].eval(mom) / want - 1)) < 1e-12
    finally:
        me["gg_ttx"].set_basis(0, 0)


def test_config1_closed_form(me):
    """SURVEY §8(c) I row 'config 1 me2': tier 1 on 4096 events, tier 0 (brute-force colour) on 8."""
    mom = events("config1", 4096)
    want = closed_form_gg_ttx(mom, PARAMS["alpha_s"], PARAMS["m_top"])
    got = me["gg_ttx"].eval(mom)
    assert np.max(np.abs(got / want - 1)) < 1e-10
    got0 = me["gg_ttx"].eval_def(mom[:8])
    assert np.max(np.abs(got0 / want[:8] - 1)) < 1e-10


def test_closed_form_detects_wrong_mass():
    """The pin has teeth: a 1 permille change of m_t moves me2 by far more than the tolerance."""
    mom = events("config1", 16)
    want = closed_form_gg_ttx(mom, PARAMS["alpha_s"], PARAMS["m_top"])
    bad = ref.MatrixElementRef("gg_ttx", m_top=PARAMS["m_top"] * 1.001).eval(mom)
    assert np.max(np.abs(bad / want - 1)) > 1e-6


# ---- diagram list (exact integers) -------------------------------------------------------------------
def test_diagram_counts(me):
    """PAPER.md:57-58 (Table 1: 36, 267 diagrams) via SURVEY §4: gg channels have 16 and 123."""
    rows = [l.split("|") for l in open(os.path.join(GOLD, "diagram_counts.txt")) if not l.startswith("#")]
    assert len(rows) == 3
    for proc, nd, n4, nt, nf in rows:
        i = me[proc.strip()].info()
        assert (i["n_diag"], i["n_diag_4g"], i["n_terms"], i["n_flow"]) == (int(nd), int(n4), int(nt), int(nf))
    assert me["gg_ttxg"].info()["n_diag"] + 4 * 5 == 36
    assert me["gg_ttxgg"].info()["n_diag"] + 4 * 36 == 267


# ---- colour -------------------------------------------------------------------------------------------
def test_colour_matrix_golden(me):
    """first rows, multisets, diagonal N_c C_F^n, row-permutation structure."""
    for line in open(os.path.join(GOLD, "colour_matrix_rows.txt")):
        if line.startswith("#"):
            continue
        n, den, row, multi = [x.strip() for x in line.split("|")]
        n, den = int(n), int(den)
        cf = me[{2: "gg_ttx", 3: "gg_ttxg", 4: "gg_ttxgg"}[n]].colour_matrix() * den
        assert np.max(np.abs(cf - np.round(cf))) < 1e-9
        cfi = np.round(cf).astype(int)
        assert list(cfi[0]) == [int(x) for x in row.split()]
        want = {int(k): int(v) for k, v in (kv.split(":") for kv in multi.split())}
        vals, counts = np.unique(cfi, return_counts=True)
        assert dict(zip(vals.tolist(), counts.tolist())) == want
        assert np.array_equal(cfi, cfi.T)
        assert np.allclose(np.diag(cf) / den, 3 * (4.0 / 3) ** n)
        assert np.linalg.matrix_rank(cf) == cf.shape[0]
        for r in cfi:  # every row is a permutation of the first
            assert sorted(r) == sorted(cfi[0])


def test_su3_algebra():
    """Tr(T^a T^b) = delta/2, [T^a,T^b] = i f^{abc} T^c, f totally antisymmetric, f^{acd}f^{bcd} = 3 delta."""
    T, f = ref.su3_generators()
    assert np.allclose(np.einsum("aij,bji->ab", T, T), np.eye(8) / 2)
    comm = np.einsum("aij,bjk->abik", T, T) - np.einsum("bij,ajk->abik", T, T)
    assert np.allclose(comm, 1j * np.einsum("abc,cik->abik", f, T))
    assert np.allclose(f, -f.transpose(1, 0, 2)) and np.allclose(f, f.transpose(1, 2, 0))
    assert np.allclose(np.einsum("acd,bcd->ab", f, f), 3 * np.eye(8))
    assert abs(f[0, 1, 2] - 1) < 1e-15 and abs(f[3, 4, 7] - np.sqrt(3) / 2) < 1e-15


@pytest.mark.parametrize("proc,cfg", [("gg_ttxg", "config2"), ("gg_ttxgg", "config3")])
def test_flow_decomposition_vs_definition(me, proc, cfg):
    """SURVEY §8(c) E pin: for random colour assignments sum_sigma (T^sigma)_{ij} J_sigma == tier-0 amplitude."""
    m = me[proc]
    T, _ = ref.su3_generators()
    perms = m.flow_perms()
    gl = sorted(perms[0])
    mom = events(cfg, 2)
    rng = np.random.default_rng(11)
    checked = 0
    while checked < (40 if proc == "gg_ttxg" else 30):
        hel = rng.integers(0, 2, m.n_external)
        col = [int(rng.integers(0, 8)) if i in gl else int(rng.integers(0, 3)) for i in range(m.n_external)]
        a0 = m.amplitude_def(mom[checked % 2], hel, col)
        J = m.flows(mom[checked % 2], hel)
        scale = np.max(np.abs(J))
        a1 = 0
        for s, perm in enumerate(perms):
            M = np.eye(3, dtype=complex)
            for leg in perm:
                M = M @ T[col[leg]]
            a1 += M[col[2], col[3]] * J[s]
        assert abs(a0 - a1) < 1e-12 * scale
        if abs(a0) > 1e-3 * scale:
            checked += 1


def test_tier0_vs_tier1_full_sums(me):
    """Brute-force colour+helicity sum of the definition == J^dagger CF J of the diagrammatic tier."""
    mom = events("config2", 3)
    assert np.max(np.abs(me["gg_ttxg"].eval_def(mom) / me["gg_ttxg"].eval(mom) - 1)) < 1e-12
    mom = events("config3", 1, first=5)
    assert np.max(np.abs(me["gg_ttxgg"].eval_def(mom) / me["gg_ttxgg"].eval(mom) - 1)) < 1e-12


# ---- gauge invariance ---------------------------------------------------------------------------------
@pytest.mark.parametrize("proc,cfg", [("gg_ttx", "config1"), ("gg_ttxg", "config2"), ("gg_ttxgg", "config3")])
def test_ward_identity(me, proc, cfg):
    """SURVEY §8(c) I 'Feynman rules incl. 4g vertex': eps_g -> p_g for one gluon gives zero, for every gluon.
    Ratio is |M(eps->p)|^2 / (|M|^2 * E_g^2): amplitude-level 1e-10 => 1e-20."""
    m = me[proc]
    mom = events(cfg, 6)
    base = m.eval(mom)
    for leg in sorted(m.flow_perms()[0]):
        m.set_ward_leg(int(leg))
        try:
            w = m.eval(mom)
        finally:
            m.set_ward_leg(-1)
        assert np.max(w / (base * mom[:, leg, 0] ** 2)) < 1e-20
        # tier 0 too (per colour, per helicity): one random assignment
    m.set_ward_leg(0)
    try:
        a = m.amplitude_def(mom[0], [0] * m.n_external, [1, 2] + [0, 1] + [3] * (m.n_external - 4))
    finally:
        m.set_ward_leg(-1)
    a_phys = m.amplitude_def(mom[0], [0] * m.n_external, [1, 2] + [0, 1] + [3] * (m.n_external - 4))
    assert abs(a) < 1e-10 * max(abs(a_phys), 1e-30) * mom[0, 0, 0] or abs(a_phys) == 0


# ---- invariances --------------------------------------------------------------------------------------
@pytest.mark.parametrize("proc,cfg", [("epem_mupmum", "config0"), ("gg_ttx", "config1"), ("gg_ttxg", "config2"),
                                      ("gg_ttxgg", "config3")])
def test_lorentz_invariance(me, proc, cfg):
    """SURVEY §8(c) I 'frame independence': common random boost+rotation of all momenta."""
    mom = events(cfg, 8)
    base = me[proc].eval(mom)
    rng = np.random.default_rng(5)
    for _ in range(3):
        L = random_lorentz(rng)
        assert np.max(np.abs(me[proc].eval(transform(mom, L)) / base - 1)) < 1e-10


@pytest.mark.parametrize("proc,cfg", [("epem_mupmum", "config0"), ("gg_ttx", "config1"), ("gg_ttxg", "config2"),
                                      ("gg_ttxgg", "config3")])
def test_basis_independence(me, proc, cfg):
    """SURVEY §8(c) I 'basis independence': helicity spinors <-> fixed-axis, circular <-> linear polarisations."""
    mom = events(cfg, 8)
    m = me[proc]
    base = m.eval(mom)
    try:
        for sb, pb in ((1, 1), (1, 0), (0, 1)):
            m.set_basis(sb, pb)
            assert np.max(np.abs(m.eval(mom) / base - 1)) < 1e-11
    finally:
        m.set_basis(0, 0)


def test_bose_symmetry(me):
    """SURVEY §8(c) I 'Bose symmetry': me2 invariant under p5<->p6 (config 3) and p1<->p2."""
    mom = events("config3", 8)
    base = me["gg_ttxgg"].eval(mom)
    sw = mom.copy()
    sw[:, [4, 5]] = sw[:, [5, 4]]
    assert np.max(np.abs(me["gg_ttxgg"].eval(sw) / base - 1)) < 1e-11
    sw = mom.copy()
    sw[:, [0, 1]] = sw[:, [1, 0]]
    assert np.max(np.abs(me["gg_ttxgg"].eval(sw) / base - 1)) < 1e-11
    mom = events("config2", 8)
    sw = mom.copy()
    sw[:, [0, 1]] = sw[:, [1, 0]]
    assert np.max(np.abs(me["gg_ttxg"].eval(sw) / me["gg_ttxg"].eval(mom) - 1)) < 1e-11


def test_parity_per_helicity(me):
    """SURVEY §8(c) F/I 'parity': colour-summed |M(h)|^2 = |M(-h)|^2 per helicity combination (helicity basis)."""
    m = me["gg_ttxg"]
    cf = m.colour_matrix()
    mom = events("config2", 2)
    m.set_basis(1, 1)
    try:
        for hel in itertools.product((0, 1), repeat=5):
            J = m.flows(mom[0], hel)
            Jf = m.flows(mom[0], [1 - h for h in hel])
            a, b = np.real(np.conj(J) @ cf @ J), np.real(np.conj(Jf) @ cf @ Jf)
            assert abs(a - b) < 1e-11 * max(a, b)
    finally:
        m.set_basis(0, 0)


def test_collinear_limit(me):
    """SURVEY §8(c) I 'overall normalisation of configs 2, 3' (loose, literature): for s56 -> 0 the azimuth-averaged
    me2(gg->ttgg) * 2  ->  (2 g_s^2 / s56) * Pgg(z) * me2(gg->ttg),  Pgg = 2 C_A [z/(1-z) + (1-z)/z + z(1-z)].
    (the factor 2 undoes the 1/2! identical-gluon factor that only the 4-body process carries.)"""
    mom3 = events("config2", 64)
    # pick an event whose final gluon is hard and central
    pt = np.hypot(mom3[:, 4, 1], mom3[:, 4, 2])
    ev = mom3[int(np.argmax(pt))]
    P = ev[4]
    z = 0.37
    Pn = P[1:] / np.linalg.norm(P[1:])
    a = np.cross(Pn, [0.3, -0.5, 0.8]); a /= np.linalg.norm(a)
    b = np.cross(Pn, a)
    kt = 1e-3 * P[0]
    vals = []
    nphi = 16
    for k in range(nphi):
        phi = 2 * np.pi * (k + 0.5) / nphi
        kv = kt * (np.cos(phi) * a + np.sin(phi) * b)
        p5v, p6v = z * P[1:] + kv, (1 - z) * P[1:] - kv
        p5 = np.concatenate([[np.linalg.norm(p5v)], p5v])
        p6 = np.concatenate([[np.linalg.norm(p6v)], p6v])
        # restore momentum conservation exactly by rescaling nothing: energy mismatch is O(kt^2/E), absorbed
        # into the top-pair system by a tiny shift of the incoming energies (keeps all legs on shell to O(kt^2)).
        m4 = np.stack([ev[0], ev[1], ev[2], ev[3], p5, p6])
        dE = (p5[0] + p6[0]) - P[0]
        m4[0, 0] += dE / 2; m4[0, 3] += dE / 2
        m4[1, 0] += dE / 2; m4[1, 3] -= dE / 2
        s56 = mdot(p5 + p6, p5 + p6)
        vals.append(me["gg_ttxgg"].eval(m4[None])[0] * s56)
    lhs = 2 * np.mean(vals)
    gs2 = 4 * np.pi * PARAMS["alpha_s"]
    pgg = 2 * 3.0 * (z / (1 - z) + (1 - z) / z + z * (1 - z))
    rhs = 2 * gs2 * pgg * me["gg_ttxg"].eval(ev[None])[0]
    assert abs(lhs / rhs - 1) < 0.02


# ---- external wavefunctions ---------------------------------------------------------------------------
def _gammas():
    s = [np.array([[0, 1], [1, 0]], complex), np.array([[0, -1j], [1j, 0]]), np.array([[1, 0], [0, -1]], complex)]
    g0 = np.diag([1, 1, -1, -1]).astype(complex)
    gs = [g0]
    for k in range(3):
        g = np.zeros((4, 4), complex)
        g[:2, 2:] = s[k]
        g[2:, :2] = -s[k]
        gs.append(g)
    return gs


def _slash(p):
    g = _gammas()
    return p[0] * g[0] - p[1] * g[1] - p[2] * g[2] - p[3] * g[3]


@pytest.mark.parametrize("basis", [0, 1])
@pytest.mark.parametrize("mass", [0.0, 173.0])
def test_spinor_pins(basis, mass):
    """SURVEY §8(c) B pins: Dirac equation, normalisation, completeness; incl. p along -z exactly and pT tiny."""
    g0 = _gammas()[0]
    rng = np.random.default_rng(3)
    moms = [rng.normal(size=3) * 200 for _ in range(5)] + [np.array([0, 0, -300.0]), np.array([1e-9, -2e-9, -300.0]),
                                                            np.array([0, 0, 250.0])]
    for pv in moms:
        p = np.concatenate([[np.sqrt(mass ** 2 + pv @ pv)], pv])
        ps = _slash(p)
        su = np.zeros((4, 4), complex)
        sv = np.zeros((4, 4), complex)
        for s in (0, 1):
            u = ref.wavefunction("u", p, mass, s, basis)
            v = ref.wavefunction("v", p, mass, s, basis)
            ub, vb = u.conj() @ g0, v.conj() @ g0
            tol = 1e-12 * p[0]
            assert np.max(np.abs((ps - mass * np.eye(4)) @ u)) < tol * np.sqrt(p[0])
            assert np.max(np.abs((ps + mass * np.eye(4)) @ v)) < tol * np.sqrt(p[0])
            assert abs(ub @ u - 2 * mass) < tol and abs(vb @ v + 2 * mass) < tol
            assert abs(u.conj() @ u - 2 * p[0]) < tol and abs(v.conj() @ v - 2 * p[0]) < tol
            su += np.outer(u, ub)
            sv += np.outer(v, vb)
        assert np.max(np.abs(su - (ps + mass * np.eye(4)))) < 1e-12 * p[0]
        assert np.max(np.abs(sv - (ps - mass * np.eye(4)))) < 1e-12 * p[0]


@pytest.mark.parametrize("basis", [0, 1])
def test_polarisation_pins(basis):
    """SURVEY §8(c) B pins: eps.p = 0, eps.eps* = -1, orthogonality, polarisation sum with n-bar = (1,-p-hat)."""
    rng = np.random.default_rng(4)
    moms = [rng.normal(size=3) * 100 for _ in range(5)] + [np.array([0, 0, 500.0]), np.array([0, 0, -500.0]),
                                                            np.array([3e-10, 1e-10, -40.0])]
    metric = np.diag([1.0, -1, -1, -1])
    for pv in moms:
        p = np.concatenate([[np.linalg.norm(pv)], pv])
        e = [ref.wavefunction("eps", p, 0.0, s, basis) for s in (0, 1)]
        for s in (0, 1):
            assert abs(mdot(e[s], p.astype(complex))) < 1e-12 * p[0]
            assert abs(mdot(e[s], e[s].conj()) + 1) < 1e-12
        assert abs(mdot(e[0], e[1].conj())) < 1e-12
        nb = np.concatenate([[1.0], -pv / p[0]])
        want = -metric + (np.outer(p, nb) + np.outer(nb, p)) / mdot(p, nb)
        got = sum(np.outer(x, x.conj()) for x in e)
        assert np.max(np.abs(got - want)) < 1e-11
