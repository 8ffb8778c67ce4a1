"""Pins for the oracle's quark-initiated channels (Table 1): q qbar -> t tbar (g)(g) and
q g -> t tbar q (g).  Two quark lines of different flavour: tier 0 (oracle/me_tier0.cpp, colour-dressed recursion +
brute-force sums) is the definition, tier 1 runs in the diagram basis (oracle/me_tier1g.cpp).  CPU only (-m "not gpu").
"""
import os

import numpy as np
import pytest

from oracle import ref
from paper_2211_14056_b200.workloads import BY_NAME, PARAMS
from tests.helpers import mdot, random_lorentz, transform

GOLD = os.path.join(os.path.dirname(__file__), "golden")
CHANNELS = ["qqx_ttx", "qqx_ttxg", "qg_ttxq", "qqx_ttxgg", "qg_ttxqg"]


def events(cfg, n, first=0):
    w = BY_NAME[cfg]
    u = ref.philox_uniform(w.seed, 0, first, w.n_dim, n)
    return ref.rambo_generate(u, w.sqrt_s, w.masses, w.ps_mode)[0]


@pytest.fixture(scope="module")
def me():
    return {p: ref.MatrixElementRef(p) for p in CHANNELS + ["gg_ttx", "gg_ttxg", "gg_ttxgg"]}


def closed_form_qqx_ttx(mom, alpha_s, m):
    """Textbook heavy-quark production by light-quark annihilation, averaged over initial spins and colours:
    g_s^4 (4/9) [tau1^2 + tau2^2 + rho/2], tau1 = (m^2 - t)/s, tau2 = (m^2 - u)/s, rho = 4 m^2 / s."""
    s = mdot(mom[:, 0] + mom[:, 1], mom[:, 0] + mom[:, 1])
    t = mdot(mom[:, 0] - mom[:, 2], mom[:, 0] - mom[:, 2])
    u = mdot(mom[:, 0] - mom[:, 3], mom[:, 0] - mom[:, 3])
    t1, t2, rho = (m * m - t) / s, (m * m - u) / s, 4 * m * m / s
    return (4 * np.pi * alpha_s) ** 2 * (4.0 / 9) * (t1 ** 2 + t2 ** 2 + rho / 2)


def test_diagram_counts_reproduce_the_papers_totals(me):
    """36 and 267 diagrams = the gg channel + four quark channels (tests/golden/..._quark_channels.txt)."""
    rows = [l.split("|") for l in open(os.path.join(GOLD, "diagram_counts_quark_channels.txt")) if not l.startswith("#")]
    assert len(rows) == 5
    for proc, nd, n4, nt in rows:
        i = me[proc.strip()].info()
        assert (i["n_diag"], i["n_diag_4g"], i["n_terms"]) == (int(nd), int(n4), int(nt))
    n = lambda p: me[p].info()["n_diag"]
    assert n("gg_ttxg") + 2 * n("qqx_ttxg") + 2 * n("qg_ttxq") == 36
    assert n("gg_ttxgg") + 2 * n("qqx_ttxgg") + 2 * n("qg_ttxqg") == 267


def test_qqx_ttx_closed_form(me):
    """Every event of a 4096-event sample against the closed form (tier 1), 8 events of tier 0; exact hand-built
    kinematics written in the scattering angle (no cancellation) at 1e-12."""
    mom = events("qqx_ttx", 4096)
    want = closed_form_qqx_ttx(mom, PARAMS["alpha_s"], PARAMS["m_top"])
    assert np.max(np.abs(me["qqx_ttx"].eval(mom) / want - 1)) < 1e-10
    assert np.max(np.abs(me["qqx_ttx"].eval_def(mom[:8]) / want[:8] - 1)) < 1e-10
    rng = np.random.default_rng(2)
    n, m, e = 128, PARAMS["m_top"], 500.0
    c, phi = rng.uniform(-1, 1, n), rng.uniform(0, 2 * np.pi, n)
    c[:3] = [1 - 1e-9, -1 + 1e-9, 0.0]
    pa, st = np.sqrt(e * e - m * m), np.sqrt(1 - c * c)
    mom = np.zeros((n, 4, 4))
    mom[:, 0], mom[:, 1] = [e, 0, 0, e], [e, 0, 0, -e]
    mom[:, 2, 0] = mom[:, 3, 0] = e
    mom[:, 2, 1:] = np.stack([pa * st * np.cos(phi), pa * st * np.sin(phi), pa * c], -1)
    mom[:, 3, 1:] = -mom[:, 2, 1:]
    beta, rho = pa / e, m * m / (e * e)
    want = (4 * np.pi * PARAMS["alpha_s"]) ** 2 * (4.0 / 9) * (((1 - beta * c) / 2) ** 2 + ((1 + beta * c) / 2) ** 2 + rho / 2)
    assert np.max(np.abs(me["qqx_ttx"].eval(mom) / want - 1)) < 1e-12


def test_closed_form_pin_has_teeth():
    """a wrong colour average (1/8 instead of 1/9) or a 1 permille top mass is far outside the tolerance"""
    mom = events("qqx_ttx", 16)
    want = closed_form_qqx_ttx(mom, PARAMS["alpha_s"], PARAMS["m_top"])
    bad = ref.MatrixElementRef("qqx_ttx", m_top=PARAMS["m_top"] * 1.001).eval(mom)
    assert np.max(np.abs(bad / want - 1)) > 1e-6


@pytest.mark.parametrize("proc,n", [("qqx_ttxg", 3), ("qg_ttxq", 3), ("qqx_ttxgg", 1), ("qg_ttxqg", 1)])
def test_tier0_vs_tier1_full_sums(me, proc, n):
    """Brute-force colour + helicity sum of the definition == the diagram-basis sum A^T CM A*."""
    mom = events(proc, n, first=3)
    assert np.max(np.abs(me[proc].eval_def(mom) / me[proc].eval(mom) - 1)) < 1e-12


@pytest.mark.parametrize("proc", CHANNELS)
def test_amplitude_per_colour_and_helicity(me, proc):
    """sum_k C_k[colours] A_k[helicities] of the diagram basis == the tier-0 amplitude, for random assignments."""
    m = me[proc]
    mom = events(proc, 2)
    rng = np.random.default_rng(17)
    n, checked, tries = m.n_external, 0, 0
    gluon = [i for i in range(n) if (proc.startswith("qg") and i == 1) or i >= (5 if proc.startswith("qg") else 4)]
    draw = lambda: (rng.integers(0, 2, n), [int(rng.integers(0, 8)) if i in gluon else int(rng.integers(0, 3)) for i in range(n)])
    scale = max(abs(m.amplitude_def(mom[0], *draw())) for _ in range(60))   # most assignments vanish by colour conservation
    assert scale > 0
    while checked < 12 and tries < 4000:
        tries += 1
        hel, col = draw()
        a0 = m.amplitude_def(mom[tries % 2], hel, col)
        a1 = m.amplitude_diag(mom[tries % 2], hel, col)
        assert abs(a0 - a1) < 1e-12 * scale
        if abs(a0) > 1e-3 * scale:
            checked += 1
    assert checked == 12


@pytest.mark.parametrize("proc", ["qqx_ttxg", "qg_ttxq", "qqx_ttxgg", "qg_ttxqg"])
def test_ward_identity(me, proc):
    """eps_g -> p_g for any one external gluon gives zero, per colour and helicity assignment, in both tiers (the
    amplitude is linear in the diagrams, so the cancellation shows to ~1e-13 of the physical amplitude x E_g).  The summed
    |M|^2 of the diagram basis is a quadratic form A^T CM A* evaluated on a null vector of CM's kernel: it vanishes only
    to the rounding of that form, ~1e-15 of |M|^2 E_g^2 (the flow basis of the gg channels reaches 1e-20)."""
    m = me[proc]
    mom = events(proc, 6)
    base = m.eval(mom)
    n = m.n_external
    gluon = [i for i in range(n) if (proc.startswith("qg") and i == 1) or i >= (5 if proc.startswith("qg") else 4)]
    assert len(gluon) == m.info()["n_gluon"]
    rng = np.random.default_rng(23)
    draw = lambda: (rng.integers(0, 2, n), [int(rng.integers(0, 8)) if i in gluon else int(rng.integers(0, 3)) for i in range(n)])
    picks = [draw() for _ in range(300)]    # most random colour assignments vanish: keep the largest amplitudes
    phys = [abs(m.amplitude_diag(mom[0], h, c)) for h, c in picks]
    scale = max(phys)
    assert scale > 0
    picks = [picks[i] for i in np.argsort(phys)[::-1][:(40 if n < 6 else 12)]]
    for leg in gluon:
        m.set_ward_leg(leg)
        try:
            w = m.eval(mom)
            a1 = [m.amplitude_diag(mom[0], h, c) for h, c in picks]
            a0 = [m.amplitude_def(mom[0], h, c) for h, c in picks[:6]]
        finally:
            m.set_ward_leg(-1)
        assert np.max(w / (base * mom[:, leg, 0] ** 2)) < 1e-13
        assert max(abs(a) for a in a1) < 1e-11 * scale * mom[0, leg, 0]
        assert max(abs(a) for a in a0) < 1e-11 * scale * mom[0, leg, 0]


@pytest.mark.parametrize("proc", CHANNELS)
def test_lorentz_and_basis_independence(me, proc):
    mom = events(proc, 6)
    m = me[proc]
    base = m.eval(mom)
    rng = np.random.default_rng(5)
    for _ in range(2):
        L = random_lorentz(rng)
        assert np.max(np.abs(m.eval(transform(mom, L)) / base - 1)) < 1e-10
    try:
        for sb, pb in ((1, 1), (1, 0), (0, 1)):
            m.set_basis(sb, pb)
            assert np.max(np.abs(m.eval(mom) / base - 1)) < 1e-11
    finally:
        m.set_basis(0, 0)


def test_bose_and_charge_conjugation_symmetry(me):
    """q qbar -> t tbar g g is symmetric under p4 <-> p5 (identical gluons); QCD conserves C: exchanging q <-> qbar
    together with t <-> tbar (momenta p0 <-> p1, p2 <-> p3) leaves the summed |M|^2 of q qbar -> t tbar + gluons unchanged."""
    mom = events("qqx_ttxgg", 6)
    base = me["qqx_ttxgg"].eval(mom)
    sw = mom.copy()
    sw[:, [4, 5]] = sw[:, [5, 4]]
    assert np.max(np.abs(me["qqx_ttxgg"].eval(sw) / base - 1)) < 1e-11
    for proc in ("qqx_ttx", "qqx_ttxg", "qqx_ttxgg"):
        mom = events(proc, 6)
        cc = mom.copy()
        cc[:, [0, 1]] = cc[:, [1, 0]]
        cc[:, [2, 3]] = cc[:, [3, 2]]
        assert np.max(np.abs(me[proc].eval(cc) / me[proc].eval(mom) - 1)) < 1e-11


@pytest.mark.parametrize("proc,cfg,n", [("gg_ttx", "config1", 16), ("gg_ttxg", "config2", 8), ("gg_ttxgg", "config3", 3)])
def test_diagram_basis_equals_flow_basis(me, proc, cfg, n):
    """The two tier-1 organisations of the SAME diagrams — attachment sequences + colour flows (me_tier1.cpp) and explicit
    trees + the colour matrix between diagrams (me_tier1g.cpp) — give the same |M|^2 and the same diagram counts."""
    mom = events(cfg, n)
    m = me[proc]
    assert np.max(np.abs(m.eval_diag(mom) / m.eval(mom) - 1)) < 1e-12
    i, d = m.info(), m.info_diag()
    assert (i["n_diag"], i["n_terms"], i["n_diag_4g"]) == (d["n_diag"], d["n_terms"], d["n_diag_4g"])


def test_antiquark_initiated_mirror_channels():
    """qbar g -> t tbar qbar (g): 5 / 36 diagrams like q g -> t tbar q (g); tier 0 == tier 1; by charge conjugation the
    summed |M|^2 equals that of the quark-initiated channel with the t and tbar momenta exchanged."""
    for a, b, nd in (("qxg_ttxqx", "qg_ttxq", 5), ("qxg_ttxqxg", "qg_ttxqg", 36)):
        ma, mb = ref.MatrixElementRef(a), ref.MatrixElementRef(b)
        assert ma.info()["n_diag"] == nd
        mom = events(a, 6)
        cc = mom.copy()
        cc[:, [2, 3]] = cc[:, [3, 2]]
        assert np.max(np.abs(ma.eval(mom) / mb.eval(cc) - 1)) < 1e-12
        k = 2 if nd == 5 else 1
        assert np.max(np.abs(ma.eval_def(mom[:k]) / ma.eval(mom[:k]) - 1)) < 1e-12


# ---- crossing ----------------------------------------------------------------------------------------------------
def _gamma():
    s = [np.array([[0, 1], [1, 0]], complex), np.array([[0, -1j], [1j, 0]]), np.array([[1, 0], [0, -1]], complex)]
    g = [np.diag([1, 1, -1, -1]).astype(complex)]
    for k in range(3):
        m = np.zeros((4, 4), complex)
        m[:2, 2:] = s[k]
        m[2:, :2] = -s[k]
        g.append(m)
    return g


def _spin_sum(kind, k, mass):
    """sum over the spin states of w_a conj(w_b) for the wavefunction w the oracle puts on a leg of this kind with
    all-incoming momentum k, written with the completeness relations sum u ubar = pslash + m, sum v vbar = pslash - m,
    sum eps*_mu eps_nu = -g_mu_nu (one external gluon) — analytic in k, so it continues to crossed (unphysical) momenta."""
    g = _gamma()
    sl = lambda p: p[0] * g[0] - p[1] * g[1] - p[2] * g[2] - p[3] * g[3]
    one = np.eye(4)
    if kind == "g":
        return np.diag([-1.0, 1.0, 1.0, 1.0]).astype(complex)
    if kind == "u":      # incoming fermion, column, p = k
        return (sl(k) + mass * one) @ g[0]
    if kind == "vbar":   # incoming antifermion, row, p = k
        return g[0] @ ((sl(k) - mass * one) @ g[0]).T @ g[0]
    if kind == "ubar":   # outgoing fermion, row, p = -k
        return g[0] @ ((sl(-k) + mass * one) @ g[0]).T @ g[0]
    if kind == "v":      # outgoing antifermion, column, p = -k
        return (sl(-k) - mass * one) @ g[0]
    raise ValueError(kind)


def _summed_me2_from_open_tensor(m, k, kinds, masses):
    """sum over colours and spins of |M|^2 from the wavefunction-stripped tier-0 amplitude and completeness relations"""
    S = [_spin_sum(kd, k[i], masses[i]) for i, kd in enumerate(kinds)]
    total = 0.0
    for c0 in range(3):
        for c1 in range(3):
            for c2 in range(3):
                for c3 in range(3):
                    for a in range(8):
                        T = m.open_tensor(k, [c0, c1, c2, c3, a])
                        if not np.any(T):
                            continue
                        X = np.einsum("abcde,af,bg,ch,di,ej->fghij", T, S[0], S[1], S[2], S[3], S[4], optimize=True)
                        total += np.real(np.vdot(T, X))      # sum conj(T)[fghij] X[fghij]
    return total


def test_crossing_qqx_ttxg_to_qg_ttxq(me):
    """SURVEY §8(f) N1 pin: the colour- and spin-summed |M|^2 of q g -> t tbar q is minus that of q qbar -> t tbar g
    continued to crossed momenta (antiquark in -> quark out, gluon out -> gluon in; one crossed fermion: the minus sign).
    The continuation uses the q qbar -> t tbar g amplitude of tier 0 with its wavefunctions stripped (it is a rational
    function of the momenta) and completeness relations; first checked on physical momenta against the same process."""
    mt = PARAMS["m_top"]
    kinds, masses = ["u", "vbar", "ubar", "v", "g"], [0.0, 0.0, mt, mt, 0.0]
    qqx = me["qqx_ttxg"]
    p = events("qqx_ttxg", 1)[0]
    k = np.array([p[0], p[1], -p[2], -p[3], -p[4]])
    assert abs(_summed_me2_from_open_tensor(qqx, k, kinds, masses) / 36.0 / qqx.eval(p[None])[0] - 1) < 1e-11
    # q(p0) g(p1) -> t(p2) tbar(p3) q(p4): in the q qbar -> t tbar g amplitude the antiquark leg carries k = -p4 and the
    # gluon leg k = +p1
    q = events("qg_ttxq", 2)[1]
    kx = np.array([q[0], -q[4], -q[2], -q[3], q[1]])
    crossed = -_summed_me2_from_open_tensor(qqx, kx, kinds, masses) / 96.0
    assert abs(crossed / me["qg_ttxq"].eval(q[None])[0] - 1) < 1e-10
