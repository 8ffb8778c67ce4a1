"""GPU parity of the quark-initiated channels (Table 1: the other 20 of the 36 and
144 of the 267 diagrams of p p -> t tbar g / t tbar g g): q qbar -> t tbar (g)(g), q g -> t tbar q (g) through the C ABI
against the oracle's diagram-basis tier 1 (oracle/me_tier1g.cpp), per event at 1e-10, on the same seeded momenta."""
import numpy as np
import pytest
import torch

from oracle import ref
from paper_2211_14056_b200 import api
from paper_2211_14056_b200.workloads import BY_NAME, PARAMS, VEGAS_ALPHA, VEGAS_BINS
from tests.helpers import mdot, momentum_violation, random_lorentz, transform

pytestmark = pytest.mark.gpu
ME_RTOL = 1e-10
CHANNELS = ["qqx_ttx", "qqx_ttxg", "qg_ttxq", "qqx_ttxgg", "qg_ttxqg", "qxg_ttxqx", "qxg_ttxqxg"]


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def oracle_events(cfg, n, first=0):
    w = BY_NAME[cfg]
    r = ref.philox_uniform(w.seed, 0, first, w.n_dim, n)
    return ref.rambo_generate(r, w.sqrt_s, w.masses, w.ps_mode)[0]


@pytest.fixture(scope="module")
def handles():
    return {p: api.me_init(p, PARAMS) for p in CHANNELS}


@pytest.mark.parametrize("proc,n", [("qqx_ttx", 20000 + 13), ("qqx_ttxg", 6000 + 5), ("qg_ttxq", 6000 + 5), ("qqx_ttxgg", 3000 + 7),
                                    ("qg_ttxqg", 3000 + 7), ("qxg_ttxqx", 3000 + 5), ("qxg_ttxqxg", 3000 + 7)])
def test_me_eval_matches_oracle(handles, proc, n):
    """Element by element; sizes span many CTAs and a ragged tail."""
    mom = oracle_events(proc, n)
    want = ref.MatrixElementRef(proc).eval(mom)
    got = api.me_eval(handles[proc], dev(mom)).cpu().numpy()
    rel = np.abs(got / want - 1)
    assert momentum_violation(mom).max() < 1e-12
    assert np.max(rel) < ME_RTOL, (np.argmax(rel), np.max(rel))


def test_qqx_ttx_closed_form_full_size(handles):
    """All 2^20 events against the textbook closed form g_s^4 (4/9)[tau1^2 + tau2^2 + rho/2] (a property computable at any size)."""
    w = BY_NAME["qqx_ttx"]
    r = api.philox_uniform(w.seed, 0, 0, w.n_dim, w.n_events)
    momg, _ = api.rambo_generate(r, w.sqrt_s, w.masses, 0)
    got = api.me_eval(handles["qqx_ttx"], momg).cpu().numpy()
    mom = momg.cpu().numpy()
    s = mdot(mom[:, 0] + mom[:, 1], mom[:, 0] + mom[:, 1])
    t = mdot(mom[:, 0] - mom[:, 2], mom[:, 0] - mom[:, 2])
    u = mdot(mom[:, 0] - mom[:, 3], mom[:, 0] - mom[:, 3])
    m = PARAMS["m_top"]
    want = (4 * np.pi * PARAMS["alpha_s"]) ** 2 * (4.0 / 9) * (((m * m - t) / s) ** 2 + ((m * m - u) / s) ** 2 + 2 * m * m / s)
    assert momentum_violation(mom).max() < 1e-12
    assert np.max(np.abs(got / want - 1)) < ME_RTOL


@pytest.mark.parametrize("proc", ["qqx_ttxgg", "qg_ttxqg"])
def test_sampled_at_full_size(handles, proc):
    """The workload's full 2^22 events on the GPU; a strided sample of 2048 of them against the oracle."""
    w = BY_NAME[proc]
    r = api.philox_uniform(w.seed, 0, 0, w.n_dim, w.n_events)
    momg, _ = api.rambo_generate(r, w.sqrt_s, w.masses, 0)
    got = api.me_eval(handles[proc], momg)
    assert bool(torch.isfinite(got).all()) and bool((got > 0).all())
    idx = np.arange(0, w.n_events, w.n_events // 2048)
    mom = momg[torch.from_numpy(idx).cuda()].cpu().numpy()
    want = ref.MatrixElementRef(proc).eval(mom)
    rel = np.abs(got.cpu().numpy()[idx] / want - 1)
    cut = ref.cuts(mom, w.is_gluon, PARAMS["ptj_min"], PARAMS["dr_min"]) != 0
    assert np.max(rel[cut]) < ME_RTOL, np.max(rel[cut])
    assert np.max(rel) < 1e-8    # cut-failing events (weight 0): soft / collinear cancellations, DESIGN.md §7


@pytest.mark.parametrize("proc", ["qqx_ttxg", "qg_ttxqg"])
def test_lorentz_invariance(handles, proc):
    mom = oracle_events(proc, 2048)
    base = api.me_eval(handles[proc], dev(mom)).cpu().numpy()
    L = random_lorentz(np.random.default_rng(9))
    got = api.me_eval(handles[proc], dev(transform(mom, L))).cpu().numpy()
    assert np.max(np.abs(got / base - 1)) < 1e-9


@pytest.mark.parametrize("proc,mode,n", [("qqx_ttxg", 1, 3000 + 1), ("qg_ttxq", 0, 3000 + 1), ("qqx_ttxgg", 1, 1500 + 3), ("qg_ttxqg", 1, 1500 + 3)])
def test_vegas_integrand_matches_oracle(handles, proc, mode, n):
    """Fused a1-a11 (the cuts take the final light quark of q g -> t tbar q (g) as a jet) against the oracle."""
    nf = len(BY_NAME[proc].masses)
    D = 4 * nf if mode == 0 else 3 * nf - 4
    go = ref.GridRef(D, VEGAS_BINS, VEGAS_ALPHA, seed=6, ps_mode=mode)
    gg = api.VegasGrid(D, VEGAS_BINS, VEGAS_ALPHA, 6, mode)
    so, fo = ref.MatrixElementRef(proc).vegas_integrand(go, 1000.0, 77, n, want_f=True)
    sg, fg = api.vegas_integrand(handles[proc], gg, 1000.0, 77, n, want_f=True)
    sg, fg = sg.cpu().numpy(), fg.cpu().numpy()
    assert np.array_equal(fg != 0, fo != 0)
    nz = fo != 0
    assert 0.05 < nz.mean() < 1.0
    assert np.max(np.abs(fg[nz] / fo[nz] - 1)) < ME_RTOL
    assert sg[2] == so[2]
    assert np.max(np.abs(sg - so) / (np.abs(so) + 1e-300 + 1e-12 * np.abs(so).max())) < 1e-9


@pytest.mark.parametrize("proc", ["qg_ttxqg", "qqx_ttxgg"])
def test_vegas_hadronic_mode_matches_oracle(handles, proc):
    """ps_mode 2 with the declared toy quark / antiquark / gluon density of each beam (DESIGN.md R-N3): the hadronic
    channels behind the paper's p p -> t tbar g g."""
    D, n = 3 * 4 - 2, 1500 + 3
    go = ref.GridRef(D, VEGAS_BINS, VEGAS_ALPHA, seed=10, ps_mode=2)
    gg = api.VegasGrid(D, VEGAS_BINS, VEGAS_ALPHA, 10, 2)
    so, fo = ref.MatrixElementRef(proc).vegas_integrand(go, 13000.0, 9, n, want_f=True)
    sg, fg = api.vegas_integrand(handles[proc], gg, 13000.0, 9, n, want_f=True)
    sg, fg = sg.cpu().numpy(), fg.cpu().numpy()
    assert np.array_equal(fg != 0, fo != 0)
    nz = fo != 0
    assert nz.sum() > 100
    assert np.max(np.abs(fg[nz] / fo[nz] - 1)) < ME_RTOL
    assert np.max(np.abs(sg - so) / (np.abs(so) + 1e-300 + 1e-12 * np.abs(so).max())) < 1e-9


def test_cuts_apply_to_the_final_light_quark():
    w = BY_NAME["qg_ttxqg"]
    mom = oracle_events("qg_ttxqg", 20000)
    want = ref.cuts(mom, w.is_gluon, PARAMS["ptj_min"], PARAMS["dr_min"])
    got = api.apply_cuts(dev(mom), w.is_gluon, PARAMS["ptj_min"], PARAMS["dr_min"]).cpu().numpy()
    assert np.array_equal(got, want)


def test_edge_kinematics(handles):
    """q qbar -> t tbar with the tops exactly along the beam axis (both orientations) and 1e-9 off it: the massless beam
    spinors and the massive top spinors in their degenerate branches; closed form as the second witness."""
    m, e = PARAMS["m_top"], 500.0
    pz = np.sqrt(e * e - m * m)
    mom = np.array([[[e, 0, 0, e], [e, 0, 0, -e], [e, 0, 0, -pz], [e, 0, 0, pz]],
                    [[e, 0, 0, e], [e, 0, 0, -e], [e, 0, 0, pz], [e, 0, 0, -pz]],
                    [[e, 0, 0, e], [e, 0, 0, -e], [e, pz * 1e-9, 0, -pz * np.sqrt(1 - 1e-18)], [e, -pz * 1e-9, 0, pz * np.sqrt(1 - 1e-18)]]])
    got = api.me_eval(handles["qqx_ttx"], dev(mom)).cpu().numpy()
    want = ref.MatrixElementRef("qqx_ttx").eval(mom)
    assert np.max(np.abs(got / want - 1)) < 1e-9
    s = 4 * e * e
    t = np.array([m * m - 2 * e * (e + pz), m * m - 2 * e * (e - pz), m * m - 2 * e * (e + pz)])   # (p_q - p_t)^2
    u = 2 * m * m - s - t
    closed = (4 * np.pi * PARAMS["alpha_s"]) ** 2 * (4.0 / 9) * (((m * m - t) / s) ** 2 + ((m * m - u) / s) ** 2 + 2 * m * m / s)
    assert np.max(np.abs(got / closed - 1)) < 1e-9
    assert api.me_eval(handles["qg_ttxqg"], torch.empty((0, 6, 4), dtype=torch.float64, device="cuda")).shape == (0,)
