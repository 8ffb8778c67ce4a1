"""Parity of the CUDA path (through the C ABI, paper_2211_14056_b200.api) with the oracle, element by element on the
same seeded inputs.  Inputs and expected values come from oracle/ only; nothing expected is produced by the CUDA path.

Tolerances: integer / bit work exact; fp64 |M|^2 1e-10 relative per event
(BASELINE.json:north_star); RAMBO momenta 1e-12 sqrt(s) absolute, weights 1e-11 relative.
"""
import numpy as np
import pytest
import torch

from oracle import ref
from paper_2211_14056_b200 import api
from paper_2211_14056_b200.workloads import BY_NAME, PARAMS, VEGAS_ALPHA, VEGAS_BINS
from tests.helpers import closed_form_epem_mupmum, closed_form_gg_ttx, momentum_violation, random_lorentz, transform

pytestmark = pytest.mark.gpu
ME_RTOL = 1e-10


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def oracle_events(cfg, n, first=0):
    w = BY_NAME[cfg]
    r = ref.philox_uniform(w.seed, 0, first, w.n_dim, n)
    mom, wt = ref.rambo_generate(r, w.sqrt_s, w.masses, w.ps_mode)
    return r, mom, wt


@pytest.fixture(scope="module")
def handles():
    return {p: api.me_init(p, PARAMS) for p in ("epem_mupmum", "gg_ttx", "gg_ttxg", "gg_ttxgg")}


def test_extension_is_loaded():
    import os
    maps = open("/proc/self/maps").read()
    api.lib()
    assert "libmadme.so" in open("/proc/self/maps").read() or "libmadme.so" in maps
    assert os.path.exists(api.LIB_PATH)


# ---- a1 Philox: bit exact -------------------------------------------------------------------------------------
@pytest.mark.parametrize("seed,it,first,nd,n", [(0, 0, 0, 8, 4099), (3, 2, 12345, 16, 1000), (0x0123456789ABCDEF, 7, (1 << 33) + 5, 5, 777),
                                                 (4, 1, 0, 1, 33), (1, 0, 0, 24, 64)])
def test_philox_bit_exact(seed, it, first, nd, n):
    got = api.philox_uniform(seed, it, first, nd, n).cpu().numpy()
    want = ref.philox_uniform(seed, it, first, nd, n)
    assert np.array_equal(got.view(np.uint64), want.view(np.uint64))


def test_philox_empty():
    assert api.philox_uniform(0, 0, 0, 8, 0).shape == (0, 8)


# ---- a3 RAMBO ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,mode", [("config0", 0), ("config1", 0), ("config2", 0), ("config3", 0), ("config3", 1), ("config2", 1)])
def test_rambo_matches_oracle(cfg, mode):
    w = BY_NAME[cfg]
    nf = len(w.masses)
    nd = 4 * nf if mode == 0 else 3 * nf - 4
    n = 5000 + 37
    r = ref.philox_uniform(w.seed, 0, 0, nd, n)
    mom_o, wt_o = ref.rambo_generate(r, w.sqrt_s, w.masses, mode)
    mom_g, wt_g = api.rambo_generate(dev(r), w.sqrt_s, w.masses, mode)
    mom_g, wt_g = mom_g.cpu().numpy(), wt_g.cpu().numpy()
    assert np.max(np.abs(mom_g - mom_o)) < 1e-12 * w.sqrt_s * 10
    assert np.max(np.abs(wt_g / wt_o - 1)) < 1e-11
    # properties that hold at any size: momentum conservation, on-shell masses
    tot = mom_g[:, 2:].sum(1)
    assert np.max(np.abs(tot - np.array([w.sqrt_s, 0, 0, 0]))) < 1e-10 * w.sqrt_s
    m2 = mom_g[:, 2:, 0] ** 2 - (mom_g[:, 2:, 1:] ** 2).sum(-1)
    assert np.max(np.abs(m2 - np.array(w.masses) ** 2)) < 1e-9 * w.sqrt_s ** 2


def test_rambo_six_body_and_empty():
    masses = (0.0, 10.0, 0.0, 5.0, 0.0, 1.0)
    r = ref.philox_uniform(9, 0, 0, 24, 300)
    mom_o, wt_o = ref.rambo_generate(r, 500.0, masses, 0)
    mom_g, wt_g = api.rambo_generate(dev(r), 500.0, masses, 0)
    assert np.max(np.abs(mom_g.cpu().numpy() - mom_o)) < 1e-9
    assert np.max(np.abs(wt_g.cpu().numpy() / wt_o - 1)) < 1e-11
    m, w = api.rambo_generate(torch.empty((0, 8), dtype=torch.float64, device="cuda"), 100.0, (0.0, 0.0), 0)
    assert m.shape == (0, 4, 4) and w.shape == (0,)


# ---- a4 cuts: the decision is an integer, taken in fp64 on both sides --------------------------------------------
@pytest.mark.parametrize("cfg", ["config2", "config3"])
def test_cuts_match_oracle(cfg):
    w = BY_NAME[cfg]
    _, mom, _ = oracle_events(cfg, 20000)
    want = ref.cuts(mom, w.is_gluon, PARAMS["ptj_min"], PARAMS["dr_min"])
    got = api.apply_cuts(dev(mom), w.is_gluon, PARAMS["ptj_min"], PARAMS["dr_min"]).cpu().numpy()
    diff = np.nonzero(got != want)[0]
    # a flip is only legitimate within rounding of a cut boundary; none is expected at this size
    assert len(diff) == 0, diff[:10]
    assert 0.05 < want.mean() < 0.999 and want.min() == 0


# ---- a5-a10 me_eval -----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,n", [("config0", 1 << 14), ("config1", 20000 + 13), ("config2", 6000 + 5), ("config3", 1500 + 7)])
def test_me_eval_matches_oracle(handles, cfg, n):
    """Element by element against tier 1 of the oracle; sizes span many CTAs and a ragged tail."""
    w = BY_NAME[cfg]
    _, mom, _ = oracle_events(cfg, n)
    want = ref.MatrixElementRef(w.process).eval(mom)
    got = api.me_eval(handles[w.process], dev(mom)).cpu().numpy()
    rel = np.abs(got / want - 1)
    assert momentum_violation(mom).max() < 1e-12
    assert np.max(rel) < ME_RTOL, (np.argmax(rel), np.max(rel))


def test_me_eval_closed_forms_full_size(handles):
    """configs[0] and configs[1] at FULL size against the closed forms (properties computable at any size)."""
    _, mom, _ = oracle_events("config0", 1 << 14)
    got = api.me_eval(handles["epem_mupmum"], dev(mom)).cpu().numpy()
    assert np.max(np.abs(got / closed_form_epem_mupmum(mom, PARAMS["alpha_em"]) - 1)) < ME_RTOL
    n = 1 << 20
    r = api.philox_uniform(1, 0, 0, 8, n)
    momg, _ = api.rambo_generate(r, 1000.0, (173.0, 173.0), 0)
    got = api.me_eval(handles["gg_ttx"], momg).cpu().numpy()
    momh = momg.cpu().numpy()
    cf = closed_form_gg_ttx(momh, PARAMS["alpha_s"], PARAMS["m_top"])
    assert momentum_violation(momh).max() < 1e-12
    assert np.max(np.abs(got / cf - 1)) < ME_RTOL


def test_me_eval_per_helicity_and_parity(handles):
    """Per-helicity shares sum to me2 and obey |M(h)|^2 = |M(-h)|^2 (QCD parity invariance)."""
    for cfg, n in (("config1", 257), ("config2", 129), ("config3", 65)):
        w = BY_NAME[cfg]
        _, mom, _ = oracle_events(cfg, n)
        h = handles[w.process]
        hel = api.me_eval_helicities(h, dev(mom)).cpu().numpy()
        tot = api.me_eval(h, dev(mom)).cpu().numpy()
        assert np.max(np.abs(hel.sum(1) / tot - 1)) < 1e-13
        nh = hel.shape[1]
        flipped = hel[:, (nh - 1) - np.arange(nh)]
        assert np.max(np.abs(hel - flipped) / tot[:, None]) < 1e-10


@pytest.mark.parametrize("cfg,n", [("config1", 4096), ("config2", 4096), ("config3", 4096)])
def test_me_eval_lorentz_invariance(handles, cfg, n):
    """A property that needs no oracle: |M|^2 is invariant under a common rotation + boost of all momenta (the kernels
    rebuild every wavefunction in the new frame: incoming legs off the z axis, different helicity spinors)."""
    w = BY_NAME[cfg]
    _, mom, _ = oracle_events(cfg, n)
    h = handles[w.process]
    base = api.me_eval(h, dev(mom)).cpu().numpy()
    rng = np.random.default_rng(11)
    for _ in range(3):
        L = random_lorentz(rng, beta_max=0.8)
        got = api.me_eval(h, dev(transform(mom, L))).cpu().numpy()
        assert np.max(np.abs(got / base - 1)) < 1e-9  # boosted components are up to 3x larger: a few more ulps cancel


def test_me_eval_edge_cases(handles):
    h = handles["gg_ttx"]
    assert api.me_eval(h, torch.empty((0, 4, 4), dtype=torch.float64, device="cuda")).shape == (0,)
    # degenerate kinematics of the wavefunctions: a top exactly along -z, and at rest-frame threshold-ish
    m, e = 173.0, 500.0
    pz = np.sqrt(e * e - m * m)
    mom = np.array([[[e, 0, 0, e], [e, 0, 0, -e], [e, 0, 0, -pz], [e, 0, 0, pz]],
                    [[e, 0, 0, e], [e, 0, 0, -e], [e, 0, 0, pz], [e, 0, 0, -pz]],
                    [[e, 0, 0, e], [e, 0, 0, -e], [e, pz * 1e-9, 0, -pz * np.sqrt(1 - 1e-18)], [e, -pz * 1e-9, 0, pz * np.sqrt(1 - 1e-18)]]])
    got = api.me_eval(h, dev(mom)).cpu().numpy()
    want = ref.MatrixElementRef("gg_ttx").eval(mom)
    assert np.max(np.abs(got / want - 1)) < 1e-9
    with pytest.raises(ValueError):
        api.me_eval(h, torch.zeros((4, 5, 4), dtype=torch.float64, device="cuda"))
    with pytest.raises(TypeError):
        api.me_eval(h, torch.zeros((4, 4, 4), dtype=torch.float32, device="cuda"))


@pytest.mark.parametrize("n", [1, 7, 8, 9, 255, 257])
def test_tiny_and_ragged_batches(handles, n):
    """Batches smaller than one CTA (8 events) and ragged tails: the CTA-cooperative kernels recompute a valid event in
    the idle slots and must neither store it nor disturb the live ones."""
    _, mom, _ = oracle_events("config3", n)
    want = ref.MatrixElementRef("gg_ttxgg").eval(mom)
    guard = torch.full((n + 8,), -7.0, dtype=torch.float64, device="cuda")
    api.me_eval(handles["gg_ttxgg"], dev(mom), guard[:n])
    got = guard.cpu().numpy()
    assert np.max(np.abs(got[:n] / want - 1)) < ME_RTOL and np.all(got[n:] == -7.0)
    g_o = ref.GridRef(8, VEGAS_BINS, VEGAS_ALPHA, seed=4, ps_mode=1)
    g_g = api.VegasGrid(8, VEGAS_BINS, VEGAS_ALPHA, 4, 1)
    first = (1 << 33) + 11  # event indices beyond 32 bits reach Philox counter word 1
    so, fo = ref.MatrixElementRef("gg_ttxgg").vegas_integrand(g_o, 1000.0, first, n, want_f=True)
    sg, fg = api.vegas_integrand(handles["gg_ttxgg"], g_g, 1000.0, first, n, want_f=True)
    fg = fg.cpu().numpy()
    assert np.array_equal(fg != 0, fo != 0)
    nz = fo != 0
    assert nz.sum() == 0 or np.max(np.abs(fg[nz] / fo[nz] - 1)) < ME_RTOL
    assert sg.cpu().numpy()[2] == so[2]


def test_me_eval_sampled_at_bench_size(handles):
    """configs[3] in the launch configuration bench.py times (full persistent grid): sampled events against the oracle."""
    n = BY_NAME["config3"].n_events  # 2^24: BASELINE.json:configs[3] at full size
    r = api.philox_uniform(3, 0, 0, 16, n)
    mom, _ = api.rambo_generate(r, 1000.0, (173.0, 173.0, 0.0, 0.0), 0)
    got = api.me_eval(handles["gg_ttxgg"], mom).cpu().numpy()
    assert np.all(np.isfinite(got)) and np.all(got > 0)
    idx = np.concatenate([np.arange(0, n, n // 8192), [n - 1]])
    # oracle inputs from the ORACLE's own generators for the same event indices
    ro = np.concatenate([ref.philox_uniform(3, 0, int(i), 16, 1) for i in idx])
    momo, _ = ref.rambo_generate(ro, 1000.0, (173.0, 173.0, 0.0, 0.0), 0)
    me = ref.MatrixElementRef("gg_ttxgg")
    want = me.eval(momo)
    assert np.max(np.abs(got[idx] / want - 1)) < ME_RTOL
    # the events where rounding is at risk are the soft ones (individual diagrams >> their gauge-
    # cancelling sum): the 64 events of the whole 2^24 sample with the softest gluon, against the oracle
    soft = torch.topk(-torch.minimum(mom[:, 4, 0], mom[:, 5, 0]), 64).indices.cpu().numpy()
    ro = np.concatenate([ref.philox_uniform(3, 0, int(i), 16, 1) for i in soft])
    momo, _ = ref.rambo_generate(ro, 1000.0, (173.0, 173.0, 0.0, 0.0), 0)
    assert momo[:, 4:, 0].min() < 0.2  # GeV: these really are soft
    assert np.max(np.abs(got[soft] / me.eval(momo) - 1)) < ME_RTOL
    # properties that hold at any size: Bose symmetry under the exchange of the two final gluons (a different
    # evaluation order inside the kernel: legs 4 and 5 swap roles in every leg split)
    sub = mom[: 1 << 16].clone()
    sub[:, [4, 5]] = sub[:, [5, 4]]
    swapped = api.me_eval(handles["gg_ttxgg"], sub.contiguous()).cpu().numpy()
    assert np.max(np.abs(swapped / got[: 1 << 16] - 1)) < ME_RTOL


def test_vegas_full_size_config4(handles):
    """configs[4] at full size (5 iterations x 2^24 events, D = 8, 50 bins) in the launch configuration bench.py times:
    sampled per-event weights of iteration 0 against the oracle, the iteration results against each other."""
    w = BY_NAME["config4"]
    n = w.n_events
    h = handles["gg_ttxgg"]
    g = api.VegasGrid(8, VEGAS_BINS, VEGAS_ALPHA, w.seed, 1)
    sums, f = api.vegas_integrand(h, g, w.sqrt_s, 0, n, want_f=True)
    f = f.cpu().numpy()
    idx = np.concatenate([np.arange(0, n, n // 61), [n - 1]])
    go = ref.GridRef(8, VEGAS_BINS, VEGAS_ALPHA, seed=w.seed, ps_mode=1)
    me = ref.MatrixElementRef("gg_ttxgg")
    want = np.array([me.vegas_integrand(go, w.sqrt_s, int(i), 1, want_f=True)[1][0] for i in idx])
    assert np.array_equal(f[idx] != 0, want != 0)
    nz = want != 0
    assert np.max(np.abs(f[idx][nz] / want[nz] - 1)) < ME_RTOL
    s = sums.cpu().numpy()
    assert abs(s[0] / f.sum() - 1) < 1e-12 and s[2] == np.count_nonzero(f)
    res = [api.vegas_iterate(h, g, w.sqrt_s, n) for _ in range(5)]
    I = np.array([r["integral"] for r in res])
    sig = np.sqrt(np.array([r["variance"] for r in res]))
    assert np.all(np.isfinite(I)) and np.all(sig > 0) and g.iteration == 5
    wgt = 1 / sig ** 2
    mean = (I * wgt).sum() / wgt.sum()
    chi2 = (((I - mean) / sig) ** 2).sum() / 4
    assert chi2 < 10 and sig[-1] < sig[0]  # consistent iterations; the adapted grid reduces the error
    e = g.edges.cpu().numpy()
    assert np.all(e[:, 0] == 0) and np.all(e[:, -1] == 1) and np.all(np.diff(e, axis=1) > 0)


# ---- a2, a11, a12 Vegas pieces ----------------------------------------------------------------------------------
def _warped_grid(D, nb, seed):
    rng = np.random.default_rng(seed)
    e = np.sort(rng.uniform(size=(D, nb + 1)), axis=1)
    e[:, 0], e[:, -1] = 0.0, 1.0
    return e


def test_vegas_map_matches_oracle():
    e = _warped_grid(8, 50, 0)
    y = ref.philox_uniform(11, 0, 0, 8, 3001)
    y[0, 0] = np.nextafter(1.0, 0.0)
    xo, jo, io = ref.vegas_map(e, y)
    xg, jg, ig = api.vegas_map(dev(e), dev(y))
    assert np.array_equal(ig.cpu().numpy(), io)
    assert np.max(np.abs(xg.cpu().numpy() - xo)) < 1e-15
    assert np.max(np.abs(jg.cpu().numpy() / jo - 1)) < 1e-13


@pytest.mark.parametrize("alpha", [0.0, 0.5, 1.5])
def test_vegas_refine_matches_oracle(alpha):
    rng = np.random.default_rng(5)
    e = _warped_grid(8, 50, 1)
    S = rng.uniform(size=(8, 50)) ** 4
    S[3, 10:20] = 0.0
    S[5] = 0.0
    want = ref.vegas_refine(e, S, alpha)
    got = api.vegas_refine(dev(e), dev(S), alpha).cpu().numpy()
    assert np.max(np.abs(got - want)) < 1e-13
    assert np.all(got[:, 0] == 0) and np.all(got[:, -1] == 1) and np.all(np.diff(got, axis=1) >= 0)


@pytest.mark.parametrize("proc,mode,n", [("gg_ttx", 0, 4000 + 9), ("gg_ttxg", 1, 3000 + 1), ("gg_ttxgg", 1, 1200 + 3), ("gg_ttxgg", 0, 400)])
def test_vegas_integrand_matches_oracle(handles, proc, mode, n):
    """Fused a1-a11 against the oracle on the same Philox stream: per-event f, sums, histogram."""
    nf = {"gg_ttx": 2, "gg_ttxg": 3, "gg_ttxgg": 4}[proc]
    D = 4 * nf if mode == 0 else 3 * nf - 4
    e = _warped_grid(D, VEGAS_BINS, 2)
    go = ref.GridRef(D, VEGAS_BINS, VEGAS_ALPHA, seed=4, ps_mode=mode)
    go.edges[:] = e
    go.c.iteration = 2
    gg = api.VegasGrid(D, VEGAS_BINS, VEGAS_ALPHA, 4, mode, edges=dev(e))
    gg.iteration = 2
    first = 1000
    so, fo = ref.MatrixElementRef(proc).vegas_integrand(go, 1000.0, first, n, want_f=True)
    sg, fg = api.vegas_integrand(handles[proc], gg, 1000.0, first, n, want_f=True)
    sg, fg = sg.cpu().numpy(), fg.cpu().numpy()
    assert np.array_equal(fg != 0, fo != 0)
    nz = fo != 0
    assert np.max(np.abs(fg[nz] / fo[nz] - 1)) < ME_RTOL
    assert sg[2] == so[2]
    assert np.max(np.abs(sg - so) / (np.abs(so) + 1e-300 + 1e-12 * np.abs(so).max())) < 1e-9


@pytest.mark.parametrize("proc,n", [("gg_ttxgg", 1500 + 5), ("gg_ttxg", 2000 + 3)])
def test_vegas_hadronic_mode_matches_oracle(handles, proc, n):
    """ps_mode 2 (the literal 10-dimensional configs[4]: momentum fractions + RAMBO on diet, declared toy gluon density;
    SURVEY §8(f) N3, DESIGN.md R-N3): per-event f, sums and two iterations with feedback against the oracle."""
    nf = {"gg_ttxg": 3, "gg_ttxgg": 4}[proc]
    D, S = 3 * nf - 2, 13000.0
    e = _warped_grid(D, VEGAS_BINS, 7)
    go = ref.GridRef(D, VEGAS_BINS, VEGAS_ALPHA, seed=5, ps_mode=2)
    go.edges[:] = e
    gg = api.VegasGrid(D, VEGAS_BINS, VEGAS_ALPHA, 5, 2, edges=dev(e))
    me = ref.MatrixElementRef(proc)
    so, fo = me.vegas_integrand(go, S, 77, n, want_f=True)
    sg, fg = api.vegas_integrand(handles[proc], gg, S, 77, n, want_f=True)
    sg, fg = sg.cpu().numpy(), fg.cpu().numpy()
    assert np.array_equal(fg != 0, fo != 0) and (fo == 0).any()
    nz = fo != 0
    assert np.max(np.abs(fg[nz] / fo[nz] - 1)) < ME_RTOL
    assert sg[2] == so[2] and abs(sg[0] / so[0] - 1) < 1e-10
    for it in range(2):
        ro = me.vegas_iterate(go, S, n)
        rg = api.vegas_iterate(handles[proc], gg, S, n)
        assert rg["n_pass"] == ro["n_pass"] and abs(rg["integral"] / ro["integral"] - 1) < 1e-9
        assert np.max(np.abs(gg.edges.cpu().numpy() - go.edges)) < 1e-9
    with pytest.raises(api.MadmeError):
        api.vegas_integrand(handles[proc], api.VegasGrid(D + 1, VEGAS_BINS, VEGAS_ALPHA, 5, 2), S, 0, 10)


def test_vegas_iterate_matches_oracle(handles):
    """Three full iterations (integrand + refinement feedback) of config 4 at a size the oracle finishes in seconds."""
    n = 6000
    go = ref.GridRef(8, VEGAS_BINS, VEGAS_ALPHA, seed=4, ps_mode=1)
    gg = api.VegasGrid(8, VEGAS_BINS, VEGAS_ALPHA, 4, 1)
    me = ref.MatrixElementRef("gg_ttxgg")
    for it in range(3):
        ro = me.vegas_iterate(go, 1000.0, n)
        rg = api.vegas_iterate(handles["gg_ttxgg"], gg, 1000.0, n)
        assert rg["n_pass"] == ro["n_pass"]
        assert abs(rg["integral"] / ro["integral"] - 1) < 1e-9
        assert abs(rg["variance"] / ro["variance"] - 1) < 1e-8
        assert np.max(np.abs(gg.edges.cpu().numpy() - go.edges)) < 1e-9
        assert gg.iteration == go.iteration == it + 1


def test_vegas_two_phase_space_maps_agree(handles):
    """The integral must not depend on how the unit cube is mapped onto phase space: D = 8 (RAMBO on diet) and D = 16
    (classic RAMBO) agree within the Monte-Carlo error (the only pin of the value of sigma)."""
    def run(D, mode):
        g = api.VegasGrid(D, VEGAS_BINS, VEGAS_ALPHA, 4, mode)
        res = [api.vegas_iterate(handles["gg_ttxgg"], g, 1000.0, 1 << 20) for _ in range(3)]
        I = np.array([r["integral"] for r in res])
        w = 1.0 / np.array([r["variance"] for r in res])
        return (I * w).sum() / w.sum(), w.sum() ** -0.5
    a, ea = run(8, 1)
    b, eb = run(16, 0)
    assert abs(a - b) < 5 * np.hypot(ea, eb) and ea / a < 0.01 and eb / b < 0.01


def test_vegas_is_deterministic(handles):
    """Fixed-shape reduction: two runs give bit-identical sums."""
    res = []
    for _ in range(2):
        g = api.VegasGrid(8, VEGAS_BINS, VEGAS_ALPHA, 4, 1)
        s, _ = api.vegas_integrand(handles["gg_ttxgg"], g, 1000.0, 0, 5000)
        res.append(s.cpu().numpy())
    assert np.array_equal(res[0], res[1])
