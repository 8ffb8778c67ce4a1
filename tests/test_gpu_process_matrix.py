"""Every QCD process through every generic entry point (small sizes): per-helicity shares, the fused Vegas integrand in the
three phase-space modes, a Vegas iteration with refinement — against the oracle.  The per-process parity tests cover
me_eval at size; this matrix is for the combinations (process x mode) the others do not reach."""
import numpy as np
import pytest
import torch

from oracle import ref
from paper_2211_14056_b200 import api
from paper_2211_14056_b200.workloads import BY_NAME, PARAMS, VEGAS_ALPHA, VEGAS_BINS

pytestmark = pytest.mark.gpu
QCD = ["gg_ttx", "gg_ttxg", "gg_ttxgg", "gg_ttxggg", "qqx_ttx", "qqx_ttxg", "qqx_ttxgg", "qg_ttxq", "qg_ttxqg", "qxg_ttxqx", "qxg_ttxqxg"]
WL = {"gg_ttx": "config1", "gg_ttxg": "config2", "gg_ttxgg": "config3"}


def workload(proc):
    return BY_NAME[WL.get(proc, proc)]


@pytest.fixture(scope="module")
def both():
    return {p: (api.me_init(p, PARAMS), ref.MatrixElementRef(p)) for p in QCD}


@pytest.mark.parametrize("proc", QCD)
def test_per_helicity_shares(both, proc):
    h, o = both[proc]
    w = workload(proc)
    n = 6 if proc == "gg_ttxggg" else 64
    r = ref.philox_uniform(w.seed, 0, 40, w.n_dim, n)
    mom = ref.rambo_generate(r, w.sqrt_s, w.masses, w.ps_mode)[0]
    hel = api.me_eval_helicities(h, torch.from_numpy(mom).cuda()).cpu().numpy()
    assert hel.shape == (n, 1 << h.n_external)
    assert np.max(np.abs(hel.sum(1) / o.eval(mom) - 1)) < 1e-10
    assert np.array_equal(hel, hel[:, ::-1])          # |M(h)|^2 = |M(-h)|^2


@pytest.mark.parametrize("mode", [0, 1, 2])
@pytest.mark.parametrize("proc", QCD)
def test_vegas_integrand_every_mode(both, proc, mode):
    h, o = both[proc]
    nf = h.n_external - 2
    if mode == 1 and nf == 2:
        pytest.skip("RAMBO on diet needs three final particles for a free mass")
    D = {0: 4 * nf, 1: 3 * nf - 4, 2: 3 * nf - 2}[mode]
    rs = 13000.0 if mode == 2 else 1000.0
    n = 48 if proc == "gg_ttxggg" else 700 + 3
    go = ref.GridRef(D, VEGAS_BINS, VEGAS_ALPHA, seed=12, ps_mode=mode)
    gg = api.VegasGrid(D, VEGAS_BINS, VEGAS_ALPHA, 12, mode)
    so, fo = o.vegas_integrand(go, rs, 31, n, want_f=True)
    sg, fg = api.vegas_integrand(h, gg, rs, 31, n, want_f=True)
    sg, fg = sg.cpu().numpy(), fg.cpu().numpy()
    assert np.array_equal(fg != 0, fo != 0)
    nz = fo != 0
    if nz.any():
        assert np.max(np.abs(fg[nz] / fo[nz] - 1)) < 1e-10
    assert sg[2] == so[2]
    assert np.max(np.abs(sg - so) / (np.abs(so) + 1e-300 + 1e-12 * np.abs(so).max())) < 1e-9


@pytest.mark.parametrize("proc", ["qqx_ttxgg", "qg_ttxq", "gg_ttxggg"])
def test_vegas_iterate_with_refinement(both, proc):
    h, o = both[proc]
    nf = h.n_external - 2
    D = 3 * nf - 4
    n = 64 if proc == "gg_ttxggg" else 2000
    go = ref.GridRef(D, VEGAS_BINS, VEGAS_ALPHA, seed=14, ps_mode=1)
    gg = api.VegasGrid(D, VEGAS_BINS, VEGAS_ALPHA, 14, 1)
    for _ in range(2):
        ro = o.vegas_iterate(go, 1000.0, n)
        rg = api.vegas_iterate(h, gg, 1000.0, n)
        assert rg["n_pass"] == ro["n_pass"]
        assert abs(rg["integral"] / ro["integral"] - 1) < 1e-9
        assert abs(rg["variance"] / ro["variance"] - 1) < 1e-8
    assert np.max(np.abs(gg.edges.cpu().numpy() - go.edges)) < 1e-9
