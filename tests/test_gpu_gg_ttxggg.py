"""GPU parity of g g -> t tbar g g g: 1 240 diagrams, 120 colour flows — the
colour-flow vector lives in tensor memory and is processed in chunks, the event is evaluated in two passes over the
helicity of the last gluon (me_kernel.cuh::cta_me2_chunked).  Per event at 1e-10 against the oracle's tier 1."""
import numpy as np
import pytest
import torch

from oracle import ref
from paper_2211_14056_b200 import api
from paper_2211_14056_b200.workloads import BY_NAME, PARAMS, VEGAS_ALPHA, VEGAS_BINS
from tests.helpers import momentum_violation

pytestmark = pytest.mark.gpu
ME_RTOL = 1e-10
W = BY_NAME["gg_ttxggg"]


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def oracle_events(n, first=0):
    r = ref.philox_uniform(W.seed, 0, first, W.n_dim, n)
    return ref.rambo_generate(r, W.sqrt_s, W.masses, W.ps_mode)[0]


@pytest.fixture(scope="module")
def handle():
    return api.me_init("gg_ttxggg", PARAMS)


@pytest.fixture(scope="module")
def oracle():
    return ref.MatrixElementRef("gg_ttxggg")


def test_info(handle):
    assert api.me_info(handle, 0) == 1240 and api.me_info(handle, 2) == 295 and api.me_info(handle, 3) == 120
    assert api.me_info(handle, 1) == 1890


@pytest.mark.parametrize("n", [1, 3, 4, 5, 197])
def test_me_eval_matches_oracle(handle, oracle, n):
    """Element by element: ragged batches around the 4 events of a CTA, and a size that spans many CTAs."""
    mom = oracle_events(n, first=1000 * n)
    want = oracle.eval(mom)
    out = torch.full((n + 4,), -7.0, dtype=torch.float64, device="cuda")
    api.me_eval(handle, dev(mom), me2=out[:n])
    got = out.cpu().numpy()
    assert np.all(got[n:] == -7.0)
    assert momentum_violation(mom).max() < 1e-12
    rel = np.abs(got[:n] / want - 1)
    assert np.max(rel) < ME_RTOL, (np.argmax(rel), np.max(rel))


def test_per_helicity_shares(handle, oracle):
    """The 128 helicity shares (two passes x 32 lanes x parity) sum to me2 and obey |M(h)|^2 = |M(-h)|^2."""
    mom = oracle_events(8, first=77)
    hel = api.me_eval_helicities(handle, dev(mom)).cpu().numpy()
    assert hel.shape == (8, 128)
    assert np.max(np.abs(hel.sum(1) / oracle.eval(mom) - 1)) < ME_RTOL
    flipped = hel[:, ::-1]
    assert np.array_equal(hel, flipped)
    assert (hel > 0).sum() > 64 * 8


def test_sampled_at_full_size(handle, oracle):
    """The workload's 2^20 events on the GPU; 256 of them, equally spaced, against the oracle."""
    r = api.philox_uniform(W.seed, 0, 0, W.n_dim, W.n_events)
    momg, _ = api.rambo_generate(r, W.sqrt_s, W.masses, 0)
    got = api.me_eval(handle, momg)
    assert bool(torch.isfinite(got).all()) and bool((got > 0).all())
    idx = np.arange(0, W.n_events, W.n_events // 256)
    mom = momg[torch.from_numpy(idx).cuda()].cpu().numpy()
    want = oracle.eval(mom)
    rel = np.abs(got.cpu().numpy()[idx] / want - 1)
    cut = ref.cuts(mom, W.is_gluon, PARAMS["ptj_min"], PARAMS["dr_min"]) != 0
    assert np.max(rel[cut]) < ME_RTOL, np.max(rel[cut])
    assert np.max(rel) < 1e-8    # cut-failing events (weight 0): soft / collinear cancellations, DESIGN.md §7


def test_vegas_integrand_matches_oracle(handle, oracle):
    D = 3 * 5 - 4
    go = ref.GridRef(D, VEGAS_BINS, VEGAS_ALPHA, seed=8, ps_mode=1)
    gg = api.VegasGrid(D, VEGAS_BINS, VEGAS_ALPHA, 8, 1)
    n = 301
    so, fo = oracle.vegas_integrand(go, 1000.0, 5, n, want_f=True)
    sg, fg = api.vegas_integrand(handle, gg, 1000.0, 5, n, want_f=True)
    sg, fg = sg.cpu().numpy(), fg.cpu().numpy()
    assert np.array_equal(fg != 0, fo != 0)
    nz = fo != 0
    assert 0.05 < nz.mean() < 1.0
    assert np.max(np.abs(fg[nz] / fo[nz] - 1)) < ME_RTOL
    assert sg[2] == so[2]
    assert np.max(np.abs(sg - so) / (np.abs(so) + 1e-300 + 1e-12 * np.abs(so).max())) < 1e-9
