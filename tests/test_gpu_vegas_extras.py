"""GPU parity of the calls around vegas_iterate that round 2 added to the C ABI: me_reserve (no allocation inside calls),
vegas_combine / vegas_finish (the sharded iteration's arithmetic behind the boundary), and unweighted-event extraction
(vegas_max_weight, vegas_unweight, vegas_generate).  Expected values come from oracle/ only."""
import ctypes as C

import numpy as np
import pytest
import torch

from oracle import ref
from paper_2211_14056_b200 import api
from paper_2211_14056_b200.workloads import BY_NAME, PARAMS

pytestmark = pytest.mark.gpu


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def random_grid(n_dim, seed):
    rng = np.random.default_rng(seed)
    e = np.sort(rng.uniform(size=(n_dim, 51)), axis=1)
    e[:, 0], e[:, -1] = 0.0, 1.0
    return e


def test_reserve_then_no_call_allocates():
    h = api.me_init("gg_ttxg", PARAMS)
    g = api.VegasGrid(5, 50, 1.5, 4, 1)
    # the raw C call refuses a batch beyond the reserved scratch instead of allocating
    sums = torch.empty(3 + 5 * 50, dtype=torch.float64, device="cuda")
    rc = api.lib().vegas_integrand(h.ptr, C.byref(g.c), 1000.0, 0, 1000, C.c_void_p(sums.data_ptr()), None, None)
    assert rc == api.ME_EINVAL and b"me_reserve" in api.lib().me_last_error()
    api.me_reserve(h, 50000)
    assert api.me_info(h, 11) == 50000
    ptr = api.me_info(h, 13)
    assert ptr != 0
    api.vegas_iterate(h, g, 1000.0, 64)                    # first launch: the CUDA runtime loads the kernels (its own memory)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for n in (100, 5000, 50000, 777):
        api.vegas_iterate(h, g, 1000.0, n)
        assert api.me_info(h, 13) == ptr and api.me_info(h, 11) == 50000
    assert torch.cuda.mem_get_info()[0] == free0          # nothing was allocated or freed on the device
    api.me_reserve(h, 10)                                  # smaller: a no-op
    assert api.me_info(h, 13) == ptr
    assert api.me_info(h, 12) == torch.cuda.current_device()


def test_combine_and_finish_match_the_oracle():
    """Two shards of one iteration: per-shard sums from the fused kernel, vegas_combine in rank order, vegas_finish;
    against the oracle's sums and its by-hand result on the same events."""
    h = api.me_init("gg_ttxg", PARAMS)
    edges = random_grid(5, 3)
    n = 3001
    g = api.VegasGrid(5, 50, 1.5, 9, 1, edges=dev(edges))
    g.iteration = 2
    s1, _ = api.vegas_integrand(h, g, 1000.0, 0, 1500)
    s2, _ = api.vegas_integrand(h, g, 1000.0, 1500, n - 1500)
    tot = api.vegas_combine(torch.stack([s1, s2]).contiguous())
    assert torch.equal(tot, s1 + s2)                       # two terms: any order gives the same bits
    res = api.vegas_finish(tot, n)
    me = ref.MatrixElementRef("gg_ttxg")
    go = ref.GridRef(5, 50, 1.5, seed=9, ps_mode=1)
    go.edges[:] = edges
    go.c.iteration = 2
    want, f = me.vegas_integrand(go, 1000.0, 0, n, want_f=True)
    got = tot.cpu().numpy()
    assert got[2] == want[2]
    assert np.max(np.abs(got - want) / (np.abs(want) + 1e-300)) < 1e-9
    I = f.sum() / n
    assert abs(res["integral"] / I - 1) < 1e-9 and res["n_pass"] == int(want[2])
    assert abs(res["variance"] / (((f * f).sum() / n - I * I) / (n - 1)) - 1) < 1e-8
    # three parts, fixed order
    parts = torch.stack([s1, s2, s1]).contiguous()
    assert torch.equal(api.vegas_combine(parts), (s1 + s2) + s1)


def test_unweight_matches_oracle_bit_exact():
    """The same weights on both sides: the accepted lists must be identical (integer work: bit exact)."""
    h = api.me_init("gg_ttxgg", PARAMS)
    rng = np.random.default_rng(11)
    for n, first in ((0, 0), (1, 5), (255, 0), (256, 7), (70001, (1 << 33) + 3)):
        f = rng.exponential(2.0, n) * (rng.uniform(size=n) < 0.7)
        w_max = 9.0
        want, over = ref.vegas_unweight(f, w_max, seed=4, iteration=6, first_event=first)
        got, n_over = api.vegas_unweight(h, dev(f), w_max, 4, 6, first)
        assert np.array_equal(got.cpu().numpy(), want) and n_over == over
    f = dev(rng.exponential(1.0, 4097))
    assert float(api.vegas_max_weight(f)[0]) == float(f.max())
    assert float(api.vegas_max_weight(torch.zeros(0, dtype=torch.float64, device="cuda"))[0]) == 0.0


@pytest.mark.parametrize("cfg,ps_mode,n_dim,sqrt_s", [("config4", 1, 8, 1000.0), ("config3", 0, 16, 1000.0), ("config4_hadronic", 2, 10, 13000.0),
                                                      ("gg_ttxggg", 1, 11, 1000.0), ("qg_ttxqg", 2, 10, 13000.0)])
def test_generate_matches_oracle(cfg, ps_mode, n_dim, sqrt_s):
    proc = BY_NAME[cfg].process
    h = api.me_init(proc, PARAMS)
    edges = random_grid(n_dim, 21)
    g = api.VegasGrid(n_dim, 50, 1.5, 4, ps_mode, edges=dev(edges))
    g.iteration = 1
    ids = np.array([0, 5, 3, 99999, (1 << 34) + 1, 17], dtype=np.int64)
    ids = np.concatenate([ids, np.arange(1000, 1400, dtype=np.int64)])
    mom, w = api.vegas_generate(h, g, sqrt_s, dev(ids))
    go = ref.GridRef(n_dim, 50, 1.5, seed=4, ps_mode=ps_mode)
    go.edges[:] = edges
    go.c.iteration = 1
    mom_o, w_o = ref.MatrixElementRef(proc).vegas_generate(go, sqrt_s, ids)
    scale = np.maximum(mom_o[:, 0, 0] * 2, 1.0)[:, None, None]
    assert np.max(np.abs(mom.cpu().numpy() - mom_o) / scale) < 1e-11
    nz = w_o != 0
    assert np.array_equal(w.cpu().numpy() != 0, nz)
    assert np.max(np.abs(w.cpu().numpy()[nz] / w_o[nz] - 1)) < 1e-10


@pytest.mark.parametrize("cfg,D,n", [("config4", 8, 1 << 17), ("qg_ttxqg", 8, 1 << 17), ("gg_ttxggg", 11, 1 << 13)])
def test_unweighted_events_end_to_end(cfg, D, n):
    """integrand -> max weight -> hit-or-miss -> kinematics of the kept events: for every kept event the regenerated
    momenta pass the cuts and weight x |M|^2 reproduces its integrand value; the kept fraction is <f>/w_max within
    its binomial error; the oracle keeps the same events when given the GPU's weights.  Also for a quark-initiated channel
    (the final light quark is a jet) and for g g -> t tbar g g g."""
    w = BY_NAME[cfg]
    h = api.me_init(w.process, PARAMS)
    g = api.VegasGrid(D, 50, 1.5, w.seed, 1)
    api.vegas_iterate(h, g, w.sqrt_s, n)                       # one adaptation step, then unweight iteration 1
    _, f = api.vegas_integrand(h, g, w.sqrt_s, 0, n, want_f=True)
    w_max = float(api.vegas_max_weight(f)[0])
    ids, n_over = api.vegas_unweight(h, f, w_max, w.seed, g.iteration, 0)
    assert n_over == 0 and len(ids) > (100 if n > 10000 else 5)
    fh = f.cpu().numpy()
    want, _ = ref.vegas_unweight(fh, w_max, w.seed, g.iteration, 0)
    assert np.array_equal(ids.cpu().numpy(), want)
    p = fh / w_max
    assert abs(len(ids) - p.sum()) < 5 * np.sqrt((p * (1 - p)).sum())
    mom, wgt = api.vegas_generate(h, g, w.sqrt_s, ids)
    ok = api.apply_cuts(mom, w.is_gluon, PARAMS["ptj_min"], PARAMS["dr_min"])
    assert bool(ok.all())
    me2 = api.me_eval(h, mom)
    assert float(((wgt * me2) / f[ids] - 1).abs().max()) < 1e-10
