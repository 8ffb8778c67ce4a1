"""vegas_unweight_static — the unweighting entry point that allocates nothing (its scratch is a file-scope device array,
csrc/unweight_static.cu) — against the existing path vegas_unweight on the same weights: the accepted event lists and the
counters must be IDENTICAL (integer work: bit-exact), on two calls in a row that share the scratch.
Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

from paper_2211_14056_b200 import api
from paper_2211_14056_b200.workloads import BY_NAME, PARAMS

pytestmark = pytest.mark.gpu


def _weights(h, w, n, iteration, first):
    g = api.VegasGrid(w.n_dim, 50, 1.5, w.seed, w.ps_mode)
    g.iteration = iteration
    _, f = api.vegas_integrand(h, g, w.sqrt_s, first, n, want_f=True)
    return f.clone()


def test_static_unweight_equals_the_existing_path_on_two_calls_in_a_row():
    w = BY_NAME["config4"]
    h = api.me_init(w.process, PARAMS)
    api.vegas_unweight_static_init()
    # set-up: the first launch of a kernel loads its code onto the device (CUDA loads modules lazily); do that before
    # free memory is compared around a call
    api.vegas_unweight_static(torch.ones(8, dtype=torch.float64, device="cuda"), 2.0, 1, 0)
    # the second call is SMALLER and has other weights: the scratch still holds the first call's counters beyond its range
    calls = [((1 << 17) + 5, 0, 0), (1000 + 3, 3, 777)]
    for n, iteration, first in calls:
        f = _weights(h, w, n, iteration, first)
        w_max = 0.25 * float(api.vegas_max_weight(f)[0])          # some events lie above w_max: the second counter moves too
        want_ids, want_over = api.vegas_unweight(h, f, w_max, w.seed, iteration, first)
        accepted = torch.full((n,), -1, dtype=torch.int64, device="cuda")
        counts = torch.full((2,), -1, dtype=torch.int64, device="cuda")
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        api.vegas_unweight_static(f, w_max, w.seed, iteration, first, accepted=accepted, counts=counts)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before       # the call allocated and freed nothing on the device
        c = counts.tolist()
        assert c[0] == len(want_ids) and c[1] == want_over and c[0] > 10 and c[1] > 0
        assert torch.equal(accepted[:c[0]], want_ids)
        assert bool((accepted[c[0]:] == -1).all())               # nothing written past the kept events
        ids = accepted[:c[0]].cpu().numpy()
        assert np.all(np.diff(ids) > 0) and ids[0] >= first and ids[-1] < first + n
    # the convenience form of the binding (allocates its outputs itself) gives the same
    got_ids, got_over = api.vegas_unweight_static(f, w_max, w.seed, iteration, first)
    assert torch.equal(got_ids, want_ids) and got_over == want_over


def test_static_unweight_limits_and_empty_input():
    f = torch.ones(api.UNWEIGHT_STATIC_MAX_EVENTS + 1, dtype=torch.float64, device="cuda")
    with pytest.raises(api.MadmeError) as e:
        api.vegas_unweight_static(f, 2.0, 1, 0)
    assert "VEGAS_UNWEIGHT_STATIC_MAX_EVENTS" in str(e.value)
    # exactly the maximum is accepted; all weights equal w_max / 2: about half are kept, none is overweight
    ids, over = api.vegas_unweight_static(f[:-1], 2.0, 1, 0)
    n = api.UNWEIGHT_STATIC_MAX_EVENTS
    assert over == 0 and abs(len(ids) - n / 2) < 5 * (n / 4) ** 0.5
    ids, over = api.vegas_unweight_static(f[:0], 2.0, 1, 0)
    assert len(ids) == 0 and over == 0
    with pytest.raises(api.MadmeError):
        api.vegas_unweight_static(f[:8], 0.0, 1, 0)
