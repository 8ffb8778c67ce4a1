"""vegas_iterate_sharded: two ranks (two processes sharing cuda:0, gloo for the 3.2 KB exchange — their kernels never
wait on one another) reproduce the single-process vegas_iterate: same integrals, same refined grids."""
import os

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu


def _worker(rank, world, port, n_total, n_iter, q):
    import torch.distributed as dist
    from paper_2211_14056_b200 import api
    from paper_2211_14056_b200.workloads import PARAMS, VEGAS_ALPHA, VEGAS_BINS
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    h = api.me_init("gg_ttxgg", PARAMS)
    g = api.VegasGrid(8, VEGAS_BINS, VEGAS_ALPHA, 4, 1)
    res = [api.vegas_iterate_sharded(h, g, 1000.0, n_total) for _ in range(n_iter)]
    torch.cuda.synchronize()
    q.put((rank, res, g.edges.cpu().numpy()))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_match_one():
    from paper_2211_14056_b200 import api
    from paper_2211_14056_b200.workloads import PARAMS, VEGAS_ALPHA, VEGAS_BINS
    n_total, n_iter = 30001, 3
    h = api.me_init("gg_ttxgg", PARAMS)
    g = api.VegasGrid(8, VEGAS_BINS, VEGAS_ALPHA, 4, 1)
    want = [api.vegas_iterate(h, g, 1000.0, n_total) for _ in range(n_iter)]
    # world size 1 (no process group): the sharded call is the plain one
    g1 = api.VegasGrid(8, VEGAS_BINS, VEGAS_ALPHA, 4, 1)
    one = [api.vegas_iterate_sharded(h, g1, 1000.0, n_total) for _ in range(n_iter)]
    for a, b in zip(one, want):
        assert a["n_pass"] == b["n_pass"] and abs(a["integral"] / b["integral"] - 1) < 1e-12
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, 29671, n_total, n_iter, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted([q.get(timeout=300) for _ in range(2)], key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, r0, e0), (_, r1, e1) = got
    assert np.array_equal(e0, e1)  # bit-identical grids on both ranks
    for a, b, c in zip(r0, r1, want):
        assert a == b
        assert a["n_pass"] == c["n_pass"]
        assert abs(a["integral"] / c["integral"] - 1) < 1e-11 and abs(a["variance"] / c["variance"] - 1) < 1e-9
    assert np.max(np.abs(e0 - g.edges.cpu().numpy())) < 1e-10
