"""The N > 1 path on CPU (gloo, world_size 2): event-range sharding reproduces the single-process stream, the fixed-order
combination of per-shard Vegas sums equals the unsharded sums, max-over-ranks timing, and the reference arm prints one line."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2211_14056_b200.sharding import strong_shard, weak_shard

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_shard_ranges_tile_the_index_space():
    for world in (1, 2, 3, 8):
        for total in (0, 1, 7, 64, 1000):
            spans = [strong_shard(r, world, total) for r in range(world)]
            assert spans[0][0] == 0 and sum(n for _, n in spans) == total
            for (f0, n0), (f1, _) in zip(spans[:-1], spans[1:]):
                assert f0 + n0 == f1
        assert [weak_shard(r, world, 10)[0] for r in range(world)] == [10 * r for r in range(world)]
    with pytest.raises(ValueError):
        strong_shard(2, 2, 10)


def _worker(rank, world, port, n_total, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import ref
    first, n = strong_shard(rank, world, n_total)
    u = torch.from_numpy(ref.philox_uniform(4, 1, first, 8, n))
    # per-shard Vegas sums of a cheap stand-in integrand on the shard's own uniforms (host logic only)
    e = np.tile(np.linspace(0, 1, 51), (8, 1))
    x, jac, idx = ref.vegas_map(e, u.numpy())
    f = jac * np.prod(1.0 + x, axis=1)
    sums = torch.from_numpy(ref.vegas_accumulate(f, idx, 50))
    gathered = [torch.zeros_like(sums) for _ in range(world)]
    dist.all_gather(gathered, sums)
    total = gathered[0].clone()      # what vegas_combine does on the device: fixed rank order
    for part in gathered[1:]:
        total = total + part
    ms = torch.tensor([10.0 + rank])
    dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    sizes = [torch.zeros(1, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(sizes, torch.tensor([n]))
    if rank == 0:
        q.put((total.numpy(), float(ms.item()), [int(s.item()) for s in sizes]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_reproduce_the_single_stream():
    from oracle import ref
    n_total, world, port = 1001, 2, 29653
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_total, q)) for r in range(world)]
    for p in procs:
        p.start()
    total, ms, sizes = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert sizes == [501, 500] and ms == 11.0
    u = ref.philox_uniform(4, 1, 0, 8, n_total)
    e = np.tile(np.linspace(0, 1, 51), (8, 1))
    x, jac, idx = ref.vegas_map(e, u)
    want = ref.vegas_accumulate(jac * np.prod(1.0 + x, axis=1), idx, 50)
    assert total[2] == want[2]
    assert np.max(np.abs(total - want) / (np.abs(want) + 1e-300)) < 1e-12


def test_reference_arm_prints_one_line_on_rank0_only():
    env = dict(os.environ, RANK="1", WORLD_SIZE="2")
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0 and out.stdout.strip() == ""
    env["RANK"] = "0"
    env["MADME_REF_SECONDS"] = "3"
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1", "--warmup", "0"],
                         capture_output=True, text=True, env=env, timeout=300)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0
