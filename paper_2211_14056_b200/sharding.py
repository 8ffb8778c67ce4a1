"""Event-range sharding over ranks: events are independent and event e's random numbers
depend only on (seed, iteration, e), so rank r of N takes the global event indices [first, first + n) below and the
union over ranks is the single-GPU stream, whatever N is.  No arithmetic of the method lives here: the one exchange of
a sharded Vegas iteration is gathered here and ADDED by the library (vegas_combine, fixed rank order).
"""


def weak_shard(rank: int, world: int, events_per_rank: int):
    """Weak scaling (bench.py): every rank processes `events_per_rank` events; returns (first_event, n_events)."""
    if not (0 <= rank < world) or events_per_rank < 0:
        raise ValueError("bad shard request")
    return rank * events_per_rank, events_per_rank


def strong_shard(rank: int, world: int, total_events: int):
    """Strong scaling: `total_events` split into contiguous ranges whose sizes differ by at most one."""
    if not (0 <= rank < world) or total_events < 0:
        raise ValueError("bad shard request")
    base, extra = divmod(total_events, world)
    first = rank * base + min(rank, extra)
    return first, base + (1 if rank < extra else 0)


def gather_sums(sums, group=None):
    """All-gather every rank's (sum f, sum f^2, n_pass, S_{d,i}) vector; returns them stacked in RANK order,
    [world, n_out], on the device of `sums` (through the host with the gloo backend).  The addition is the library's
    (vegas_combine): no arithmetic here."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    on_host = dist.get_backend(group) == "gloo"
    mine = sums.cpu() if on_host else sums
    parts = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(parts, mine, group=group)
    return torch.stack(parts).to(sums.device).contiguous()
