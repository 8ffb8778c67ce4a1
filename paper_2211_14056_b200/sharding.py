"""Event-range sharding over ranks: events are independent and event e's random numbers
depend only on (seed, iteration, e), so rank r of N takes the global event indices [first, first + n) below and the
union over ranks is the single-GPU stream, whatever N is.  No arithmetic of the method lives here.
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


def combine_vegas_sums(per_rank_sums):
    """Sum the per-shard (sum f, sum f^2, n_pass, S_{d,i}) vectors in FIXED rank order (reproducible whatever the
    arrival order): what a multi-GPU vegas_iterate does between vegas_integrand and vegas_refine."""
    total = None
    for s in per_rank_sums:
        total = s.clone() if total is None else total + s
    return total
