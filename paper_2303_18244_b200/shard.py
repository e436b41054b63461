"""Event sharding for multi-GPU runs: events are independent units (PAPER.md line 16,
"same functions on different data items"), so rank r of W takes a contiguous range of whole AoSoA pages
and no collective touches the data path.  Philox is counter-based on the GLOBAL event index
(include/me.h me_philox_uniform `first_event`), so the union of the shards is bit-identical to the
single-GPU batch."""


def shard_range(n_events, rank, world, page=32):
    """-> (first_event, count) for `rank`; ranges are contiguous, page-aligned starts, cover [0, n) exactly once."""
    if world < 1 or not (0 <= rank < world) or n_events < 0:
        raise ValueError("bad shard arguments")
    npages = (n_events + page - 1) // page
    base, extra = divmod(npages, world)
    p0 = rank * base + min(rank, extra)
    p1 = p0 + base + (1 if rank < extra else 0)
    first = min(p0 * page, n_events)
    last = min(p1 * page, n_events)
    return first, last - first
