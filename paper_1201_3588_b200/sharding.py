"""Packet sharding over ranks: host logic only.

Within a batch packets are independent (temperatures frozen, per-packet Philox streams), so a
batch [first, first+n) is dealt to the ranks in contiguous ranges; every rank transports its
own range, tallying the batch's absorptions into a per-batch uint32 array
(`transport_batch_delta`), the ranks sum those arrays with ONE all-reduce (4 bytes per storage
slot, in the library's storage order: no layout conversion, no allocation), and every rank adds
the sum to its cumulative tally and updates the temperatures with the global package count
(`accumulate_update`).  Integer sums commute, so tallies and temperatures are bit-identical
to a single-rank run over the same packet ids, and every rank ends up with the global tally.

The engine is anything with the binding's calls (mcrt.Context on a GPU); torch is used for the
collective only.
"""
from __future__ import annotations


def rank_range(first: int, n: int, world: int, rank: int):
    """Contiguous near-equal split of packet ids [first, first+n) -> (first_r, n_r).
    The first (n mod world) ranks take one extra packet; ranges tile the batch exactly."""
    if world < 1 or not (0 <= rank < world) or n < 0:
        raise ValueError("rank_range: bad world / rank / n")
    base, extra = divmod(n, world)
    lo = rank * base + min(rank, extra)
    return first + lo, base + (1 if rank < extra else 0)


class ShardedRunner:
    """Runs batches of a job whose packets are sharded over the ranks of a process group."""

    def __init__(self, engine, dist=None, group=None):
        self.engine, self.dist, self.group = engine, dist, group
        self.world = dist.get_world_size(group) if dist is not None else 1
        self.rank = dist.get_rank(group) if dist is not None else 0
        self.n_cum = 0                      # packages emitted by ALL ranks so far

    def run_batch(self, seed: int, first: int, n: int, stream=None):
        """One batch [first, first+n) of the whole job.  Returns this rank's (first, count)."""
        f, c = rank_range(first, n, self.world, self.rank)
        self.n_cum += n
        if self.world == 1:
            self.engine.run_batch(seed, f, c, stream)
            return f, c
        delta = self.engine.transport_batch_delta(seed, f, c, stream)   # this rank's counts of this batch
        self.dist.all_reduce(delta, op=self.dist.ReduceOp.SUM, group=self.group)
        self.engine.accumulate_update(delta, self.n_cum, stream)
        return f, c

    def reduce_counts(self, t):
        """Sum an integer tensor (SED, counters) over ranks at read-out."""
        if self.world > 1:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM, group=self.group)
        return t
