"""Host-side logic of the N > 1 path.

Histories are independent given their counter-based ids, so the path shards with no data-path
collective.  Two ways, both used by bench.py / the tests:
  * weak scaling  -- every rank runs the same workload with its own Philox seed (`rank_seed`);
  * id sharding   -- one workload, contiguous primary-id ranges per rank (`id_range`), children stay with
                     their root.
Either way the only exchange is one sum of the (n_th x n_nu x 4) tally at the end (`reduce_tally`).
"""
from __future__ import annotations


def rank_seed(base_seed: int, rank: int) -> int:
    """Distinct 64-bit Philox key per rank; rank 0 keeps the base seed (so N = 1 reproduces the config)."""
    return (int(base_seed) + 0x9E3779B97F4A7C15 * int(rank)) & 0xFFFFFFFFFFFFFFFF


def id_range(n_primaries: int, rank: int, world: int) -> tuple[int, int]:
    """(first, count) of the contiguous primary-id range of `rank`; ranges tile [0, n) exactly."""
    base, rem = divmod(int(n_primaries), int(world))
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def reduce_tally(tensors, dist):
    """Sum the tally accumulators (sum wE, sum (wE)^2, sum w, count) over all ranks, in place."""
    for t in tensors:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return tensors
