"""Host logic of the multi-GPU split of the perturbative triples (the three nested occupied loops run over
"only the unique blocks"; the occupied triples i<j<k are independent units of equal cost).  One process per GPU, every
rank holds the same amplitudes, rank r evaluates a contiguous range of the lexicographic list of triples
(ccsd_triples_range) and the three complex partial sums are added with ONE all-reduce of six doubles: no data-path
collective.  Importable without a CUDA device (the gloo tests run it on CPU); there is no arithmetic of the method here.
"""
from __future__ import annotations

KEYS = ("+T", "(T)", "-T")


def shard_range(n: int, rank: int, world: int) -> tuple[int, int]:
    """(first, count) of rank's contiguous share of n equal-cost units: counts differ by at most one, ranges tile
    [0, n) in rank order (contiguous ranges keep consecutive triples, which share integral slices in L2, together)."""
    if n < 0 or world < 1 or not (0 <= rank < world):
        raise ValueError(f"shard_range({n}, {rank}, {world})")
    base, extra = divmod(n, world)
    first = rank * base + min(rank, extra)
    return first, base + (1 if rank < extra else 0)


def allreduce_energies(partial: dict, group=None, device="cpu") -> dict:
    """Sum the {"+T", "(T)", "-T"} complex partial sums over the ranks of `group` (six doubles, one all-reduce)."""
    import torch
    import torch.distributed as dist
    flat = []
    for k in KEYS:
        flat += [partial[k].real, partial[k].imag]
    t = torch.tensor(flat, dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    t = t.cpu().tolist()
    return {k: complex(t[2 * q], t[2 * q + 1]) for q, k in enumerate(KEYS)}
