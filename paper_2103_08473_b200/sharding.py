"""Host logic of the two multi-GPU splits.

(1) Slab sharding of the CCSD iteration (replaces the paper's block-distributed tensors and remote
MPI_Accumulate, which the authors name as what limits their scaling): one process and
one context per GPU, every rank holds the same amplitudes, rank r evaluates its slab of every large contraction
(ccsd_options.shard_rank / shard_world) into an S2 that is zero elsewhere; ONE all-reduce of the packed S2 per iteration
(allreduce_complex_, 214 MiB at cfg3) completes the residual, the Jacobi / DIIS / energy step is replicated
(iterate_sharded).  The library itself issues no collective.

(2) Host logic of the multi-GPU split of the perturbative triples (the three nested occupied loops run over
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


def allreduce_complex_(t, group=None):
    """In-place sum of a complex128 tensor over the ranks of `group` (NCCL has no complex dtype: the (re, im) pairs are
    reduced as float64).  Every rank ends with the same bits (the reduction order of an all-reduce does not depend on the
    rank), so the replicated update that follows keeps the ranks in lock step.  No-op without an initialised group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return t
    dist.all_reduce(torch.view_as_real(t), op=dist.ReduceOp.SUM, group=group)
    return t


def iterate_sharded(ctx, group=None):
    """One iteration of a sharded context `ctx` (anything with residual(), s2_view(), update()): this rank's slab of the
    residual, the all-reduce of S2, the replicated update.  CCSD.iterate does exactly this; spelled out here so that the
    protocol can be exercised without a GPU (tests/test_sharding_cpu.py)."""
    ctx.residual()
    allreduce_complex_(ctx.s2_view(), group)
    return ctx.update()
