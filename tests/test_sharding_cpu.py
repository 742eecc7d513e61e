"""Host logic of the multi-GPU split of the triples (paper_2103_08473_b200/sharding.py) on CPU: the ranges tile the list
of occupied triples exactly once with counts differing by at most one, and (world_size 2, gloo) the all-reduce of the
per-rank partial sums returns the total on every rank."""
import itertools
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


@pytest.mark.parametrize("n,world", [(0, 1), (1, 4), (4, 4), (5984, 8), (5984, 3), (10, 7), (1330, 2)])
def test_shard_range_tiles_the_list(n, world):
    from paper_2103_08473_b200.sharding import shard_range
    pieces = [shard_range(n, r, world) for r in range(world)]
    pos = 0
    for first, count in pieces:
        assert first == pos and count >= 0
        pos += count
    assert pos == n
    counts = [c for _, c in pieces]
    assert max(counts) - min(counts) <= 1
    with pytest.raises(ValueError):
        shard_range(n, world, world)
    with pytest.raises(ValueError):
        shard_range(-1, 0, world)


def _value(i, j, k):
    # a stand-in per-triple contribution with a non-trivial dependence on every index (no arithmetic of the method)
    return complex(1.0 / (1 + i + 2 * j + 3 * k), (i - k) * 0.125 + j * 0.015625)


def _rank_main(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import torch.distributed as dist
    from paper_2103_08473_b200.sharding import allreduce_energies, shard_range
    dist.init_process_group("gloo", rank=rank, world_size=world)
    o = 9
    triples = list(itertools.combinations(range(o), 3))        # lexicographic i<j<k, the order of ccsd_triples_range
    first, count = shard_range(len(triples), rank, world)
    mine = triples[first:first + count]
    part = {"+T": sum(_value(*t).real for t in mine) + 0j, "(T)": sum(_value(*t) for t in mine),
            "-T": sum(_value(*t).conjugate() for t in mine)}
    tot = allreduce_energies(part, device="cpu")
    q.put((rank, count, tot["+T"], tot["(T)"], tot["-T"]))
    dist.destroy_process_group()


def test_two_rank_partial_sums_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    triples = list(itertools.combinations(range(9), 3))
    full = sum(_value(*t) for t in triples)
    assert res[0][1] + res[1][1] == len(triples) == 84
    for r in res:
        assert abs(r[2] - full.real) < 1e-13 and abs(r[3] - full) < 1e-13 and abs(r[4] - full.conjugate()) < 1e-13
    assert res[0][2:] == res[1][2:]                      # every rank ends with the same numbers
