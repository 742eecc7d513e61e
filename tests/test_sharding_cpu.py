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


# ---- slab sharding of the CCSD iteration --------------------------------------------------------------
@pytest.mark.parametrize("o,v", [(4, 16), (16, 96), (34, 224), (5, 7), (40, 256)])
@pytest.mark.parametrize("world", [1, 2, 3, 7, 8])
def test_slab_ranges_tile_every_index_range_once(o, v, world):
    """ccsd_shard_ranges (host arithmetic of the C library, no GPU): over the ranks the virtual-index slabs tile [0, v),
    the packed (a<b) row slabs tile [0, vv) on boundaries of the first virtual index, the (i<j) row slabs tile [0, oo);
    the row slabs are balanced to within one value of the first index."""
    from paper_2103_08473_b200.binding import shard_ranges, CCSDError
    if world > v:
        with pytest.raises(CCSDError):
            shard_ranges(o, v, 0, world)
        return
    oo, vv = o * (o - 1) // 2, v * (v - 1) // 2
    rs = [shard_ranges(o, v, r, world) for r in range(world)]
    for lo, hi, total in (("a_lo", "a_hi", v), ("w_lo", "w_hi", vv), ("ij_lo", "ij_hi", oo)):
        pos = 0
        for r in rs:
            assert r[lo] == pos and r[hi] >= r[lo]
            pos = r[hi]
        assert pos == total
    before = lambda a: a * v - a * (a + 1) // 2             # packed rows before the pairs of first index a
    for r in rs:
        assert r["w_lo"] == before(r["wa_lo"]) and r["w_hi"] == min(vv, before(r["wa_hi"]))
        assert abs((r["w_hi"] - r["w_lo"]) - vv / world) <= v
        assert abs((r["a_hi"] - r["a_lo"]) - v / world) <= 1
    with pytest.raises(CCSDError):
        shard_ranges(o, v, world, world)


class _FakeSlabContext:
    """Stands in for a sharded CCSD context on CPU: residual() writes this rank's slab of a known matrix (zero elsewhere),
    update() reduces the summed matrix to two numbers.  No arithmetic of the method."""

    def __init__(self, rank, world, rows=12, cols=40):
        import torch
        self.rank, self.world = rank, world
        g = torch.Generator().manual_seed(5)
        self.full = torch.view_as_complex(torch.randn((rows, cols, 2), generator=g, dtype=torch.float64))
        self.s2 = torch.zeros((rows, cols), dtype=torch.complex128)
        from paper_2103_08473_b200.sharding import shard_range
        self.first, self.count = shard_range(cols, rank, world)

    def residual(self):
        self.s2.zero_()
        self.s2[:, self.first:self.first + self.count] = self.full[:, self.first:self.first + self.count]

    def s2_view(self):
        return self.s2

    def update(self):
        return complex(self.s2.sum()), float(self.s2.abs().max())


def _slab_rank_main(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import torch
    import torch.distributed as dist
    from paper_2103_08473_b200.sharding import iterate_sharded
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ctx = _FakeSlabContext(rank, world)
    out = [iterate_sharded(ctx) for _ in range(2)]
    q.put((rank, out, bool(torch.equal(ctx.s2, ctx.full))))
    dist.destroy_process_group()


def test_two_rank_slab_iteration_protocol_gloo():
    """residual (slab) -> all-reduce of the complex S2 -> replicated update, world_size 2 over gloo: both ranks end with the
    complete S2 and identical update results."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 33500 + os.getpid() % 2000
    procs = [ctx.Process(target=_slab_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][2] and res[1][2]
    assert res[0][1] == res[1][1] and res[0][1][0] == res[0][1][1]
    ref = _FakeSlabContext(0, 1)
    ref.residual()
    assert abs(res[0][1][0][0] - ref.update()[0]) < 1e-12
