"""Host-side logic of bench.py on CPU: flop accounting, the reference arm's JSON line, and the N>1 launch path
(world_size 2, gloo): one process per rank, max-over-ranks timing, rank 0 alone reports."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def test_flop_table_matches_survey_totals():
    import bench
    # 0.091 / 1.446 / 11.18 TFLOP per iteration at cfg 1 / 2 / 3; ladder 0.020 / 0.357 / 2.80
    for (o, v), tot, lad in (((16, 96), 0.091e12, 0.020e12), ((24, 160), 1.446e12, 0.357e12), ((34, 224), 11.18e12, 2.80e12)):
        f = bench.flops_per_iteration(o, v)
        assert abs(f["total"] / tot - 1) < 0.02
        assert abs(f["pp_ladder"] / lad - 1) < 0.02
        assert f["Hvovo_quad"] == f["ring_gemm"] == 8 * (o * v) ** 3


def test_reference_arm_prints_contract_line():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "cfg0",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert out.returncode == 0, out.stderr
    line = json.loads(out.stdout.strip().splitlines()[-1])
    assert line["impl"] == "reference" and line["unit"] == "s/iteration" and line["higher_is_better"] is False
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0


def _rank_main(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # every rank measured a different time; the reported one is the max; only rank 0 reports
    t = bench.max_over_ranks(10.0 + rank, dist, device="cpu")
    q.put((rank, t, bench.is_reporting_rank()))
    dist.destroy_process_group()


def test_two_rank_replicas_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0] == (0, 11.0, True) and res[1] == (1, 11.0, False)
