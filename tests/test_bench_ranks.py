"""The N > 1 path of bench.py is "replicas only": the only cross-rank logic is the
max-over-ranks timing and the whole-job update count.  Covered here with 2 gloo ranks on the CPU."""
import os
import sys
from pathlib import Path

import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parent.parent


def _rank(rank, world, port, q):
    sys.path.insert(0, str(ROOT))
    import torch.distributed as dist
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms, upd = bench.aggregate_over_ranks(10.0 + 5.0 * rank, 1000, world, device="cpu")
        q.put((rank, ms, upd))
    finally:
        dist.destroy_process_group()


def test_replicas_aggregate_max_time_and_sum_updates():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29000 + os.getpid() % 2000
    procs = [ctx.Process(target=_rank, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got == [(0, 15.0, 2000), (1, 15.0, 2000)]


def test_reference_arm_other_ranks_do_no_work(monkeypatch, capsys):
    sys.path.insert(0, str(ROOT))
    import bench
    monkeypatch.setenv("RANK", "1")
    bench.run_reference(type("A", (), {"config": 1, "n": 16, "steps": 1, "warmup": 0, "gpus": 2})())
    assert capsys.readouterr().out == ""
