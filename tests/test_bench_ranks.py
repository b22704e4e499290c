"""The N > 1 path of bench.py is "replicas only": a barrier and the MAX of a timing scalar over ranks.
Covered here with two gloo processes on the CPU (no GPU needed)."""
import os
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import bench
    R = bench.Ranks("gloo")
    R.barrier()
    slowest = R.max(1.0 + rank)                       # rank 1 is "slower"
    agg = R.aggregate(units_per_rank=100.0, seconds_local=1.0 + rank)
    out.put((rank, R.world, slowest, agg))
    R.close()


def test_two_rank_replicas_take_the_slowest_time():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, world, slowest, agg in res:
        assert world == 2
        assert slowest == 2.0                           # max over ranks
        assert agg == 2 * 100.0 / 2.0                   # all ranks' units / slowest time


def test_reference_arm_runs_on_rank0_only(monkeypatch, capsys):
    sys.path.insert(0, ROOT)
    import bench
    import workloads as W
    monkeypatch.setenv("RANK", "1")
    bench.run_reference(bench.argparse.Namespace(config=0, steps=1, warmup=0, gpus=2), W)
    assert capsys.readouterr().out == ""               # other ranks print nothing and do no work
    monkeypatch.setenv("RANK", "0")
    bench.run_reference(bench.argparse.Namespace(config=0, steps=1, warmup=0, gpus=2), W)
    line = bench.json.loads(capsys.readouterr().out)
    assert line["impl"] == "reference" and line["cpu_baseline"]["kind"] == "oracle" and line["value"] > 0
