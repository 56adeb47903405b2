"""N > 1 path of bench.py on CPU: world_size-2 gloo processes (replicas only, no data-path
collective; job time = max over ranks, commits / launches = sum over ranks, value = whole-job steps/s)."""
import os
import sys

import pytest

torch = pytest.importorskip("torch")
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r measured (1000 + 500 r) us of device time, (2 + r) s of wall time, 10 + r commits, 100 launches
    dev_us, wall, commits, launches = bench.reduce_over_ranks(dist, "cpu", 1000.0 + 500.0 * rank, 2.0 + rank, 10 + rank, 100)
    dist.barrier()
    out.put((rank, dev_us, wall, commits, launches, bench.job_value(world, 4, dev_us)))
    dist.destroy_process_group()


def test_two_rank_gloo_reduction():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29000 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, dev_us, wall, commits, launches, value in res:
        assert dev_us == 1500.0 and wall == 3.0          # max over ranks
        assert commits == 21 and launches == 200          # sum over ranks
        assert abs(value - 2 * 4 / 1500e-6) < 1e-6        # whole-job steps/s: both replicas' steps over the slowest rank's time


def test_reference_arm_runs_on_rank0_only(monkeypatch):
    sys.path.insert(0, ROOT)
    import bench

    class A:
        workload, steps, warmup, gpus = "C2", 1, 0, 2
    monkeypatch.setenv("RANK", "1")
    called = []
    monkeypatch.setattr(bench, "cpu_baseline", lambda *a, **k: called.append(1))
    assert bench.run_reference(A) is None and not called   # ranks > 0 exit without work
