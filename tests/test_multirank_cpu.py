"""The N>1 path of bench.py is "replicas only": no data-path collective, only a barrier and a max-over-ranks
of the step time.  These world_size-2 gloo tests cover that host logic on CPU."""
import os
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist  # noqa: E402
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r measured (1 + r) s on the device and (3 - r) s end to end: the job's times are the per-entry maxima
    got = bench.max_over_ranks([1.0 + rank, 3.0 - rank])
    dist.barrier()
    seeds = bench.rank_gauge_seed(1001, rank)
    q.put((rank, got, seeds, bench.whole_job_seconds_per_rhs(got[0], 5, 8, world)))
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_metric_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, got, seed, val in res:
        assert got == [2.0, 3.0]                       # max over ranks, identical on every rank
        assert seed == 1001 + rank                     # independent gauge configuration per replica
        assert val == pytest.approx(2.0 / 5 / 16)      # whole-job seconds per RHS: 16 RHS per step over 2 ranks


def test_single_process_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks([0.25, 4.0]) == [0.25, 4.0]
    assert bench.whole_job_seconds_per_rhs(10.0, 5, 8, 1) == 0.25


def test_reference_arm_nonzero_ranks_do_no_work(monkeypatch, capsys):
    sys.path.insert(0, ROOT)
    import bench

    class A:
        pass
    a = A(); a.workload = "cfg1"; a.steps = 1; a.warmup = 0; a.gpus = 2
    bench.run_reference(a, rank=1, world=2)
    assert capsys.readouterr().out == ""
