"""The N > 1 path of bench.py (replicas only) on CPU: two processes, gloo backend."""
import os
import socket

import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist                      # noqa: E402
import torch.multiprocessing as mp                    # noqa: E402

from paper_2603_24532_b200 import replicas, workloads as W   # noqa: E402


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        assert replicas.world_size() == world and replicas.rank() == rank
        wl = W.workload("cfg1")
        runs = replicas.replica_runs(wl)
        assert [r.name for r in runs] == [r.name for r in wl.runs]          # every rank: the whole workload
        cfg = runs[0].configurations(16)
        replicas.barrier()
        local = 0.010 * (rank + 1)                                          # rank 1 is the slow replica
        t = replicas.max_over_ranks(local)
        rate = replicas.whole_job_rate(wl.evals, 3, t)
        # identical seeded inputs on every rank: replicas integrate the same configurations
        chk = torch.tensor([float(cfg.sum())], dtype=torch.float64)
        both = [torch.zeros_like(chk) for _ in range(world)]
        dist.all_gather(both, chk)
        out.put((rank, t, rate, float(both[0]), float(both[1])))
    finally:
        dist.destroy_process_group()


def test_two_replicas_time_as_the_slowest_and_count_both():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    evals = W.workload("cfg1").evals
    for rank, t, rate, c0, c1 in res:
        assert t == pytest.approx(0.020)                                    # MAX over ranks
        assert rate == pytest.approx(2 * evals * 3 / 0.020)                 # whole-job aggregate
        assert c0 == c1


def test_single_process_helpers_do_not_need_a_process_group():
    assert replicas.world_size() == 1 and replicas.rank() == 0
    replicas.barrier()
    assert replicas.max_over_ranks(0.5) == 0.5
    assert replicas.whole_job_rate(100, 2, 0.5) == 400.0
