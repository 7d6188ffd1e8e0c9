"""CPU, world_size 2, gloo: the host logic of the N > 1 bench path ("replicas only": no data-path collective; the only
exchange is the max-over-ranks of the device times and the barrier around the timed region)."""
import os
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # rank r measured (1 + r) s on the device and (2 + 0.5 r) s end to end
        t_dev, t_e2e = bench.max_over_ranks([1.0 + rank, 2.0 + 0.5 * rank], dist, torch.device("cpu"))
        dist.barrier()
        out.put((rank, t_dev, t_e2e, bench.rank_seed(7, rank)))
    finally:
        dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_gloo():
    import torch.multiprocessing as mp
    import bench
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    world, port = 2, 29400 + os.getpid() % 500
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[0] for r in res] == [0, 1]
    for _, t_dev, t_e2e, _ in res:          # every rank sees the slowest rank's times
        assert t_dev == pytest.approx(2.0) and t_e2e == pytest.approx(2.5)
    assert [r[3] for r in res] == [7, 8]    # distinct Philox keys per replica
    # whole-job aggregate: both replicas' units over the max time
    assert bench.whole_job_value(49152, 20, world, 2.0) == pytest.approx(2 * 49152 * 20 / 2.0)


def test_single_process_needs_no_collective():
    import torch
    import bench
    assert bench.max_over_ranks([0.25, 0.5], None, torch.device("cpu")) == [0.25, 0.5]
    assert bench.whole_job_value(100, 3, 1, 0.5) == pytest.approx(600.0)
