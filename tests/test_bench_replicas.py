"""Host-side logic of `bench.py --gpus N` (replicas only, no data-path collective): the whole-job
value is all ranks' grid-point steps over the slowest rank's time.  Two gloo processes on CPU."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    seconds = 0.5 if rank == 0 else 0.8            # rank 1 is the slow one
    v = bench.whole_job_value(seconds, 1000, 4, world)
    m = bench.max_over_ranks(float(rank), world)
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, v, m))


def test_whole_job_value_uses_the_slowest_rank_world_size_two():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, v, m in got:
        assert v == pytest.approx(2 * 1000 * 4 / 0.8)
        assert m == 1.0


def test_single_rank_is_the_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.whole_job_value(0.25, 1000, 5, 1) == pytest.approx(20000.0)
    assert bench.max_over_ranks(3.5, 1) == 3.5
