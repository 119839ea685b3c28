"""The N > 1 path of bench.py on CPU: the path does not shard (replicas only), so all that is
shared between ranks is the timing: max over ranks, whole-job throughput = world x per-rank units / that time.
Two gloo ranks on 127.0.0.1."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        got = bench.reduce_times_max([10.0 + rank, 20.0 - rank], torch.device("cpu"))
        dist.barrier()
        out.put((rank, got))
    finally:
        dist.destroy_process_group()


def test_times_are_max_over_ranks_and_value_is_whole_job():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0] == [11.0, 20.0] and res[1] == [11.0, 20.0]
    sys.path.insert(0, ROOT)
    import bench
    assert bench.job_throughput(12_096_000, 2, 10.0) == pytest.approx(2 * 12_096_000 / 0.010)
    assert bench.reduce_times_max([3.0], "cpu") == [3.0]           # no process group: identity
