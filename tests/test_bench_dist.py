"""Host logic of bench.py's N > 1 path ("replicas only") with world_size 2 over gloo on the CPU:
the per-rank times are reduced with MAX and the whole-job value is all ranks' steps over the slowest rank's time."""
import os
import socket
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parents[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, str(ROOT))
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
    ms_max = bench.reduce_max(ms, world, "cpu")
    dist.barrier()
    out.put((rank, ms_max, bench.replicas_value(world, 4, ms_max)))
    dist.destroy_process_group()


def test_replicas_max_over_ranks_gloo():
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms_max, val in res:
        assert ms_max == 15.0
        assert val == pytest.approx(2 * 4 / 15e-3)


def test_single_rank_is_identity():
    sys.path.insert(0, str(ROOT))
    import bench
    assert bench.reduce_max(3.5, 1) == 3.5
    assert bench.replicas_value(1, 10, 100.0) == pytest.approx(100.0)
