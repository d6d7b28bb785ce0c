"""N > 1 is 'replicas only': each rank runs its own replica and only the elapsed time (MAX) and the
launch count (SUM) cross ranks.  world_size-2 gloo test of that aggregation on CPU."""
import os
import socket
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = [10.0, 12.5][rank]
    e2e = [30.0, 20.0][rank]
    (ms_max, e2e_max), (launches,) = bench.reduce_over_ranks(dist, [ms, e2e], [600 + rank], "cpu")
    value = bench.job_throughput(64, 64, 100, 5, world, ms_max)
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, ms_max, e2e_max, launches, value))


def test_replica_aggregation_world_size_2():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms_max, e2e_max, launches, value in out:
        assert ms_max == 12.5 and e2e_max == 30.0           # time = max over ranks
        assert launches == 1201                             # counts are summed
        assert abs(value - 64 * 64 * 100 * 2 * 5 / 12.5e-3) < 1e-6   # units of ALL ranks / max time


def test_single_rank_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks(None, [3.0], [7]) == ([3.0], [7])
