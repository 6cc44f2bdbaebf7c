"""N > 1 path of bench.py on CPU: world_size-2 gloo.  The decode does not shard (replicas only), so
the only cross-rank logic is the max-over-ranks of the timings and the whole-job aggregate."""
import os
import socket

import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world)          # rank 1 is the slow replica
    dist.barrier()
    q.put((rank, ms, bench.aggregate_gbs(1 << 30, ms, world)))
    dist.destroy_process_group()


def test_replicas_max_over_ranks_gloo():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, agg in got:
        assert ms == 15.0                                          # every rank reports the slowest replica's time
        assert abs(agg - 2 * (1 << 30) / 15e-3 / 1e9) < 1e-9       # whole job = both replicas' bytes over that time


def test_single_rank_is_identity():
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.aggregate_gbs(10**9, 1.0, 1) == 1000.0
