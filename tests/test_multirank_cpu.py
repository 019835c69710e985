"""The N > 1 path of bench.py shards rows across ranks with no data-path collective:
the only distributed logic is the rendezvous, the barrier and the max-over-ranks timing.  Covered here
with world_size 2 on the gloo backend (CPU)."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dist.barrier()
    t = bench.reduce_max_over_ranks(1.0 + rank, dist, "cpu")      # rank 1 is the slow one
    out.put((rank, t, bench.rank_seed(rank)))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_gloo_max_time_and_distinct_shards():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g[1] for g in got] == [2.0, 2.0]          # both ranks see the slowest rank's time
    assert got[0][2] != got[1][2]                     # every rank draws its own rows


def test_single_rank_passthrough():
    import bench
    assert bench.reduce_max_over_ranks(3.5, None, "cpu") == 3.5
