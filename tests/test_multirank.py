"""Host logic of the N > 1 bench path (replicas only, no data-path collective): world-size-2 gloo
run on CPU of bench.aggregate_over_ranks -- slowest rank's time, sum of the ranks' units."""
import os
import socket

import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms, units = bench.aggregate_over_ranks(10.0 + 5.0 * rank, 1000.0 * (rank + 1))
    out.put((rank, ms, units))
    dist.barrier()
    dist.destroy_process_group()


def test_aggregate_over_two_ranks_gloo():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    for rank, ms, units in got:
        assert ms == 15.0          # max over ranks
        assert units == 3000.0     # whole-job units


def test_single_process_is_identity():
    import bench
    assert bench.aggregate_over_ranks(7.5, 42.0) == (7.5, 42.0)
