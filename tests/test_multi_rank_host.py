"""world_size-2 gloo test of bench.py's N > 1 host logic ("replicas only"): the barrier,
the max-over-ranks reduction of device-measured times and the whole-job aggregation, run on CPU."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    sys.path.insert(0, ROOT)
    import bench
    r, w, local = bench.dist_setup(world)
    assert (r, w, local) == (rank, world, rank)
    bench.barrier(w)
    ms = 2.0 + rank                       # rank 1 is the slow replica
    worst = bench.max_over_ranks(ms, w)
    # whole-job value as run_cuda_arm forms it: every replica processes cells_per_step in the slowest time
    value = w * 1000.0 / (worst * 1e-3) / 1e9
    q.put((rank, worst, value))
    dist.destroy_process_group()


def test_max_over_ranks_and_aggregate_with_two_gloo_ranks():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [3.0, 3.0]               # both ranks see the slowest replica's time
    assert abs(res[0][2] - 2 * 1000.0 / 3e-3 / 1e9) < 1e-12  # aggregate = N x per-replica work / max time


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(1.5, 1) == 1.5
    bench.barrier(1)
    assert not dist.is_initialized()
