"""Multi-GPU is "replicas only": the only cross-rank logic is the barrier + max-over-ranks timing and the
whole-job aggregation in bench.py.  This runs exactly those functions in two processes over gloo on CPU."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, ws, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(ws), LOCAL_RANK=str(rank))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=ws)
    assert bench._dist() == (ws, rank, rank)
    bench.replica_barrier(ws)
    my_ms = 10.0 + 5.0 * rank            # rank 1 is the slow replica
    slowest = bench.replica_max(my_ms, ws, torch.device("cpu"))
    fps = bench.aggregate_fps(ws, 80, slowest)
    bench.replica_barrier(ws)
    out.put((rank, slowest, fps))
    dist.destroy_process_group()


def test_two_replicas_barrier_and_max_over_ranks():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, slowest, fps in res:
        assert slowest == 15.0                                   # both ranks agree on the slowest replica
        assert abs(fps - 2 * 80 / 15.0e-3) < 1e-6                # whole-job frames/s over both replicas


def test_single_rank_needs_no_process_group():
    import bench
    assert bench.replica_max(3.5, 1, None) == 3.5
    assert bench.aggregate_fps(1, 8, 2.0) == 4000.0
    bench.replica_barrier(1)
