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


def test_gpus_flag_without_torchrun_relaunches_itself_and_never_claims_more_ranks_than_it_runs(monkeypatch):
    """`python bench.py --gpus N` outside torchrun must start N ranks (round-1 finding: it silently ran one replica and
    printed n_gpus 1); a WORLD_SIZE that disagrees with --gpus is an error, not a quiet single-replica run."""
    import subprocess
    import bench
    calls = []
    monkeypatch.setattr(subprocess, "call", lambda cmd: calls.append(cmd) or 0)
    monkeypatch.delenv("WORLD_SIZE", raising=False)
    monkeypatch.setattr(sys, "argv", ["bench.py", "--gpus", "4", "--steps", "3", "--config", "2"])
    assert bench.main() == 0
    (cmd,) = calls
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--nnodes=1"] and cmd[cmd.index("--nproc-per-node") + 1] == "4"
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[-6:] == ["--gpus", "4", "--steps", "3", "--config", "2"]
    assert os.path.basename(cmd[cmd.index("--master-port") + 2]) == "bench.py"
    monkeypatch.setenv("WORLD_SIZE", "2")                       # launched by someone else with the wrong world size
    assert bench.main() == 2 and len(calls) == 1
