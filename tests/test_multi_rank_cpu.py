"""-m "not gpu": the N > 1 path of bench.py on CPU, world_size 2 over gloo.  The path does not shard
("replicas only"): each rank runs the whole workload with its own seed and the only
exchange is the max-over-ranks of the timings and the sum of the work counts."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    seed = bench.replica_seed(4, rank)
    ms = 100.0 + 50.0 * rank            # rank 1 is the slower one
    steps = 1000 * (rank + 1)
    (t_ms, t_e2e), (c_steps, c_e2e) = bench.reduce_over_ranks([ms, 2 * ms], [steps, 2 * steps], "cpu")
    dist.barrier()
    out[rank] = (seed, t_ms, t_e2e, c_steps, c_e2e)
    dist.destroy_process_group()


def test_replicas_reduce_max_time_and_sum_work_over_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
    assert out[0][0] == 4 and out[1][0] == 1004                       # independent histories per replica
    for r in (0, 1):
        assert out[r][1:] == (150.0, 300.0, 3000.0, 6000.0)           # max of the times, sum of the work


def test_single_rank_reduce_is_the_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks([1.5], [7], "cpu") == ([1.5], [7.0])
