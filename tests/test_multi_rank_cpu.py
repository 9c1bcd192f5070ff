"""-m "not gpu": the N > 1 paths on CPU, world_size 2 over gloo.  Default of bench.py:
replicas -- each rank runs the whole workload with its own seed and the only exchange is the max-over-ranks of
the timings and the sum of the work counts.  `--shard` / paper_2203_09467_b200/shard.py: one workload cut by
primaries, the one exchange being the final sum of tallies, totals and counters."""
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


# ---------------- sharding by primaries (paper_2203_09467_b200/shard.py) ----------------

def test_shard_ranges_are_contiguous_disjoint_and_cover():
    sys.path.insert(0, ROOT)
    from paper_2203_09467_b200 import shard
    for n in (0, 1, 7, 100000, 100003):
        for world in (1, 2, 3, 8):
            r = [shard.shard_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1
    import numpy as np
    prim = dict(E=np.arange(10.0), ptype=np.arange(10, dtype=np.int32))
    first, part = shard.shard_primaries(prim, 1, 3)
    assert first == 3 and part["E"].tolist() == [3.0, 4.0, 5.0] and part["ptype"].tolist() == [3, 4, 5]


def _fake_result(rank):
    import numpy as np
    return dict(edep=np.array([1.0, 2.0, 4.0]) * (rank + 1), escaped=0.5 + rank, below_cut=0.25, looper=0.0,
                E_in=10.0 * (rank + 1), steps=np.array([10, 20, 30], dtype=np.uint64) * (rank + 1),
                tracks=np.array([1, 2, 3], dtype=np.uint64), inter=np.arange(8, dtype=np.uint64) + rank,
                null_int=rank, track_steps=60 * (rank + 1), stalls=0, iterations=100 + rank, peak_live=7 - rank,
                peak_queue=1000 * (rank + 1), ms=5.0 - rank)


def _shard_worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import numpy as np
    from paper_2203_09467_b200 import shard
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    hist = np.full((3, 96), rank + 1, dtype=np.uint64)
    res, h = shard.all_reduce_results(_fake_result(rank), hist, "cpu")
    dist.barrier()
    out[rank] = ({k: (v.tolist() if hasattr(v, "tolist") else v) for k, v in res.items()}, h.tolist())
    dist.destroy_process_group()


def test_sharded_results_are_summed_over_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_shard_worker, args=(2, port, out), nprocs=2, join=True)
    for r in (0, 1):
        res, h = out[r]
        assert res["edep"] == [3.0, 6.0, 12.0] and res["escaped"] == 2.0 and res["below_cut"] == 0.5
        assert res["E_in"] == 30.0 and res["looper"] == 0.0
        assert res["steps"] == [30, 60, 90] and res["tracks"] == [2, 4, 6]
        assert res["inter"] == [2 * k + 1 for k in range(8)]
        assert res["null_int"] == 1 and res["track_steps"] == 180 and res["stalls"] == 0
        assert res["iterations"] == 101 and res["peak_live"] == 7 and res["peak_queue"] == 2000 and res["ms"] == 5.0
        assert h == [[3] * 96] * 3


def test_single_rank_shard_reduce_is_the_identity():
    sys.path.insert(0, ROOT)
    from paper_2203_09467_b200 import shard
    res, h = shard.all_reduce_results(_fake_result(0), None, "cpu")
    assert res["track_steps"] == 60 and h is None
