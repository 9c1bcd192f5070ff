"""Sharding a transport by primaries over the ranks of a torch.distributed job.

PAPER.md:54: "domain replication ... particle events are decomposed across MPI ranks".  Every rank holds the
whole problem (geometry, tables: < 1 MB) and its own track store; rank r transports the contiguous range
shard_range(n, r, world) of the primaries with `Problem.set_primary_offset(first)`, so that every history is
the one the unsharded run would produce (a history depends on the seed and its primary index only).  The ONE
exchange of the job is the sum of the tallies, the energy totals and the counters at the end: a few hundred
bytes, one all-reduce per dtype (NCCL over NVLink on GPUs; any backend works, the tests use gloo on CPU).
No step of the hot path runs here: this is plumbing around `emx_transport`.
"""
import numpy as np

SUMMED = ("edep", "escaped", "below_cut", "looper", "E_in")                       # float64
COUNTED = ("steps", "tracks", "inter", "null_int", "track_steps", "stalls")       # integers
MAXED = ("iterations", "peak_live", "peak_queue", "ms")


def shard_range(n, rank, world):
    """[first, last) of the n primaries that rank `rank` of `world` transports: contiguous, disjoint, covering,
    sizes differing by at most one."""
    if not (0 <= rank < world) or n < 0:
        raise ValueError("shard_range: need 0 <= rank < world and n >= 0")
    return (n * rank) // world, (n * (rank + 1)) // world


def shard_primaries(prim, rank, world):
    """(first, the slice of every array of the primary dict) for this rank"""
    a, b = shard_range(len(prim["E"]), rank, world)
    return a, {k: v[a:b] for k, v in prim.items()}


def all_reduce_results(res, hist=None, device="cpu"):
    """Sum (tallies, energies, counters, histogram) and max (iterations, peaks, milliseconds) of the per-rank
    results of `Problem.transport` over all ranks; every rank gets the totals.  Without an initialised process
    group (or with one rank) the input is returned unchanged."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return dict(res), hist
    out = dict(res)
    # float64 sums: one flat buffer
    parts = [np.atleast_1d(np.asarray(res[k], dtype=np.float64)).ravel() for k in SUMMED]
    f = torch.from_numpy(np.concatenate(parts)).to(device)
    dist.all_reduce(f, op=dist.ReduceOp.SUM)
    f = f.cpu().numpy()
    o = 0
    for k, p in zip(SUMMED, parts):
        v = f[o:o + p.size]
        out[k] = v.copy() if np.ndim(res[k]) else float(v[0])
        o += p.size
    # integer sums (counters fit int64)
    iparts = [np.atleast_1d(np.asarray(res[k]).astype(np.int64)).ravel() for k in COUNTED]
    if hist is not None:
        iparts.append(np.asarray(hist).astype(np.int64).ravel())
    c = torch.from_numpy(np.concatenate(iparts)).to(device)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    c = c.cpu().numpy()
    o = 0
    for k, p in zip(COUNTED, iparts):
        v = c[o:o + p.size]
        out[k] = v.astype(np.uint64) if np.ndim(res[k]) else int(v[0])
        o += p.size
    hist_out = None
    if hist is not None:
        hist_out = c[o:].astype(np.uint64).reshape(np.asarray(hist).shape)
    m = torch.tensor([float(res[k]) for k in MAXED], dtype=torch.float64, device=device)
    dist.all_reduce(m, op=dist.ReduceOp.MAX)
    for k, v in zip(MAXED, m.tolist()):
        out[k] = v if k == "ms" else int(v)
    return out, hist_out
