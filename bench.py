"""bench.py -- track-steps/s and primaries/s of the EM-shower step loop on B200 (BASELINE.json `metric`).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--primaries n] [--slots s] [--shard]
                    [--impl reference]

One "step" = one pass of the whole hot path (refill, step kernels, secondaries, tallies, until no track is
left) over one batch of synthetic primaries: by default the full BASELINE config 4 ("throughput stress":
barrel detector in a 4 T field, 100 000 primaries of 1-100 GeV, 2^20 track slots), the largest
single-GPU configuration.  Inputs are seeded and synthetic (paper_2203_09467_b200/workloads.py).
`value` is device-timed with the primaries already resident in HBM; `e2e` is the same metric through
emx_transport_host with HOST buffers (uploads and the tally read-back inside the timed region).
N > 1 (torchrun): independent replicas, one per GPU, different seeds (the default), or with
--shard ONE workload cut by primaries over the ranks with a final all-reduce of the tallies (strong scaling).
`--impl reference` times the oracle (plain fp64 C, oracle/) on the host cores on a bounded sample.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
from paper_2203_09467_b200 import workloads as W  # noqa: E402

METRIC, UNIT = "track_steps_per_sec", "track-steps/s"
# Algorithmic bytes per unit of each step kernel (five 16-byte words per slot -- (x, y), (z, ux),
# (uy, uz), (E, track id), (prim, step, vol, surf) -- plus one-byte flags; 80-byte stack records).  Units = the slots
# the kernel processed, counted by the kernel itself (emx_get_lanes).
B_STAGE = {
    "k_a<gamma>": 82 + 50,        # slot read (5 words, alive, stage) + (x, y), (z, ux), ids, alive, stage written
    "k_a<charged>": 83 + 66,      # + ptype read; + (E, id) written
    "k_a0": 35 + 10,              # (E, id), ids, stage, ptype read; s_phys, act, stage written
    "k_field": 91 + 62,           # slot + s_phys, act, ptype, stage read; 3 words + path, surface hit, act, stage written
    "k_a2": 97 + 34,              # slot + act, path, hit, stage, alive, ptype read; (E, id), ids, alive, stage written
    "k_b<gamma>": 4 + 81 + 66,    # list entry + slot read; (z, ux), (uy, uz), (E, id), ids, alive, stage written
    "k_b<charged>": 4 + 82 + 66,
}
B_SEC = 80                        # one stack record per secondary, written by the phase-B kernels


def load_ncu_profile(config):
    """ncu-derived constants of the committed capture of this workload (profiles/r2_ncu_config<k>.json, written by
    `python -m paper_2203_09467_b200.diagnostics.ncu_extract` from the .ncu-rep): DRAM bytes per launch and fp64
    instructions per unit of each kernel.  None when no capture of this workload is committed."""
    path = os.path.join(ROOT, "profiles", "r2_ncu_config%d.json" % config)
    try:
        with open(path) as f:
            d = json.load(f)
        d["file"] = os.path.relpath(path, ROOT)
        return d
    except (OSError, ValueError):
        return None


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--primaries", type=int, default=0, help="0 = the config's full count")
    ap.add_argument("--slots", type=int, default=0, help="track slots (0 = the config's: 2^20 for config 4)")
    ap.add_argument("--integrator", type=int, default=0, choices=[0, 1],
                    help="field integrator: 0 = RK4 with step doubling (what BASELINE's configs name; default), "
                         "1 = Dormand-Prince 5(4) (DESIGN.md R-INT)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--shard", action="store_true",
                    help="N > 1: ONE workload sharded by primaries over the ranks + final all-reduce of the tallies "
                         "(strong scaling) instead of N replicas (default, weak scaling)")
    return ap.parse_args()


def workload(args):
    desc, prim = W.get(args.config) if args.primaries <= 0 else W.get(args.config, args.primaries)
    if getattr(args, "slots", 0) > 0:
        desc = dict(desc, n_slots=int(args.slots))
    if getattr(args, "integrator", 0):
        desc = dict(desc, physics=dict(desc["physics"], integrator=int(args.integrator)))
    return desc, prim


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.proc.terminate()
        self.th.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[k] for r in self.rows if len(r) >= 7 for k in range(4) if r[3 + k].lower() == "active"})
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=reasons, samples=len(sm))


def oracle_run(desc, prim, n_sample, threads=None):
    """The oracle as it stands on the host cores: (track_steps, seconds, threads)."""
    from oracle import emo
    P = emo.Problem(desc)
    threads = threads or (os.cpu_count() or 1)
    sub = W.prefix(prim, n_sample)
    t0 = time.perf_counter()
    r = P.transport(sub, desc["seed"], n_threads=threads)
    dt = time.perf_counter() - t0
    return r["track_steps"], dt, threads


def oracle_sample_size(desc, prim, threads):
    """primaries whose oracle transport takes roughly 10-30 s: probe with a few, then scale"""
    n0 = min(len(prim["E"]), 4 * threads)
    steps, dt, _ = oracle_run(desc, prim, n0, threads)
    rate = max(n0 / max(dt, 1e-3), 1e-9)          # primaries / s
    return int(max(n0, min(len(prim["E"]), rate * 15.0)))


def replica_seed(base_seed, rank):
    """Replicas (N > 1): the same problem on every GPU with independent histories."""
    return base_seed + 1000 * rank


def reduce_over_ranks(times, counts, device):
    """The only exchange of an N-GPU run: max over ranks of the timed durations, sum over ranks of the work
    done.  Works on any torch.distributed backend (nccl on GPUs; gloo on CPU in the tests)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return [float(t) for t in times], [float(c) for c in counts]
    t = torch.tensor([float(x) for x in times], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor([float(x) for x in counts], device=device, dtype=torch.float64)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return t.tolist(), c.tolist()


def run_reference(args):
    """--impl reference: the oracle on the host cores; each step = a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    desc, prim = workload(args)
    threads = os.cpu_count() or 1
    n_s = oracle_sample_size(desc, prim, threads)
    for _ in range(args.warmup):
        oracle_run(desc, prim, max(1, n_s // 8), threads)
    tot_steps, tot_t = 0, 0.0
    for _ in range(args.steps):
        s, dt, _ = oracle_run(desc, prim, n_s, threads)
        tot_steps += s
        tot_t += dt
    v = tot_steps / tot_t
    sample = "first %d of %d primaries of %s per step" % (n_s, len(prim["E"]), desc["name"])
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": desc["name"], "primaries_per_step": n_s},
        "primaries_per_sec": n_s * args.steps / tot_t,
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2203_09467_b200 import emx
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the emx path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    desc, prim = workload(args)
    sharded = bool(args.shard) and world > 1
    seed = desc["seed"] if sharded else replica_seed(desc["seed"], rank)
    G = emx.Problem(desc)
    if sharded:      # contiguous ranges of the primaries, histories as in the unsharded run
        from paper_2203_09467_b200 import shard
        first, prim = shard.shard_primaries(prim, rank, world)
        G.set_primary_offset(first)
    n_prim = len(prim["E"])
    pdev = G.upload_primaries(prim)
    pinned = {k: torch.from_numpy(np.array(v, order="C")).pin_memory() for k, v in prim.items()}
    phost = {k: v.numpy() for k, v in pinned.items()}
    h2d = sum(v.numel() * v.element_size() for v in pinned.values())
    d2h = 8 * G.n_tally + 200

    G.set_profile(False)
    for _ in range(args.warmup):
        G.transport(pdev, seed)
    barrier()

    # ---- timed region: K steps, device-resident inputs (the loop runs as a CUDA graph)
    G.set_profile(False)
    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    tot = dict(steps=0, sec=0, launches=0, per_type=np.zeros(3), sec_type=np.zeros(3), iters=0)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        r = G.transport(pdev, seed)
        pr = G.profile()
        tot["steps"] += r["track_steps"]
        tot["per_type"] += r["steps"].astype(np.float64)
        sec = r["tracks"].astype(np.float64).copy()
        for k in range(3):
            sec[k] -= float((prim["ptype"] == k).sum())
        tot["sec_type"] += sec
        tot["launches"] += pr["launches"]
        tot["iters"] += r["iterations"]
        if sharded:  # the one exchange of the job: tallies, totals and counters summed over the ranks
            shard.all_reduce_results(r, G.read_step_hist(), "cuda")
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    clk = clocks.stop() if rank == 0 else None
    last = r
    # ---- kernel durations for the roofline: one profiled pass of the same step (kernel-by-kernel launches
    # bracketed by CUDA events on the launching stream; the graph path cannot be bracketed per kernel)
    G.set_profile(True)
    rp = G.transport(pdev, seed)
    prof = G.profile()
    prof_ms = rp["ms"]
    G.set_profile(False)

    # ---- e2e: host buffers in, tallies out, through the public entry point
    G.set_profile(False)
    barrier()
    t0 = time.perf_counter()
    e2e_steps = 0
    for _ in range(args.steps):
        r2 = G.transport_host(phost, seed)
        e2e_steps += r2["track_steps"]
    barrier()
    e2e_s = time.perf_counter() - t0

    (ms, e2e_s), (all_steps, all_e2e) = reduce_over_ranks([ms, e2e_s], [tot["steps"], e2e_steps], "cuda")
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = all_steps / (ms * 1e-3)
    # roofline of the dominant kernel.  The profiled pass brackets every step kernel of every iteration with CUDA
    # events; the dominant one is the kernel with the largest total.  Its algorithmic bytes = the track slots it
    # processed (counted by the kernel) x bytes per slot (B_STAGE).
    names = list(emx.STAGES)
    kms = prof["ms"]                      # ms of the profiled pass per kernel
    dom = max(names, key=lambda k: kms[k])
    lanes = float(prof["lanes"][dom])
    n_sec = float(tot["sec_type"].sum()) / args.steps
    alg_bytes = lanes * B_STAGE[dom]
    if dom.startswith("k_b"):
        nb = float(prof["lanes"]["k_b<gamma>"] + prof["lanes"]["k_b<charged>"])
        alg_bytes += n_sec * B_SEC * (lanes / max(nb, 1.0))
    k_s = kms[dom] * 1e-3
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        pass
    peak = float(peaks.get("hbm_gbs", 6650.0))
    ach = alg_bytes / k_s / 1e9 if k_s > 0 else 0.0
    n_launch = max(rp["iterations"], 1)
    ncu = load_ncu_profile(args.config)
    kn = (ncu or {}).get("kernels", {}).get(dom, {})
    all_bytes = sum(float(prof["lanes"][k]) * B_STAGE[k] for k in names) + n_sec * B_SEC
    hbm = {"bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
           "peak_source": "MEASURED_PEAKS.json hbm_gbs" if peaks else "fallback 6650 GB/s",
           "algorithmic_bytes_per_launch": alg_bytes / n_launch}
    common = {"kernel": dom, "traffic": kn.get("dram_bytes_per_launch"), "avg_launch_ms": kms[dom] / n_launch,
              "units_per_launch": lanes / n_launch,
              "kernel_ms_profiled_pass": {k: float(v) for k, v in kms.items()},
              "kernel_share_of_profiled_pass": float(kms[dom] / prof_ms), "profiled_pass_ms": prof_ms,
              "all_step_kernels": {"achieved_GBs": float(all_bytes / (kms["all_step_kernels"] * 1e-3) / 1e9)},
              "ncu_capture": None if ncu is None else {"file": ncu["file"], "build": ncu.get("build"), "measured_by_this_run": False}}
    # Which roof binds (profiles/r2_peaks.md): the propagation kernel is plain fp64 arithmetic -- its
    # track store is L2-resident and its DRAM traffic a few percent of the HBM peak -- so when it dominates the line
    # reports "alu": achieved = fp64 instructions per substep attempt (counted by ncu on the committed capture of this
    # workload, one flop each: the library is built without fused multiply-adds) x the attempts THIS run counted
    # / the kernel time THIS run measured; peak = the DMUL + DADD rate measured by diagnostics/peaks.cu on this pool's
    # B200.  The HBM and L2 figures stay beside it.  Without a committed capture, or for a memory-side kernel, the
    # line falls back to the HBM roof.
    pk = (ncu or {}).get("peaks", {})
    if (dom == "k_field" and kn.get("fp64_inst_per_attempt") and pk.get("fp64_tinst_per_s")
            and not desc["physics"].get("integrator", 0)):       # the committed capture counted the step-doubling kernel
        work = float(kn["fp64_inst_per_attempt"]) * float(prof["attempts"])
        roof = {"bound": "alu", "achieved": work / k_s / 1e12, "peak": pk["fp64_tinst_per_s"] / 1e12, "unit": "TFLOP/s",
                "frac": work / k_s / pk["fp64_tinst_per_s"],
                "peak_source": "profiles/r2_peaks.json fp64_tinst_per_s (DMUL + DADD thread-instructions/s, 1 flop each)",
                "fp64_flops_per_attempt": float(kn["fp64_inst_per_attempt"]),
                "attempts_per_launch": float(prof["attempts"]) / n_launch, "hbm": hbm}
    else:
        roof = dict(hbm)
    roof.update(common)
    if pk.get("l2_gbs"):
        roof["l2"] = {"achieved": ach, "peak": pk["l2_gbs"], "unit": "GB/s", "frac": ach / pk["l2_gbs"]}
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "strong" if sharded else "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": desc["name"], "primaries_per_step": n_prim, "n_slots": desc["n_slots"],
                      "queue_capacity": desc["queue_capacity"], "integrator": int(desc["physics"].get("integrator", 0)),
                      "parallelism": ("primaries sharded x%d + final all-reduce" if sharded else "replicas x%d") % world,
                      "l2": "inputs larger than L2: track store + stacks > 126 MB, every step re-reads the stacks"},
           "primaries_per_sec": n_prim * args.steps * world / (ms * 1e-3),
           "iterations_per_step": tot["iters"] / args.steps, "peak_live": last["peak_live"], "peak_queue": last["peak_queue"],
           "e2e": {"value": all_e2e / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
           "gpu_launches": int(tot["launches"]), "clocks": clk, "roofline": roof,
           "field_attempts_per_step": float(prof["attempts"])}
    if not args.no_cpu_baseline and world == 1:
        threads = os.cpu_count() or 1
        n_s = oracle_sample_size(desc, prim, threads)
        s, dt, _ = oracle_run(desc, prim, n_s, threads)
        out["cpu_baseline"] = {"value": s / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
                               "sample": "first %d of %d primaries of %s, %.1f s" % (n_s, n_prim, desc["name"], dt)}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
