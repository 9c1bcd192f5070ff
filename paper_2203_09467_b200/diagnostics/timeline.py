"""DIAGNOSTICS: timeline of the iteration graph -- when every kernel node of an iteration starts and ends on the GPU.

    python -m paper_2203_09467_b200.diagnostics.timeline [--config 4] [--primaries 100000] [--first 2500] [--rows 6]

CUDA events cannot look inside a graph launch and a profiler serialises the parallel branches, so this
diagnostic builds a second copy of the library with -DEMX_TIMELINE (csrc/emx_diag.h: every block stamps
%globaltimer at its start and end, reduced per node with atomics) into a temporary directory, points the
binding at it, runs one transport in the normal graph mode and prints, for 64 iterations from --first on: first
block start / last block end per node, the mean durations and gaps, the mean time blocks of each kernel were
resident, and the share of the SMs' block slots that was occupied over the iteration.
The stamps cost time (the atomics of the many-block refill kernels most of all): use the numbers for the
structure of an iteration, not for its absolute length.  Never used by the product path or the tests.
"""
import argparse
import ctypes as C
import os
import subprocess
import sys
import tempfile

import numpy as np

NODES = ["k_plan", "k_fill", "k_move", "k_a<gamma>", "k_a<charged> / k_a2", "k_b<gamma>", "k_b<charged>", "k_a0", "k_field"]
STAGE_OF_NODE = {3: "k_a<gamma>", 5: "k_b<gamma>", 6: "k_b<charged>", 7: "k_a0", 8: "k_field"}
N_IT = 64


def build_instrumented(first, out_dir):
    from .. import build as B
    lib = os.path.join(out_dir, "libemx_timeline.so")
    srcs = [os.path.join(B.CSRC, s) for s in B.SRC]
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    subprocess.check_call([nvcc] + B.FLAGS + ["-DEMX_TIMELINE", "-DEMX_TL_FIRST=%d" % first, "-o", lib] + srcs)
    return lib


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--primaries", type=int, default=100000)
    ap.add_argument("--first", type=int, default=2500, help="first iteration recorded")
    ap.add_argument("--rows", type=int, default=6, help="iterations printed in full")
    a = ap.parse_args()
    tmp = tempfile.mkdtemp(prefix="emx_timeline_")
    lib_path = build_instrumented(a.first, tmp)
    from .. import emx, workloads as W
    emx.LIB_PATH = lib_path                             # the instrumented copy instead of the product library
    desc, prim = W.get(a.config, a.primaries)
    G = emx.Problem(desc)
    pd = G.upload_primaries(prim)
    G.transport(pd, desc["seed"])                       # warm-up
    L = C.CDLL(lib_path)
    buf = np.zeros((N_IT, 9, 4), dtype=np.uint64)
    L.emx_debug_timeline(C.c_void_p(0), 1)
    r = G.transport(pd, desc["seed"])
    L.emx_debug_timeline(buf.ctypes.data_as(C.c_void_p), 0)
    log = G.iteration_log()
    print("config %d, %d primaries: %.1f ms, %d iterations (instrumented build)" % (a.config, a.primaries, r["ms"], r["iterations"]))
    st = (~buf[..., 0]).astype(np.int64)
    en = buf[..., 1].astype(np.int64)
    ok = buf[:, 0, 3] > 0
    if ok.sum() < 3:
        print("fewer than 3 of the iterations %d..%d ran: choose another --first" % (a.first, a.first + N_IT))
        return 1
    its = np.flatnonzero(ok)
    t0 = st[its[0], 0]
    print("\nfirst block start - last block end per node, microseconds from the start of iteration %d" % (a.first + its[0]))
    print("| iteration | live tracks | " + " | ".join(NODES) + " |")
    print("|---|---|" + "---|" * 9)
    for it in its[:a.rows]:
        live = int(log[a.first + it, 0]) if a.first + it < len(log) else -1
        cells = ["%.1f - %.1f" % ((st[it, k] - t0) / 1e3, (en[it, k] - t0) / 1e3) for k in range(9)]
        print("| %d | %d | " % (a.first + it, live) + " | ".join(cells) + " |")
    sel = its[:-1]
    dur = (en[sel] - st[sel]) / 1e3
    nb = buf[sel, :, 3].astype(np.float64)
    resident = buf[sel, :, 2].astype(np.float64) / 1e3 / np.maximum(nb, 1)
    period = np.diff(st[its, 0]) / 1e3
    print("\nmeans over %d iterations (microseconds); iteration period %.1f" % (len(sel), period.mean()))
    print("| node | blocks | first start to last end | mean time a block was resident |")
    print("|---|---|---|---|")
    for k in range(9):
        print("| %s | %.0f | %.1f | %.1f |" % (NODES[k], nb[:, k].mean(), dur[:, k].mean(), resident[:, k].mean()))
    field = bool(np.any(nb[:, 8] > 0))
    chain = [7, 8, 4, 6] if field else [4, 6]
    gaps = [("k_plan end -> k_fill start", st[sel, 1] - en[sel, 0]), ("k_fill end -> k_move start", st[sel, 2] - en[sel, 1]),
            ("k_move end -> %s start" % NODES[chain[0]], st[sel, chain[0]] - en[sel, 2]),
            ("k_move end -> k_a<gamma> start", st[sel, 3] - en[sel, 2]),
            ("k_a<gamma> end -> k_b<gamma> start", st[sel, 5] - en[sel, 3])]
    for x, y in zip(chain[:-1], chain[1:]):
        gaps.append(("%s end -> %s start" % (NODES[x], NODES[y]), st[sel, y] - en[sel, x]))
    print("\n| gap | mean us |")
    print("|---|---|")
    for name, g in gaps:
        print("| %s | %.1f |" % (name, g.mean() / 1e3))
    # occupancy of the SMs' block slots: a resident block of kernel k holds 1 / (blocks per SM of k) of an SM
    import torch
    n_sm = torch.cuda.get_device_properties(0).multi_processor_count
    share = 0.0
    for k in range(3, 9):
        bps = max(1.0, nb[:, k].mean() / n_sm)
        share += (buf[sel, k, 2].astype(np.float64).mean() / 1e3) / bps
    print("\nblock-slot occupancy of the step kernels: %.1f %% of (iteration period x %d SMs); refill prefix %.1f us" %
          (100.0 * share / (period.mean() * n_sm), n_sm, (en[sel, 2] - st[sel, 0]).mean() / 1e3))
    return 0


if __name__ == "__main__":
    sys.exit(main())
