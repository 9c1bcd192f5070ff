"""Timeline of the iteration graph: when every kernel node of an iteration starts and ends on the GPU.

    python -m paper_2203_09467_b200.timeline [--config 4] [--primaries 100000] [--first 2500] [--rows 6]

CUDA events cannot look inside a graph launch and a profiler serialises the parallel branches, so this
diagnostic builds a second copy of the library with -DEMX_TIMELINE (csrc/emx_transport.cu: every block
stamps %globaltimer at its start and end, reduced per node with atomics) into a temporary directory, runs one
transport in the normal graph mode and prints, for 64 iterations from --first on: first block start / last
block end per node, the mean durations and gaps, and the mean time blocks of each kernel were resident.
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

HERE = os.path.dirname(os.path.abspath(__file__))
NODES = ["k_plan", "k_fill", "k_move", "A gamma", "A e-", "A e+", "B gamma", "B e-", "B e+"]
N_IT = 64


def build_instrumented(first, out_dir):
    from . import build as B
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
    os.environ["EMX_LIB_PATH"] = lib_path
    from . import emx, workloads as W
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
    gaps = [("k_plan end -> k_fill start", st[sel, 1] - en[sel, 0]), ("k_fill end -> k_move start", st[sel, 2] - en[sel, 1]),
            ("k_move end -> A e+ start", st[sel, 5] - en[sel, 2]), ("k_move end -> A e- start", st[sel, 4] - en[sel, 2]),
            ("k_move end -> A gamma start", st[sel, 3] - en[sel, 2]), ("A e+ end -> B e+ start", st[sel, 8] - en[sel, 5]),
            ("A e- end -> B e- start", st[sel, 7] - en[sel, 4]), ("A gamma end -> B gamma start", st[sel, 6] - en[sel, 3])]
    print("\n| gap | mean us |")
    print("|---|---|")
    for name, g in gaps:
        print("| %s | %.1f |" % (name, g.mean() / 1e3))
    return 0


if __name__ == "__main__":
    sys.exit(main())
