"""The paper's verification problem on the GPU: six concentric cylinders, 100 000 isotropic
1 GeV photons, and the two observables the paper compares -- cumulative energy deposition along z and steps per
track by particle type -- plus the loop diagnostics of its Fig. 5 (tracks in flight, queued initializers).

    python -m paper_2203_09467_b200.verification [--primaries 100000]

Prints markdown.  CUDA path only (the comparison with the CPU oracle is tests/test_gpu_parity.py, config 5).
"""
import argparse
import sys

import numpy as np


def bin_lower_edges(nhist):
    """lower edge of every steps-per-track bin (include/emx.h: EMX_NHIST)"""
    return np.array([b if b < 16 else (4 + (b - 16) % 4) << ((b - 16) // 4 + 2) for b in range(nhist)], dtype=np.int64)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--primaries", type=int, default=100000)
    a = ap.parse_args()
    from . import emx, workloads as W
    desc, prim = W.get(5, a.primaries)
    G = emx.Problem(desc)
    pd = G.upload_primaries(prim)
    G.transport(pd, desc["seed"])                               # warm-up
    r = G.transport(pd, desc["seed"])
    hist = G.read_step_hist()
    log = G.iteration_log()
    n = a.primaries
    print("# %s: %d primaries of 1 GeV, %.1f ms, %.3g track-steps/s, %d iterations" %
          (desc["name"], n, r["ms"], r["track_steps"] / (r["ms"] * 1e-3), r["iterations"]))
    closure = abs(r["edep"].sum() + r["escaped"] + r["looper"] - r["E_in"]) / r["E_in"]
    print("\nenergy: deposited %.4f, escaped %.4f of the %.4g MeV injected; closure %.1e; stalls %d" %
          (r["edep"].sum() / r["E_in"], r["escaped"] / r["E_in"], r["E_in"], closure, r["stalls"]))
    print("\n## cumulative energy deposition along z (fraction of the deposited energy, 28 slabs of 50 cm)\n")
    cum = np.cumsum(r["edep"]) / r["edep"].sum()
    nz = len(cum)
    z_hi = [-700.0 + (k + 1) * 1400.0 / nz for k in range(nz)]
    print("| z below (cm) | " + " | ".join("%.0f" % z for z in z_hi) + " |")
    print("|---|" + "---|" * nz)
    print("| cumulative | " + " | ".join("%.4f" % c for c in cum) + " |")
    print("\n## steps per track by particle type\n")
    lo = bin_lower_edges(hist.shape[1])
    print("| type | tracks | steps | mean steps per track | median bin | 99th percentile bin | longest bin |")
    print("|---|---|---|---|---|---|---|")
    for k, name in enumerate(("gamma", "e-", "e+")):
        h = hist[k].astype(np.float64)
        tot = h.sum()
        if tot == 0:
            continue
        c = np.cumsum(h) / tot
        med, p99 = int(np.searchsorted(c, 0.5)), int(np.searchsorted(c, 0.99))
        last = int(np.flatnonzero(h)[-1])
        print("| %s | %d | %d | %.2f | >= %d | >= %d | >= %d |" %
              (name, int(r["tracks"][k]), int(r["steps"][k]), r["steps"][k] / max(tot, 1.0), lo[med], lo[p99], lo[last]))
    print("\n## loop diagnostics (Fig. 5: tracks in flight and queued initializers per step iteration)\n")
    it = np.linspace(0, len(log) - 1, 12).astype(int)
    print("| iteration | " + " | ".join(str(int(i)) for i in it) + " |")
    print("|---|" + "---|" * len(it))
    print("| tracks in flight | " + " | ".join(str(int(log[i, 0])) for i in it) + " |")
    print("| queued initializers | " + " | ".join(str(int(log[i, 1])) for i in it) + " |")
    print("\npeak tracks in flight %d, peak queue %d records" % (r["peak_live"], r["peak_queue"]))
    return 0


if __name__ == "__main__":
    sys.exit(main())
