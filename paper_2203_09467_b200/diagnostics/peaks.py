"""DIAGNOSTICS: build and run peaks.cu on the current GPU and record the two measured roofs under profiles/.

    python -m paper_2203_09467_b200.diagnostics.peaks [--json profiles/r2_peaks.json] [--md profiles/r2_peaks.md]
                                                      [--footprint-mb 95]

fp64 arithmetic peak (DFMA, and DMUL + DADD as libemx issues them under -fmad=false) in thread-instructions per
second, and the L2 read / copy bandwidth at the footprint of the track store.
Never used by the product path or the tests; bench.py reads the json it writes.
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile

HERE = os.path.dirname(os.path.abspath(__file__))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--json")
    ap.add_argument("--md")
    ap.add_argument("--footprint-mb", type=float, default=95.0)
    a = ap.parse_args()
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    with tempfile.TemporaryDirectory() as tmp:
        exe = os.path.join(tmp, "peaks")
        subprocess.check_call([nvcc, "-O3", "-gencode", "arch=compute_100a,code=sm_100a", os.path.join(HERE, "peaks.cu"), "-o", exe])
        runs = [json.loads(subprocess.check_output([exe, str(a.footprint_mb)], text=True)) for _ in range(3)]
    best = dict(runs[0])
    for r in runs[1:]:
        for k in ("fp64_dfma_tinst_per_s", "fp64_tinst_per_s", "fp64_tflops_fma", "l2_read_gbs", "l2_gbs"):
            best[k] = max(best[k], r[k])
    CMD = "python -m paper_2203_09467_b200.diagnostics.peaks " + " ".join(sys.argv[1:])
    best["command"] = CMD
    best["runs"] = runs
    if a.json:
        with open(a.json, "w") as f:
            json.dump(best, f, indent=1)
    lines = ["# Measured roofs of the step kernels on this B200 (round 2)", "",
             "Command (one B200 through gpurun):", "", "    " + CMD, "",
             "`peaks.cu`: 8 blocks of 256 threads per SM, 8 independent chains per thread, 4096 trips; L2: a buffer of "
             "%.0f MB (the track store of 2^20 slots) read / copied 20 times after one untimed pass.  Best of 3 runs." % a.footprint_mb, "",
             "| roof | measured |", "|---|---|",
             "| SMs, SM clock reported by the runtime | %d, %.0f MHz |" % (best["sms"], best["sm_clock_mhz"]),
             "| fp64 DFMA, thread-instructions / s | %.3e (%.1f TFLOP/s) |" % (best["fp64_dfma_tinst_per_s"], best["fp64_tflops_fma"]),
             "| fp64 DMUL + DADD (what -fmad=false issues), thread-instructions / s | %.3e |" % best["fp64_tinst_per_s"],
             "| L2 read bandwidth at %.0f MB | %.0f GB/s |" % (best["l2_footprint_mb"], best["l2_read_gbs"]),
             "| L2 copy bandwidth (read + written bytes) | %.0f GB/s |" % best["l2_gbs"], ""]
    text = "\n".join(lines)
    if a.md:
        with open(a.md, "w") as f:
            f.write(text)
    print(text)
    return 0


if __name__ == "__main__":
    sys.exit(main())
