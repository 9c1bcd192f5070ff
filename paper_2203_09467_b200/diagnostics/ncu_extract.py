"""DIAGNOSTICS: turn an Nsight Compute report of the step kernels into the summaries kept under profiles/.

    python -m paper_2203_09467_b200.diagnostics.ncu_extract REPORT.ncu-rep [--md OUT.md] [--json OUT.json]
                                                            [--config 4] [--build TEXT] [--command TEXT]
                                                            [--fp64-csv FIELD.csv --fp64-json FIELD.json]

Reads the report with `ncu -i REPORT --page raw --csv` (ncu must be on PATH; no GPU needed) and writes
  --md    one table, a column per captured launch: duration, grid, registers, warp instructions, lanes active per
          instruction, issue slots busy, warps active, fp64 pipe, DRAM / L2 / L1 traffic and hit rates, the top
          stall reasons, fp64 instruction counts;
  --json  per kernel: DRAM bytes per launch, fp64 thread-instructions per launch, duration -- what bench.py quotes
          as `roofline.traffic` and uses for `roofline.alu` (it divides the fp64 instructions of k_field by the
          substep attempts of the captured launch, which the caller passes with --attempts, or leaves them per
          launch).  The measured peaks of profiles/r2_peaks.json, if present, are copied in under "peaks".
  --fp64-csv / --fp64-json  the two outputs of the diagnostics/field_work.py pass (ncu's per-launch counter list and
          the run's attempt count): the fp64 instructions of ALL k_field launches of that run divided by its substep
          attempts give `fp64_inst_per_attempt` of k_field, which is what `roofline.alu` multiplies with the attempts
          bench.py counts live.
Never used by the product path or the tests.
"""
import argparse
import csv
import json
import os
import subprocess
import sys

SHORT = [("k_a<0", "k_a<gamma>"), ("k_a<(int)0", "k_a<gamma>"), ("k_a<1", "k_a<charged>"), ("k_a<(int)1", "k_a<charged>"),
         ("k_a0", "k_a0"), ("k_a2", "k_a2"), ("k_field", "k_field"), ("k_b<0", "k_b<gamma>"), ("k_b<(int)0", "k_b<gamma>"),
         ("k_b<1", "k_b<charged>"), ("k_b<(int)1", "k_b<charged>"), ("k_plan", "k_plan"), ("k_fill", "k_fill"), ("k_move", "k_move")]

ROWS = [
    ("gpu__time_duration.sum", "duration (us)", 1e-3),
    ("launch__grid_size", "grid (blocks of 128)", 1),
    ("launch__registers_per_thread", "registers / thread", 1),
    ("launch__occupancy_limit_registers", "blocks / SM allowed by registers", 1),
    ("smsp__inst_executed.sum", "warp instructions (M)", 1e-6),
    ("smsp__thread_inst_executed_per_inst_executed.ratio", "lanes active per instruction (of 32)", 1),
    ("smsp__issue_active.avg.pct_of_peak_sustained_active", "issue slots busy (%)", 1),
    ("sm__warps_active.avg.pct_of_peak_sustained_active", "warps active (% of 64 per SM)", 1),
    ("sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active", "fp64 pipe (% of peak)", 1),
    ("smsp__sass_thread_inst_executed_op_dfma_pred_on.sum", "DFMA thread-instructions (M)", 1e-6),
    ("smsp__sass_thread_inst_executed_op_dmul_pred_on.sum", "DMUL thread-instructions (M)", 1e-6),
    ("smsp__sass_thread_inst_executed_op_dadd_pred_on.sum", "DADD thread-instructions (M)", 1e-6),
    ("dram__bytes_read.sum", "DRAM read (MB)", 1e-6),
    ("dram__bytes_write.sum", "DRAM written (MB)", 1e-6),
    ("gpu__dram_throughput.avg.pct_of_peak_sustained_elapsed", "DRAM throughput (% of peak)", 1),
    ("lts__t_bytes.sum", "L2 traffic (MB)", 1e-6),
    ("lts__t_sector_hit_rate.pct", "L2 hit (%)", 1),
    ("l1tex__t_sector_hit_rate.pct", "L1 hit (%)", 1),
    ("l1tex__data_pipe_lsu_wavefronts_mem_lg.sum", "L1 wavefronts, global + local (M)", 1e-6),
    ("l1tex__t_requests_pipe_lsu_mem_global_op_ld.sum", "global load requests = warp-level load instructions (M)", 1e-6),
    ("l1tex__t_sectors_pipe_lsu_mem_global_op_ld.sum", "global load sectors of 32 B (M)", 1e-6),
    ("l1tex__t_requests_pipe_lsu_mem_global_op_st.sum", "global store requests (M)", 1e-6),
    ("l1tex__t_sectors_pipe_lsu_mem_global_op_st.sum", "global store sectors (M)", 1e-6),
    ("l1tex__t_requests_pipe_lsu_mem_local_op_ld.sum", "local (spill) load requests (M)", 1e-6),
    ("l1tex__t_requests_pipe_lsu_mem_local_op_st.sum", "local (spill) store requests (M)", 1e-6),
    ("l1tex__data_pipe_lsu_wavefronts_mem_shared.sum", "shared-memory wavefronts (M)", 1e-6),
    ("smsp__inst_executed_op_global_ld.sum", "global load instructions (M)", 1e-6),
    ("smsp__inst_executed_op_global_st.sum", "global store instructions (M)", 1e-6),
    ("smsp__inst_executed_op_local_ld.sum", "local (spill) load instructions (M)", 1e-6),
    ("smsp__inst_executed_op_local_st.sum", "local (spill) store instructions (M)", 1e-6),
    ("smsp__average_warps_issue_stalled_long_scoreboard_per_issue_active.ratio", "stall long_scoreboard (cycles / issue)", 1),
    ("smsp__average_warps_issue_stalled_wait_per_issue_active.ratio", "stall wait", 1),
    ("smsp__average_warps_issue_stalled_short_scoreboard_per_issue_active.ratio", "stall short_scoreboard", 1),
    ("smsp__average_warps_issue_stalled_no_instruction_per_issue_active.ratio", "stall no_instruction", 1),
    ("smsp__average_warps_issue_stalled_branch_resolving_per_issue_active.ratio", "stall branch_resolving", 1),
    ("smsp__average_warps_issue_stalled_math_pipe_throttle_per_issue_active.ratio", "stall math_pipe_throttle", 1),
    ("smsp__average_warps_issue_stalled_not_selected_per_issue_active.ratio", "stall not_selected", 1),
    ("smsp__average_warps_issue_stalled_lg_throttle_per_issue_active.ratio", "stall lg_throttle", 1),
]


def short_name(full):
    f = full.replace("void ", "").replace("emx::", "")
    for key, name in SHORT:
        if f.startswith(key):
            return name
    return f.split("(")[0]


def read_raw(report):
    out = subprocess.run(["ncu", "-i", report, "--page", "raw", "--csv"], capture_output=True, text=True)
    if out.returncode != 0:
        sys.exit("ncu failed: " + out.stderr[-400:])
    rows = list(csv.reader(out.stdout.splitlines()))
    hdr, units = rows[0], rows[1]
    # the raw page scales every column to a unit of its own choosing: bring times to ns and sizes to bytes
    to_base = {"ns": 1.0, "us": 1e3, "ms": 1e6, "s": 1e9, "nsecond": 1.0, "usecond": 1e3, "msecond": 1e6, "second": 1e9,
               "byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
    data = []
    for r in rows[2:]:
        r = list(r)
        for k, u in enumerate(units):
            if u in to_base and to_base[u] != 1.0:
                v = num(r[k])
                if v is not None:
                    r[k] = repr(v * to_base[u])
        data.append(r)
    return hdr, data


def num(v):
    try:
        return float(v.replace(",", ""))
    except ValueError:
        return None


def per_attempt(csv_path, json_path):
    """sums of the counters over every k_field launch of the field_work.py run, per substep attempt of that run"""
    with open(json_path) as f:
        run = json.loads(f.read().strip().splitlines()[-1])
    with open(csv_path) as f:
        lines = [ln for ln in f if not ln.startswith("==")]
    rows = list(csv.reader(lines))
    hdr = rows[0]
    ik, im, iv = hdr.index("Kernel Name"), hdr.index("Metric Name"), hdr.index("Metric Value")
    tot, launches = {}, set()
    for r in rows[1:]:
        if len(r) <= iv or "k_field" not in r[ik]:
            continue
        v = num(r[iv])
        if v is None:
            continue
        tot[r[im]] = tot.get(r[im], 0.0) + v
        launches.add(r[0])
    fp64 = sum(tot.get(m, 0.0) for m in ("smsp__sass_thread_inst_executed_op_dfma_pred_on.sum",
                                         "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum",
                                         "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum"))
    att = float(run["attempts"])
    return {"fp64_inst_per_attempt": fp64 / att, "thread_inst_per_attempt": tot.get("smsp__thread_inst_executed.sum", 0.0) / att,
            "warp_inst_per_attempt": tot.get("smsp__inst_executed.sum", 0.0) / att,
            "per_attempt_from": {"run": run, "k_field_launches": len(launches), "fp64_thread_inst": fp64}}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("report")
    ap.add_argument("--md")
    ap.add_argument("--json")
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--build", default="")
    ap.add_argument("--command", default="")
    ap.add_argument("--attempts", type=float, default=0.0, help="substep attempts of the captured k_field launch")
    ap.add_argument("--title", default="")
    ap.add_argument("--fp64-csv")
    ap.add_argument("--fp64-json")
    a = ap.parse_args()
    hdr, data = read_raw(a.report)
    idx = {h: i for i, h in enumerate(hdr)}
    names = [short_name(r[idx["Kernel Name"]]) for r in data]
    lines = []
    if a.title:
        lines += ["# " + a.title, ""]
    if a.command:
        lines += ["Command (one B200 through gpurun; the same command had exited 0 without ncu directly before):", "",
                  "    " + a.command, ""]
    lines += ["Read with `python -m paper_2203_09467_b200.diagnostics.ncu_extract %s`." % os.path.basename(a.report), ""]
    lines.append("| metric | " + " | ".join(names) + " |")
    lines.append("|---|" + "---|" * len(names))
    for metric, label, scale in ROWS:
        if metric not in idx:
            continue
        vals = []
        for r in data:
            v = num(r[idx[metric]])
            if v is None:
                vals.append(r[idx[metric]])
            else:
                v *= scale
                vals.append("%.0f" % v if abs(v) >= 1000 or float(v).is_integer() else ("%.1f" % v if abs(v) >= 10 else "%.2f" % v))
        lines.append("| %s | " % label + " | ".join(vals) + " |")
    text = "\n".join(lines) + "\n"
    if a.md:
        with open(a.md, "w") as f:
            f.write(text)
    else:
        print(text)
    if a.json:
        kernels = {}
        for r, name in zip(data, names):
            g = lambda m: (num(r[idx[m]]) if m in idx else None)
            fp64 = sum(g(m) or 0.0 for m in ("smsp__sass_thread_inst_executed_op_dfma_pred_on.sum",
                                              "smsp__sass_thread_inst_executed_op_dmul_pred_on.sum",
                                              "smsp__sass_thread_inst_executed_op_dadd_pred_on.sum"))
            k = {"duration_us": (g("gpu__time_duration.sum") or 0.0) * 1e-3,
                 "registers": g("launch__registers_per_thread"),
                 "dram_bytes_per_launch": (g("dram__bytes_read.sum") or 0.0) + (g("dram__bytes_write.sum") or 0.0),
                 "fp64_thread_inst_per_launch": fp64,
                 "warp_inst_per_launch": g("smsp__inst_executed.sum"),
                 "fp64_pipe_pct": g("sm__inst_executed_pipe_fp64.avg.pct_of_peak_sustained_active"),
                 "issue_active_pct": g("smsp__issue_active.avg.pct_of_peak_sustained_active"),
                 "warps_active_pct": g("sm__warps_active.avg.pct_of_peak_sustained_active"),
                 "lanes_per_inst": g("smsp__thread_inst_executed_per_inst_executed.ratio")}
            if name == "k_field" and a.attempts > 0:
                k["attempts_in_launch"] = a.attempts
                k["fp64_inst_per_attempt"] = fp64 / a.attempts
            kernels[name] = k
        if a.fp64_csv and a.fp64_json and "k_field" in kernels:
            kernels["k_field"].update(per_attempt(a.fp64_csv, a.fp64_json))
        out = {"config": a.config, "build": a.build, "report": os.path.basename(a.report), "command": a.command, "kernels": kernels}
        peaks = os.path.join(os.path.dirname(os.path.abspath(a.json)), "r2_peaks.json")
        if os.path.exists(peaks):
            with open(peaks) as f:
                out["peaks"] = json.load(f)
        with open(a.json, "w") as f:
            json.dump(out, f, indent=1)
    return 0


if __name__ == "__main__":
    sys.exit(main())
