"""DIAGNOSTICS: a small transport launched kernel by kernel, for counting instructions per substep attempt with ncu.

    ncu --metrics smsp__sass_thread_inst_executed_op_dfma_pred_on.sum,smsp__sass_thread_inst_executed_op_dmul_pred_on.sum,\
smsp__sass_thread_inst_executed_op_dadd_pred_on.sum,smsp__thread_inst_executed.sum,smsp__inst_executed.sum \
        --clock-control none -k regex:k_field --csv --log-file OUT.csv \
        python -m paper_2203_09467_b200.diagnostics.field_work [--config 4] [--primaries 48] > OUT.json

(--stage-faces 1 switches the shared-memory copy of the face table on: the before / after pair of profiles/r2_staging.md.)
Runs ONE transport of the workload on the flat path (emx_set_profile(2): every kernel a launch of its own, which a
profiler can see; the results are those of the graph path, tests/test_gpu_parity.py) and prints one JSON object with
the substep attempts and the slots the propagation kernel processed.  The counts are deterministic, so the sum of a
counter over all k_field launches of the run divided by `attempts` is that counter per attempt; ncu_extract.py
(--fp64-csv / --fp64-json) does the division.  Never used by the product path or the tests.
"""
import argparse
import json
import sys


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--primaries", type=int, default=48)
    ap.add_argument("--stage-faces", type=int, default=0, help="1: k_field stages the face table in shared memory (emx_schedule)")
    ap.add_argument("--stage-tables", type=int, default=0, help="1: k_a<gamma> stages the photon tables in shared memory")
    a = ap.parse_args()
    from .. import emx, workloads as W
    desc, prim = W.get(a.config, a.primaries)
    G = emx.Problem(desc)
    pd = G.upload_primaries(prim)
    G.set_profile(2)
    if a.stage_faces:
        G.set_schedule(stage_faces=True)
    if a.stage_tables:
        G.set_schedule(stage_tables=True)
    r = G.transport(pd, desc["seed"])
    p = G.profile()
    print(json.dumps({"config": a.config, "primaries": a.primaries, "workload": desc["name"], "iterations": int(r["iterations"]),
                      "track_steps": int(r["track_steps"]), "attempts": float(p["attempts"]),
                      "k_field_slots": float(p["lanes"]["k_field"]), "stage_faces": a.stage_faces, "stage_tables": a.stage_tables, "ms": float(r["ms"]),
                      "k_field_ms": float(p["ms"].get("k_field", 0.0))}))
    return 0


if __name__ == "__main__":
    sys.exit(main())
