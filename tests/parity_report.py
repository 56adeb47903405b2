#!/usr/bin/env python3
"""Writes the parity record of the end-to-end protocols (P-A, P-B with its control, P-D, and the
batch-shape tests) as a markdown table.

    python tests/parity_report.py [--run] [--out profiles/r03_parity.md]

--run first executes the GPU parity tests that produce the records (`pytest -m gpu -k ...` on a CUDA box); without it
the script only collates what those tests left under gpurun_out/parity/*.json.  Every number comes from
tests/test_gpu_engine.py: GPU (through the C ABI) vs oracle/ on the same seeded inputs, judged by
oracle/compare.py::compare_commits; `control` = oracle/control.py (the oracle with bf16 rounding at the fast path's
rounding points + 1e-6 relative noise) judged the same way on the same steps.
"""
import argparse
import glob
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SELECT = "teacher_forced or free_running or precise or batch_shape or full_depth"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--run", action="store_true")
    ap.add_argument("--out", default=os.path.join(ROOT, "profiles", "r03_parity.md"))
    args = ap.parse_args()
    cmd = [sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_gpu_engine.py"), "-q", "-m", "gpu", "-k", SELECT]
    if args.run:
        subprocess.run(cmd, check=True, cwd=ROOT)
    recs = sorted(glob.glob(os.path.join(ROOT, "gpurun_out", "parity", "*.json")))
    if not recs:
        raise SystemExit("no records under gpurun_out/parity/: run with --run on a CUDA box")
    lines = ["# Round-3 parity record (GPU through the C ABI vs the fp64 oracle)", "",
             "Command: `python tests/parity_report.py --run` (runs `" + " ".join(["python", "-m", "pytest", "tests/test_gpu_engine.py", "-q", "-m", "gpu", "-k", f"'{SELECT}'"]) + "`",
             "on the B200 box and collates `gpurun_out/parity/*.json`).", "",
             "Columns: steps compared; commit lists identical (`exact`); per-position differences inside north_star's 1e-3 band",
             "(`excluded`, reading G13); differences outside it (`mismatch`); the same three for the CONTROL (fp64 oracle with",
             "bf16 rounding at the fast path's rounding points + 1e-6 noise) on the same steps; `unexplained` = GPU mismatches",
             "that remain when the band is widened to 3 x the CONTROL's largest confidence error + 1e-3 (P-B rows; asserted 0;",
             "batch-shape rows have no control and use 2 x the step's measured error); max |conf_gpu - conf_oracle| over block",
             "rows; max per-row relative hidden (L2 over the row) / lse error (north_star bound 2e-2; `n/a` = not compared);",
             "median oracle gap between the best and second-best MASK confidence on steps decided by the at-least-one rule.", "",
             "| record | steps | exact | excluded | mismatch | control exact / excluded / mismatch | unexplained | max conf err (control) | max hidden | max lse | median gap |",
             "|---|---|---|---|---|---|---|---|---|---|---|"]
    for r in recs:
        d = json.load(open(r))
        c = d.get("control", {})
        has_c = (c.get("exact", 0) + c.get("excluded", 0) + c.get("mismatch", 0)) > 0
        gap = d.get("median_gap")
        lines.append("| {} | {} | {} | {} | {} | {} | {} | {:.2e}{} | {} | {:.2e} | {} |".format(
            os.path.basename(r)[:-5], d["steps"], d["exact"], d["excluded"], d["mismatch"],
            "{} / {} / {}".format(c["exact"], c["excluded"], c["mismatch"]) if has_c else "-", d.get("unexplained", 0),
            d.get("max_conf_err", 0.0), " ({:.2e})".format(c["max_conf_err"]) if has_c else "",
            "{:.2e}".format(d["max_hid"]) if d.get("max_hid") is not None else "n/a", d["max_lse"],
            "{:.2e}".format(gap) if gap is not None else "-"))
    lines += ["", "P-A / P-D rows are FREE-RUNNING (the GPU's own commits feed its next step; a mismatch fails the test);",
              "P-B rows are teacher-forced per step and assert: confidence error <= 1.5 x the control's largest (and <= 5e-2);",
              "unexplained == 0; mismatch <= control mismatch + (0 below 16 steps, else 1) and <= the round-2 count of the record",
              "(tests/test_gpu_engine.py GOLDEN_MISMATCH); hidden and lse within 2e-2 per row.  Batch-shape rows compare the hidden",
              "states of a debug-dump re-run of the same step whose lse and commits reproduce the production (graph + PDL) step's.", ""]
    os.makedirs(os.path.dirname(args.out), exist_ok=True)
    open(args.out, "w").write("\n".join(lines))
    print("\n".join(lines))


if __name__ == "__main__":
    main()
