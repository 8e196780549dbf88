"""Turns gpurun_out/parity_stats.jsonl (written by the -m gpu tests through helpers.record_stats) into the
markdown table kept in profiles/r02_parity_stats.md:  python tests/parity_table.py > table.md"""
import json
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
path = sys.argv[1] if len(sys.argv) > 1 else os.path.join(ROOT, "gpurun_out", "parity_stats.jsonl")
seen = {}
for line in open(path):
    r = json.loads(line)
    seen[r["test"]] = r


def f(r, k, fmt):
    return fmt % r[k] if k in r else ""


print("| test | plane points | worst abs err / max | noise-floor ratio (A23) | plain ratio, P<30 | common | only GPU | "
      "only oracle | outside strict window | widest window / T_h | worst rel power | flags checked |")
print("|---|---|---|---|---|---|---|---|---|---|---|---|")
for k, r in seen.items():
    print("|", k, "|", r.get("points", ""), "|", f(r, "worst_over_max", "%.2e"), "|", f(r, "noise_floor_ratio", "%.3f"), "|",
          f(r, "plain_ratio_P_lt_30", "%.3g"), "|", r.get("common", ""), "|", r.get("only_gpu", ""), "|", r.get("only_orc", ""),
          "|", r.get("outside_strict", ""), "|", f(r, "worst_window", "%.2e"), "|", f(r, "worst_rel", "%.2e"), "|",
          r.get("flags_checked", ""), "|")
