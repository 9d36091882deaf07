"""Writes profiles/parity_r2.md from gpurun_out/parity_r2.jsonl, the log tests/parity_util.compare() appends to during
`python -m pytest tests -m gpu` on the GPU box (every CUDA-vs-oracle comparison: achieved rel-L2 and largest
element-wise deviation, in units of the tolerance).

    python tests/parity_report.py [gpurun_out/parity_r2.jsonl] [profiles/parity_r2.md]
"""
import json
import os
import sys
from collections import OrderedDict

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def main():
    src = sys.argv[1] if len(sys.argv) > 1 else os.path.join(ROOT, "gpurun_out", "parity_r2.jsonl")
    dst = sys.argv[2] if len(sys.argv) > 2 else os.path.join(ROOT, "profiles", "parity_r2.md")
    groups = OrderedDict()
    for line in open(src):
        line = line.strip()
        if not line:
            continue
        r = json.loads(line)
        g = groups.setdefault(r["label"], {"n": 0, "l2": 0.0, "inf": 0.0, "tol": set(), "elements": 0})
        g["n"] += 1
        g["l2"] = max(g["l2"], r["rel_l2"] / r["tol"])
        g["inf"] = max(g["inf"], r["max_abs_over_max_ref"] / r["tol"])
        g["tol"].add(r["tol"])
        g["elements"] = max(g["elements"], r["elements"])
    out = ["# GPU-vs-oracle parity, achieved errors (round 2)", "",
           "Written by `python tests/parity_report.py` from the log of `python -m pytest tests -m gpu -q` on a B200",
           "(`tests/parity_util.compare` appends one record per comparison). Errors are in units of the tolerance of",
           "`BASELINE.json` (`north_star`): 1e-12 for complex128, 1e-5 for complex64; both bounds of every test are 1.0.", "",
           "| comparison (label in the tests) | comparisons | tolerances | largest output (elements) | worst rel-L2 / tol | worst max-abs / (tol max\\|ref\\|) |",
           "|---|---|---|---|---|---|"]
    worst_l2 = worst_inf = 0.0
    for label, g in groups.items():
        tols = ", ".join(f"{t:g}" for t in sorted(g["tol"]))
        out.append(f"| {label} | {g['n']} | {tols} | {g['elements']} | {g['l2']:.3g} | {g['inf']:.3g} |")
        worst_l2, worst_inf = max(worst_l2, g["l2"]), max(worst_inf, g["inf"])
    out += ["", f"Worst over all {sum(g['n'] for g in groups.values())} comparisons: rel-L2 {worst_l2:.3g} tol, "
            f"max-abs {worst_inf:.3g} tol-units."]
    open(dst, "w").write("\n".join(out) + "\n")
    print(dst)


if __name__ == "__main__":
    main()
