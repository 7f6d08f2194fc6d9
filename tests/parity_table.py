"""Reduce gpurun_out/parity_measured.jsonl (written by the -m gpu tests through tests/helpers.record) to the table of
profiles/r2_parity_16bit.md: one row per comparison of the 16-bit tensor path, its worst species in each A12 form.

    python -m tests.parity_table [path/to/parity_measured.jsonl]

Reads only what the tests recorded (GPU result vs oracle, and the exactly rounded fp16 chain vs oracle); calls nothing.
"""
import json
import os
import sys

FLOOR_FACTOR = 1.25   # tests/helpers.py


def rows(path):
    last = {}
    with open(path) as f:
        for line in f:
            d = json.loads(line)
            if d.get("precision") == 1 and d.get("ideal_fp16_chain"):
                last[(d["tag"], d["quantity"])] = d   # a test that ran twice: the last run counts
    out = []
    for (tag, q), d in last.items():
        ps, fl = d["per_species"], {t["k"]: t for t in d["ideal_fp16_chain"]}
        wm = max(ps, key=lambda t: t["mixed"])
        wn = max(ps, key=lambda t: t["normwise"])
        bound = max(d["tol"], FLOOR_FACTOR * fl[wm["k"]]["mixed"])
        ratios = sorted(t["normwise"] / fl[t["k"]]["normwise"] for t in ps if fl[t["k"]]["normwise"] > 0)
        med = ratios[len(ratios) // 2] if ratios else float("nan")
        out.append(f"| {tag} | {q} | {d['cells_compared']} | {d['sum_to_one']:.2e} | {wm['mixed']:.3e} (k={wm['k']}; cell {wm['cell']}) | "
                   f"{bound:.3e} | {fl[wm['k']]['mixed']:.3e} | {wn['normwise']:.3e} (k={wn['k']}) | {med:.2f} |")
    return out


if __name__ == "__main__":
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    path = sys.argv[1] if len(sys.argv) > 1 else os.path.join(root, "gpurun_out", "parity_measured.jsonl")
    print("| test | quantity | cells compared | sum(Y+dY)-1 max | worst element-wise mixed (species; cell) | its bound | floor of an "
          "exactly rounded fp16 chain (same species) | worst normwise (species) | GPU/floor normwise, median over species |")
    print("|---|---|---|---|---|---|---|---|---|")
    for r in rows(path):
        print(r)
