"""Prefix-ratio x group-size sweep (BASELINE.json configs[3]; the paper's Claim 3)
and the other bench configs, one `bench.py` run each, collected into a markdown table.

    python -m paper_2606_01143_b200.sweep [--steps K] [--configs 7b,ragged,...] > table.md

Each row is the JSON line of `bench.py --config <name>` (GPU leg only); nothing is recomputed here.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run(config: str, steps: int) -> dict:
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--config", config, "--steps", str(steps),
           "--no-cpu", "--no-e2e", "--no-wave1", "--no-offload"]
    out = subprocess.run(cmd, capture_output=True, text=True, check=True).stdout.strip().splitlines()
    return json.loads(out[-1])


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--configs", default="")
    ap.add_argument("--json", default="", help="also append the raw JSON lines to this file")
    args = ap.parse_args()
    names = [c for c in args.configs.split(",") if c] or (
        [f"sweep-r{r}-n{n}" for r in (20, 50, 83, 95) for n in (2, 4, 8, 16)] + ["7b", "ragged", "32k"])
    print("| config | step ms | step TF/s | Phase B TF/s (% burst) | replay ms | speedup | ideal (pair model) | peak HBM GB |")
    print("|---|---|---|---|---|---|---|---|")
    for name in names:
        d = run(name, args.steps)
        if args.json:
            with open(args.json, "a") as f:
                f.write(json.dumps(d) + "\n")
        r = d["replay"]
        print(f"| {name} | {d['ms_per_step']:.3f} | {d['value']:.0f} | {d['phaseB']['tflops']:.0f} "
              f"({d['phaseB']['pct_of_bf16_burst']:.1f}) | {r['ms_per_step']:.3f} | {r['speedup']:.2f} | "
              f"{r['ideal_speedup_pair_model']:.2f} | {d['peak_hbm_bytes'] / 1e9:.2f} |", flush=True)


if __name__ == "__main__":
    main()
