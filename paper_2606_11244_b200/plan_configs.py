"""Measures the dispatch table (S9, spear_plan) for the BASELINE.json config shapes and saves it.

    python -m paper_2606_11244_b200.plan_configs [--out spear_plan.txt] [--configs 1,2,4] [--max-m 512]

Prints one line per problem: the median time of every valid variant and the one AUTO will run from now on.
Load the saved table in another process with spear_plan_load().
"""
from __future__ import annotations

import argparse
import os
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default="spear_plan.txt")
    ap.add_argument("--configs", default="0,1,2,3,4", help="0-based BASELINE.json config indices")
    ap.add_argument("--max-m", type=int, default=2048)
    a = ap.parse_args()
    import paper_2606_11244_b200 as sp
    from workloads import config_shapes
    sp.init()
    seen = set()
    print(f"{'problem':46s} " + " ".join(f"{n:>13s}" for n in sp.VARIANT_NAMES[1:]) + "  chosen")
    for ci in (int(v) for v in a.configs.split(",")):
        for s in config_shapes(ci):
            key = (s.M, s.N, s.K, s.r, s.group)
            if key in seen or s.M > a.max_m:
                continue
            seen.add(key)
            chosen, us = sp.plan(s.M, s.N, s.K, s.r, s.group, gate="scalar")
            cells = " ".join(f"{t:10.1f} us" if t > 0 else f"{'-':>13s}" for t in us[1:])
            print(f"cfg{ci + 1} M={s.M:<5d} {s.K:>5d}->{s.N:<5d} g={s.group:<5d} r={s.r:<3d}      {cells}  {sp.VARIANT_NAMES[chosen]}",
                  flush=True)
    sp.plan_save(a.out)
    print(f"saved {len(seen)} problems to {a.out}")


if __name__ == "__main__":
    main()
