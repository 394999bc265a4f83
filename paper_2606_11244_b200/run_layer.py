"""Runs ONE layer shape through the C ABI a few times and prints its device time -- the command the ncu
captures under profiles/ are taken with.

    python -m paper_2606_11244_b200.run_layer M N K group r [--gate scalar|mlp|none] [--variant V] [--iters I]
                                              [--tune key=value,...] [--seed S]

Inputs are the seeded synthetic layer of workloads.make_layer (BASELINE.json value distributions).
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
    ap.add_argument("shape", type=int, nargs=5, metavar=("M", "N", "K", "group", "r"))
    ap.add_argument("--gate", default="scalar")
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--iters", type=int, default=3)
    ap.add_argument("--tune", default="")
    ap.add_argument("--seed", type=int, default=0)
    a = ap.parse_args()
    import torch
    import paper_2606_11244_b200 as sp
    from paper_2606_11244_b200 import harness
    from workloads import make_layer, algorithmic_bytes, algorithmic_flops
    sp.init()
    for kv in a.tune.split(","):
        if "=" in kv:
            k, v = kv.split("=")
            sp.tune(k.strip(), int(v))
    M, N, K, group, r = a.shape
    li = make_layer(a.seed, M, N, K, group, r, gate=a.gate)
    dl = harness.upload_layer(li)
    x = harness.dev(li.x)
    y = torch.empty((M, N), dtype=torch.float16, device=x.device)
    ts = []
    for _ in range(a.iters):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        harness.run_layer(dl, x, variant=a.variant, y=y)
        e1.record()
        e1.synchronize()
        ts.append(e0.elapsed_time(e1) * 1e3)
    us = sorted(ts)[len(ts) // 2]
    by = algorithmic_bytes(M, N, K, group, r, a.gate)
    fl = algorithmic_flops(M, N, K, group, r, a.gate)
    print(f"M={M} N={N} K={K} group={group} r={r} gate={a.gate} variant={a.variant}: median {us:.1f} us of {a.iters} "
          f"(cold L2 not enforced)  {by / us * 1e-3:.1f} GB/s  {fl / us * 1e-6:.1f} TFLOP/s")


if __name__ == "__main__":
    main()
