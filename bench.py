#!/usr/bin/env python
"""bench.py -- BASELINE.json metric on one B200: the W4A16 + gated-EC layer's decode HBM GB/s.

Workload (config.workload): BASELINE.json configs[1] -- Llama-3.2-1B-shaped decode projections
(qkv 2048->3072, o 2048->2048, gate_up 2048->16384, down 8192->2048), int4 group=128, EC rank 32 with
the scalar sigmoid gate on every projection, M in {1, 8, 16}.  One "step" = one pass of the whole hot
path over that batch = 12 layer calls (3 token counts x 4 projections), all through the C ABI
(spear_w4_ec_gemm_ex).  value = algorithmic bytes of the step (packed weights +
scales + x + y + EC factors + gate vector) / device time, whole job.  The headline step issues the 12 calls one
after the other on one stream (the dependent-chain regime: in a decoder qkv -> o -> gate_up -> down depend on each
other); the same step overlapped on the library's lanes and as one persistent layer-stream launch are reported
beside it, and the `configs` key carries SURVEY.md 8(d)'s result rows for all five configs.

L2 hygiene: every step reads a different copy of the weights and EC factors from an arena of NCOPY
copies (> 4x the 126 MB L2), so weights always come from HBM ("inputs larger than L2").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

N > 1 (torchrun): replicas only -- each rank runs the same per-GPU workload (weak scaling), no
collective on the data path; rank 0 reports the sum.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

from workloads import algorithmic_bytes, config_shapes, make_layer, with_int8_ec
from workloads.synth import make_x

METRIC = "W4A16+gated-EC layer: decode HBM GB/s (Llama-3.2-1B decode projections, r=32, M in {1,8,16})"
UNIT = "GB/s"
TOKENS = (1, 8, 16)
NCOPY_TARGET_BYTES = 640 << 20


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def step_shapes():
    """The 12 layer shapes of one step, grouped by token count."""
    shapes = config_shapes(1)
    return {M: [s for s in shapes if s.M == M] for M in TOKENS}


def step_bytes(with_ec=True, ec_int8=False):
    tot = 0
    for M, ss in step_shapes().items():
        for s in ss:
            tot += algorithmic_bytes(s.M, s.N, s.K, s.group, s.r if with_ec else 0, "scalar", ec_int8=ec_int8)
    return tot


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled while the timed regions run."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,utilization.gpu,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            f = [c.strip() for c in r.split(",")]
            if len(f) < 8:
                continue
            try:
                clk, mxc, util = float(f[0]), float(f[1]), float(f[3])
            except ValueError:
                continue
            mx = mxc
            if util > 0:
                sm.append(clk)
                for n, v in zip(names, f[4:8]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx,
                "reasons": sorted(reasons), "samples_under_load": len(sm)}


def max_over_ranks(ms, world, device):
    """Replicas only: the job's step time is the slowest rank's device time."""
    if world <= 1:
        return ms
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_value(bytes_per_rank_step, ms_per_step, world):
    """Whole-job throughput in GB/s: every rank moves the same algorithmic bytes per step (weak scaling)."""
    return world * bytes_per_rank_step / (ms_per_step * 1e-3) / 1e9


# ------------------------------------------------------------------------------------------------
# CUDA arm
# ------------------------------------------------------------------------------------------------
NOMINAL_HBM_GBS = 8000.0          # nominal 8 TB/s, 2.25 PFLOP/s dense fp16
NOMINAL_TFLOPS = 2250.0


def load_tensor_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["bf16_tflops"]), "measured (MEASURED_PEAKS.json bf16_tflops, burst)"
    return 1590.0, "fallback (B200_PROFILING.md 1.59 PFLOP/s burst)"


def profile_traffic(kernel):
    """dram__bytes_read + dram__bytes_write per launch of `kernel` (the dominant decode kernel of this run), from the committed
    ncu capture.  A capture of another kernel is not a substitute: then the figure is None and the note says what is missing."""
    p = os.path.join(ROOT, "profiles", "r02_dram_traffic.csv")
    if not os.path.exists(p):
        return None, "no capture committed"
    import csv
    with open(p) as f:
        rows = list(csv.reader(l for l in f if l.strip() and not l.startswith("#")))
    for r in rows[1:]:
        if r[0] and r[0] in kernel:
            return int(r[3]), f"{r[1]} ({r[2]}); algorithmic {r[4]} B; profiles/r02_dram_traffic.csv"
    return None, f"no capture of {kernel} in profiles/r02_dram_traffic.csv (it holds: {', '.join(sorted({r[0] for r in rows[1:]}))})"


def run_cuda(args, rank, world):
    import torch
    import torch.distributed as dist
    import paper_2606_11244_b200 as sp
    from paper_2606_11244_b200 import harness

    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    device = f"cuda:{local}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(device))
    sp.init()
    tunes = {}
    for kv in os.environ.get("SPEAR_TUNE", "").split(","):     # sweep hook: key=value,... for spear_tune; echoed in config
        if "=" in kv:
            k, v = kv.split("=")
            sp.tune(k.strip(), int(v))
            tunes[k.strip()] = int(v)

    shapes = step_shapes()
    # weights / EC factors: one seeded set per projection (the M=16 entry's seed), shared by the three
    # token counts; activations per (M, projection) from that entry's own seed
    base, base8 = {}, {}
    for s in shapes[16]:
        li = make_layer(s.seed, 16, s.N, s.K, s.group, s.r, gate="scalar")
        base[s.name] = harness.upload_layer(li, device)
        l8 = with_int8_ec(li)          # the same EC stored INT8 per-channel symmetric
        base8[s.name] = tuple(harness.dev(a, device) for a in (l8.A, l8.B, l8.A_scale, l8.B_scale))
    set_bytes = sum(dl.pw.wq.numel() + dl.pw.scales.numel() * 2 + (dl.A.numel() + dl.B.numel() + dl.w_g.numel()) * 2
                    for dl in base.values())
    ncopy = max(3, -(-NCOPY_TARGET_BYTES // set_bytes))
    ncopy = -(-ncopy // 3) * 3
    copies = []
    for c in range(ncopy):
        d = {}
        for name, dl in base.items():
            pw = sp.PackedW4(dl.pw.wq.clone(), dl.pw.scales.clone(), dl.pw.N, dl.pw.K, dl.pw.group)
            d[name] = harness.DeviceLayer(pw=pw, M=0, N=dl.N, K=dl.K, r=dl.r, group=dl.group, gate="scalar",
                                          alpha=1.0, A=dl.A.clone(), B=dl.B.clone(), w_g=dl.w_g.clone(), b_g=dl.b_g)
            A8, B8, sA, sB = base8[name]
            d[name + "/i8"] = harness.DeviceLayer(pw=pw, M=0, N=dl.N, K=dl.K, r=dl.r, group=dl.group, gate="scalar", alpha=1.0,
                                                  A=A8.clone(), B=B8.clone(), w_g=d[name].w_g, b_g=dl.b_g, A_scale=sA.clone(), B_scale=sB.clone())
        copies.append(d)
    xs, ys, xh, yh = {}, {}, {}, {}
    for M in TOKENS:
        for s in shapes[M]:
            x, _ = make_x(s.seed, M, s.K)
            xs[(M, s.name)] = harness.dev(x, device)
            ys[(M, s.name)] = torch.empty((M, s.N), dtype=torch.float16, device=device)
            xh[(M, s.name)] = torch.from_numpy(x).pin_memory()
            yh[(M, s.name)] = torch.empty((M, s.N), dtype=torch.float16).pin_memory()

    descs = {}   # keep EcDesc objects alive
    batches = {}

    def one_step(g, with_ec=True, mode="ordered", ec_resident=False, ec_int8=False):
        """One pass over the 12 layer calls of the step.  mode: "ordered" = 12 stream-ordered spear_w4_ec_gemm_ex calls, one
        after the other (PDL-chained kernels) -- the regime of SURVEY.md 8(d) and of a real decoder, whose projections
        depend on each other; "lanes" = ONE spear_w4_ec_gemm_batch over the library's concurrent lanes (the 12 calls of
        the config are independent problems); "lstream" = ONE persistent layer-stream launch.  ec_resident: the EC factors
        come from ONE copy (L2-resident, a model's EC set is a few MB) instead of rotating with the weights (cold)."""
        entries = []
        for mi, M in enumerate(TOKENS):
            cp = copies[(3 * g + mi) % ncopy]
            ecp = copies[0] if ec_resident else cp
            for s in shapes[M]:
                dl, de = cp[s.name], ecp[s.name + ("/i8" if ec_int8 else "")]
                key = (g, mi, s.name, with_ec, ec_resident, ec_int8)
                if key not in descs:
                    descs[key] = de.desc() if with_ec else sp.make_desc(gate="none")
                A, B = (de.A, de.B) if with_ec else (None, None)
                if mode == "ordered":
                    sp.w4_ec_gemm_ex(xs[(M, s.name)], dl.pw, A, B, descs[key], y=ys[(M, s.name)])
                else:
                    entries.append((xs[(M, s.name)], dl.pw, A, B, descs[key], ys[(M, s.name)]))
        if mode != "ordered":
            bk = (g, with_ec, ec_resident, ec_int8)
            if bk not in batches:
                batches[bk] = sp.Batch(entries)
            sp.tune("lstream", 1 if mode == "lstream" else 0)
            sp.w4_ec_gemm_batch(batches[bk])
            sp.tune("lstream", -1)

    stream = torch.cuda.Stream()
    ngraph = ncopy // 3

    def make_graphs(with_ec, mode, ec_resident=False, ec_int8=False):
        gs = []
        with torch.cuda.stream(stream):
            one_step(0, with_ec, mode, ec_resident, ec_int8)  # first-call work (tensor maps, attributes) outside capture
            torch.cuda.synchronize()
            for g in range(ngraph):
                cg = torch.cuda.CUDAGraph()
                with torch.cuda.graph(cg, stream=stream):
                    one_step(g, with_ec, mode, ec_resident, ec_int8)
                gs.append(cg.replay)
        return gs

    def timed(fns, steps, warmup):
        with torch.cuda.stream(stream):
            for i in range(warmup):
                fns[i % len(fns)]()
            if world > 1:
                dist.barrier()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for i in range(steps):
                fns[i % len(fns)]()
            e1.record(stream)
            torch.cuda.synchronize()
            if world > 1:
                dist.barrier()
        return max_over_ranks(e0.elapsed_time(e1), world, device)

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    b_ec, b_w4 = step_bytes(True), step_bytes(False)
    peak, peak_src = load_peaks()

    def leg(with_ec, mode, ec_resident=False, steps=None, ec_int8=False):
        steps = steps or args.steps
        ms = timed(make_graphs(with_ec, mode, ec_resident, ec_int8), steps, args.warmup) / steps
        by = (step_bytes(True, True) if ec_int8 else b_ec) if with_ec else b_w4
        gbs = aggregate_value(by, ms, world)
        return {"value": round(gbs, 1), "ms_per_step": round(ms, 6), "frac_of_measured_hbm": round(gbs / world / peak, 4),
                "frac_of_nominal_8tbs": round(gbs / world / NOMINAL_HBM_GBS, 4)}

    # headline: the dependent-chain regime (stream-ordered calls), EC factors cold (rotating with the weights)
    launches0 = sp.launch_count()
    g_head = make_graphs(True, "ordered")
    per_step_launches = (sp.launch_count() - launches0) // (ngraph + 1)
    ms_head = timed(g_head, args.steps, args.warmup) / args.steps
    sub = min(args.steps, 500)
    ordered_w4 = leg(False, "ordered")
    ordered_ec_res = leg(True, "ordered", ec_resident=True, steps=sub)
    ordered_ec_i8 = leg(True, "ordered", steps=sub, ec_int8=True)
    lanes_ec_i8 = leg(True, "lanes", steps=sub, ec_int8=True)
    lanes_ec, lanes_w4 = leg(True, "lanes", steps=sub), leg(False, "lanes", steps=sub)
    ls_ec, ls_w4 = leg(True, "lstream", steps=sub), leg(False, "lstream", steps=sub)
    # ---- which kernel runs which call, and how long each call takes in the headline regime --------------------------------
    # One CUDA graph per call of the step: that call alone, stream-ordered, once per weight copy.  The 12 graphs are replayed in
    # turn, so between two replays of one graph all the other calls' copies (677 MiB in all) have gone through L2: cold weights.
    KERNEL_OF = {sp.VARIANT_STREAM_FUSED: "spear::stream_kernel<MT,1>", sp.VARIANT_STREAM_SPLIT: "spear::stream_kernel<MT,1>",
                 sp.VARIANT_ROWS: "spear::rows_kernel<MT,false> (with an EC: behind spear::ecz_cluster_kernel<MT>, counted with it)", sp.VARIANT_LSTREAM: "spear::ls_kernel",
                 sp.VARIANT_TC_FUSED: "spear::tc_kernel", sp.VARIANT_TC_SPLIT: "spear::tc_kernel"}

    def per_call(with_ec):
        calls, graphs = [], []
        with torch.cuda.stream(stream):
            for M in TOKENS:
                for s in shapes[M]:
                    ds = [(cp[s.name].desc() if with_ec else sp.make_desc(gate="none")) for cp in copies]

                    def body(M=M, s=s, ds=ds):
                        for cp, d in zip(copies, ds):
                            dl = cp[s.name]
                            sp.w4_ec_gemm_ex(xs[(M, s.name)], dl.pw, dl.A if with_ec else None, dl.B if with_ec else None, d, y=ys[(M, s.name)])
                    body()
                    torch.cuda.synchronize()
                    cg = torch.cuda.CUDAGraph()
                    with torch.cuda.graph(cg, stream=stream):
                        body()
                    graphs.append((cg, ds))
                    v = sp.plan_query(M, s.N, s.K, s.r if with_ec else 0, s.group, gate="scalar" if with_ec else "none")
                    calls.append({"call": f"{s.name} M={M}", "variant": v, "kernel": KERNEL_OF.get(v, "?"),
                                  "bytes": algorithmic_bytes(M, s.N, s.K, s.group, s.r if with_ec else 0, "scalar" if with_ec else "none", 0)})
            ts = [[] for _ in graphs]
            for rep in range(7):
                for gi, (cg, _) in enumerate(graphs):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(stream)
                    cg.replay()
                    e1.record(stream)
                    e1.synchronize()
                    if rep >= 2:
                        ts[gi].append(e0.elapsed_time(e1) * 1e3 / ncopy)
        for c, t in zip(calls, ts):
            c["us"] = round(sorted(t)[len(t) // 2], 3)
        return calls

    def by_kernel(calls):
        tot = sum(c["us"] for c in calls)
        groups = {}
        for c in calls:
            g = groups.setdefault(c["kernel"], {"kernel": c["kernel"], "launches_per_step": 0, "us_per_step": 0.0, "bytes_per_step": 0, "calls": []})
            g["launches_per_step"] += 1
            g["us_per_step"] += c["us"]
            g["bytes_per_step"] += c["bytes"]
            g["calls"].append(c["call"])
        out = []
        for g in groups.values():
            ach = g["bytes_per_step"] / (g["us_per_step"] * 1e-6) / 1e9
            out.append({"kernel": g["kernel"], "launches_per_step": g["launches_per_step"], "calls": g["calls"],
                        "share_of_step_time": round(g["us_per_step"] / tot, 4), "avg_launch_us": round(g["us_per_step"] / g["launches_per_step"], 3),
                        "algorithmic_bytes_per_launch": int(g["bytes_per_step"] / g["launches_per_step"]),
                        "achieved": round(ach, 1), "frac": round(ach / peak, 4)})
        out.sort(key=lambda g: -g["share_of_step_time"])
        return out, tot

    calls_w4, calls_ec = per_call(False), per_call(True)
    kern_w4, sum_w4 = by_kernel(calls_w4)
    kern_ec, sum_ec = by_kernel(calls_ec)
    t_end = time.time() + 1.0      # keep the GPU under load long enough for nvidia-smi to sample it
    while rank == 0 and time.time() < t_end:
        timed(g_head, 200, 0)

    # e2e: pinned-host x -> device -> layer -> pinned-host y for every call of the step, through ONE
    # spear_w4_ec_gemm_batch_hostio (copies and kernels of different calls overlap on the lanes)
    e2e_steps = max(1, min(args.steps, 300))
    one_step(0, True, "lanes")          # builds batches[(g, True, False)] for every rotation below
    for g in range(ngraph):
        one_step(g, True, "lanes")
    torch.cuda.synchronize()

    def e2e_step(g):
        bt = batches[(g, True, False, False)]
        order = [(M, s.name) for M in TOKENS for s in shapes[M]]
        sp.w4_ec_gemm_batch_hostio(bt, [xh[k] for k in order], [yh[k] for k in order], stream=stream)

    ms_e2e = timed([lambda g=g: e2e_step(g) for g in range(ngraph)], e2e_steps, max(3, min(args.warmup, 20))) / e2e_steps
    clocks = sampler.stop() if rank == 0 else None

    value = aggregate_value(b_ec, ms_head, world)
    ncalls = sum(len(v) for v in shapes.values())
    dom = kern_w4[0]
    traffic, traffic_note = profile_traffic(dom["kernel"])
    out = {
        "metric": METRIC, "value": round(value, 1), "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": round(ms_head, 6), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f16 (int4 weights, fp32 accumulate)", "data": "synthetic (seeded, workloads/)",
        "config": {"workload": "BASELINE.json configs[1]: Llama-3.2-1B decode projections qkv/o/gate_up/down, group=128, EC r=32 "
                               "scalar sigmoid gate, M in {1,8,16}; step = the 12 layer calls issued one after the other on one "
                               "stream (dependent-chain regime of SURVEY.md 8(d); EC factors cold = rotating with the weights)",
                   "l2": f"inputs larger than L2: weights+EC rotate over {ncopy} copies ({ncopy * set_bytes >> 20} MiB)",
                   "cuda_graph": True, "bytes_per_step": b_ec, "parallelism": f"replicas x{world}",
                   "spear_tune_overrides": tunes, "env": {k: os.environ[k] for k in ("SPEAR_TUNE",) if k in os.environ}},
        "e2e": {"value": round(world * b_ec / (ms_e2e * 1e-3) / 1e9, 1), "unit": UNIT,
                "h2d_bytes_per_step": sum(t.numel() * 2 for t in xh.values()),
                "d2h_bytes_per_step": sum(t.numel() * 2 for t in yh.values()), "ms_per_step": round(ms_e2e, 6),
                "path": "spear_w4_ec_gemm_batch_hostio (per call: pinned host x -> device, layer, device -> pinned host y, on the lanes)"},
        "gpu_launches": int(per_step_launches * args.steps),
        "clocks": clocks,
        "roofline": dict(
            {"bound": "hbm", "kernel": dom["kernel"], "achieved": dom["achieved"], "peak": peak, "unit": "GB/s", "frac": dom["frac"],
             "peak_source": peak_src, "traffic": traffic, "traffic_note": traffic_note,
             "avg_launch_us": dom["avg_launch_us"], "launches_per_step": dom["launches_per_step"],
             "algorithmic_bytes_per_launch": dom["algorithmic_bytes_per_launch"], "share_of_step_time": dom["share_of_step_time"],
             "calls": dom["calls"]},
            how="the kernel with the largest share of the plain (r = 0) stream-ordered step; achieved = algorithmic bytes of ITS launches / "
                "the summed durations of ITS launches, each call timed alone in its own CUDA graph over cold weight copies (graphs replayed "
                "in turn); which kernel serves a call is asked of the library (spear_plan_query)",
            other_kernels=kern_w4[1:], with_ec=kern_ec,
            per_call_us={"no_ec": {c["call"]: c["us"] for c in calls_w4}, "ec": {c["call"]: c["us"] for c in calls_ec}},
            step={"note": "the whole step (all 12 calls, every kernel): bytes_per_step / ms_per_step of the no_ec and headline legs; "
                          "sum_of_calls_us is the per-call graphs added up (isolated calls; the mixed step differs by a few per cent)",
                  "frac_no_ec": ordered_w4["frac_of_measured_hbm"], "frac_with_ec": round(value / world / peak, 4),
                  "sum_of_calls_us": {"no_ec": round(sum_w4, 2), "ec": round(sum_ec, 2)},
                  "step_us": {"no_ec": round(ordered_w4["ms_per_step"] * 1e3, 2), "ec": round(ms_head * 1e3, 2)}}),
        "no_ec": ordered_w4,
        "ec_overhead_time_frac": round(ms_head / ordered_w4["ms_per_step"] - 1.0, 4),
        "ec_l2_resident": dict(ordered_ec_res, ec_overhead_time_frac=round(ordered_ec_res["ms_per_step"] / ordered_w4["ms_per_step"] - 1.0, 4)),
        "ec_int8": {"note": "the same step with the EC factors stored INT8 per-channel symmetric (PAPER.md:603): bytes_EC halve; cold factors",
                    "ordered": dict(ordered_ec_i8, ec_overhead_time_frac=round(ordered_ec_i8["ms_per_step"] / ordered_w4["ms_per_step"] - 1.0, 4)),
                    "lanes": dict(lanes_ec_i8, ec_overhead_time_frac=round(lanes_ec_i8["ms_per_step"] / lanes_w4["ms_per_step"] - 1.0, 4))},
        "overlapped_lanes": {"note": "same step as ONE spear_w4_ec_gemm_batch: the 12 calls are independent problems, the library overlaps "
                                     "them on 12 concurrent lanes (round 1's headline; not a dependent chain)",
                             "ec": lanes_ec, "no_ec": lanes_w4,
                             "ec_overhead_time_frac": round(lanes_ec["ms_per_step"] / lanes_w4["ms_per_step"] - 1.0, 4)},
        "layer_stream": {"note": "same step as ONE persistent cooperative launch of spear::ls_kernel (tcgen05, weights through tensor "
                                 "memory); kernel durations are multiples of ~2.05 us on this path (DESIGN.md 6.5)",
                         "ec": ls_ec, "no_ec": ls_w4,
                         "ec_overhead_time_frac": round(ls_ec["ms_per_step"] / ls_w4["ms_per_step"] - 1.0, 4)},
    }
    if rank == 0:
        del copies, base
        torch.cuda.empty_cache()
        out["prefill"] = None
        if not args.no_table:
            out["configs"] = configs_table(sp, device)
            p4 = out["configs"]["config4"]
            best = max((e for e in p4 if e["M"] == 4096 and e["r"] == 0), key=lambda e: e["tflops"])
            ec64 = [e for e in p4 if e["M"] == 4096 and e["r"] == 64][0]
            out["prefill"] = {"workload": "BASELINE.json configs[3]: M=4096, K=8192, N=28672, group=128 (see configs.config4 for the sweep)",
                              "kernel": "spear::tc_kernel<256,2> (tcgen05, TMEM accumulators, EC folded in as extra k-blocks)",
                              "tflops_no_ec": best["tflops"], "tflops_ec_r64": ec64["tflops"],
                              "ec_overhead_time_frac": ec64.get("ec_overhead_time_frac"),
                              "roofline": {"bound": "tensor", "achieved": best["tflops"], "peak": load_tensor_peak()[0], "unit": "TFLOP/s",
                                           "frac": best["frac_of_measured_roofline"], "peak_source": load_tensor_peak()[1],
                                           "frac_of_nominal_2250": best["frac_of_nominal_roofline"]}}
        out["cpu_baseline"] = cpu_baseline_sample()
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------
# SURVEY.md 8(d) result rows for all five configs (perf only: seeded device-side generator with the configs' value
# distributions -- parity on every one of these shapes is tests/test_gpu_*.py with workloads/ inputs)
# ------------------------------------------------------------------------------------------------
def configs_table(sp, device):
    import torch
    from workloads import algorithmic_flops
    hbm, _ = load_peaks()
    tpk, _ = load_tensor_peak()
    gen = torch.Generator(device=device)
    gen.manual_seed(20260611)

    def rand_layer(N, K, group, r, gate="scalar"):
        codes = torch.randint(0, 16, (N, K), dtype=torch.uint8, device=device, generator=gen)
        scales = (torch.randn(N, K // group, device=device, generator=gen).abs() * 0.02 + 1e-3).half()
        pw = sp.pack_w4(codes, scales, group)
        del codes
        L = {"pw": pw, "r": r, "gate": gate if r else "none"}
        if r:
            L["A"] = (torch.randn(r, K, device=device, generator=gen) / K ** 0.5).half()
            L["B"] = (torch.randn(N, r, device=device, generator=gen) / r ** 0.5).half()
            if gate == "scalar":
                L["w_g"] = (torch.randn(K, device=device, generator=gen) / K ** 0.5).half()
                L["b_g"] = torch.zeros(1, device=device)
            elif gate == "mlp":
                h = 4 * r
                L["W1"] = (torch.randn(h, r, device=device, generator=gen) / r ** 0.5).half()
                L["W2"] = (torch.randn(r, h, device=device, generator=gen) / h ** 0.5).half()
                L["b1"], L["b2"] = torch.zeros(h, device=device), torch.zeros(r, device=device)
        return L

    def clones(L, n, ec_too=True):
        out = [L]
        for _ in range(n - 1):
            C = dict(L)
            C["pw"] = sp.PackedW4(L["pw"].wq.clone(), L["pw"].scales.clone(), L["pw"].N, L["pw"].K, L["pw"].group)
            if L["r"] and ec_too:
                C["A"], C["B"] = L["A"].clone(), L["B"].clone()
            out.append(C)
        return out

    def desc_of(L):
        return sp.make_desc(gate=L["gate"], w_g=L.get("w_g"), b_g=L.get("b_g"), W1=L.get("W1"), b1=L.get("b1"),
                            W2=L.get("W2"), b2=L.get("b2"))

    stream = torch.cuda.Stream()

    def steady_graph(M, arena, n_calls, plain):
        K, N = arena[0]["pw"].K, arena[0]["pw"].N
        x = torch.randn(M, K, device=device, generator=gen).half()
        y = torch.empty(M, N, dtype=torch.float16, device=device)
        ds = [sp.make_desc(gate="none") if plain else desc_of(L) for L in arena]

        def body():
            for i in range(n_calls):
                L = arena[i % len(arena)]
                sp.w4_ec_gemm_ex(x, L["pw"], None if plain else L.get("A"), None if plain else L.get("B"), ds[i % len(arena)], y=y)

        with torch.cuda.stream(stream):
            body()
            torch.cuda.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                body()
            g.replay()
            torch.cuda.synchronize()
        return g, (x, y, ds)

    def time_graphs(graphs, n_calls, reps):
        """Medians (us per call) of `reps` replays of each graph, the graphs taken in turn (same clock / power state)."""
        ts = [[] for _ in graphs]
        with torch.cuda.stream(stream):
            for _ in range(reps):
                for gi, (g, _) in enumerate(graphs):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(stream)
                    g.replay()
                    e1.record(stream)
                    e1.synchronize()
                    ts[gi].append(e0.elapsed_time(e1) * 1e3 / n_calls)
        return [sorted(t)[len(t) // 2] for t in ts]

    def steady_us(M, arena, n_calls, plain=False, reps=5):
        """Steady state (SURVEY.md 8(d) regime 1): a CUDA graph of n_calls back-to-back stream-ordered calls cycling through
        the arena (>= 512 MB of weights unless the layer alone exceeds L2); microseconds per call, median of `reps` replays."""
        return time_graphs([steady_graph(M, arena, n_calls, plain)], n_calls, reps)[0]

    def steady_pair_us(M, arena, n_calls, reps=5):
        """(plain, with EC) on the same arena, replays interleaved."""
        return time_graphs([steady_graph(M, arena, n_calls, True), steady_graph(M, arena, n_calls, False)], n_calls, reps)

    def row(name, M, N, K, group, r, us, gate="scalar", extra=None):
        by = algorithmic_bytes(M, N, K, group, r, gate, 4 * r if gate == "mlp" else 0)
        fl = algorithmic_flops(M, N, K, group, r, gate, 4 * r if gate == "mlp" else 0)
        t_meas = max(by / (hbm * 1e3), fl / (tpk * 1e6))          # us at the measured peaks
        t_nom = max(by / (NOMINAL_HBM_GBS * 1e3), fl / (NOMINAL_TFLOPS * 1e6))
        e = {"name": name, "M": M, "N": N, "K": K, "group": group, "r": r, "gate": gate if r else "none", "us": round(us, 2),
             "gbs": round(by / us * 1e-3, 1), "tflops": round(fl / us * 1e-6, 2),
             "bound": "hbm" if by / hbm / 1e3 >= fl / tpk / 1e6 else "tensor",
             "frac_of_measured_roofline": round(t_meas / us, 4), "frac_of_nominal_roofline": round(t_nom / us, 4)}
        if extra:
            e.update(extra)
        return e

    def arena_for(L, M):
        wbytes = L["pw"].wq.numel() + L["pw"].scales.numel() * 2
        n = max(2, min(40, -(-(512 << 20) // wbytes)))
        return clones(L, n), (64 if M <= 16 else max(n, 4))

    def sweep(shapes, gate="scalar"):
        rows = []
        layers = {}
        for s in shapes:
            key = (s.N, s.K, s.group, s.r)
            if key not in layers:
                layers.clear()
                torch.cuda.empty_cache()
                layers[key] = rand_layer(s.N, s.K, s.group, s.r, gate)
            L = layers[key]
            arena, n_calls = arena_for(L, s.M)
            if s.r:
                us0, us1 = steady_pair_us(s.M, arena, n_calls)
            else:
                us0 = steady_us(s.M, arena, n_calls, plain=True)
            rows.append(row(s.name, s.M, s.N, s.K, s.group, 0, us0))
            if s.r:
                rows.append(row(s.name, s.M, s.N, s.K, s.group, s.r, us1, gate, {"ec_overhead_time_frac": round(us1 / us0 - 1.0, 4)}))
            del arena
        return rows

    table = {"protocol": "steady state: CUDA graph of back-to-back stream-ordered calls of one shape cycling through >= 512 MB of weight "
                         "copies (EC factors cold), median of 5 replays; us per call; roofline = max(bytes / HBM peak, flops / tensor peak) "
                         "at the measured and at the nominal (8 TB/s, 2.25 PFLOP/s) peaks",
             "peaks": {"hbm_gbs_measured": hbm, "tensor_tflops_measured": tpk}}
    table["config1"] = sweep(config_shapes(0))
    table["config2"] = sweep(config_shapes(1))
    table["config3"] = sweep(config_shapes(2))
    # config 4: one weight arena per r, all three token counts.  The EC overhead of a row is taken against the plain layer
    # timed on the SAME arena with interleaved replays (the part power-caps under these GEMMs: rows measured seconds apart
    # do not share a clock state)
    rows4 = []
    s0 = config_shapes(3)[0]
    for r in (0, 16, 64, 128):
        torch.cuda.empty_cache()
        L = rand_layer(s0.N, s0.K, s0.group, r)
        arena = clones(L, 5)
        for M in (512, 4096, 16384):
            reps = 3 if M == 16384 else 7
            if r == 0:
                us0 = steady_us(M, arena, 5, plain=True, reps=reps)
                rows4.append(row("mlp70b", M, s0.N, s0.K, s0.group, 0, us0))
            else:
                us0, us1 = steady_pair_us(M, arena, 5, reps=reps)
                rows4.append(row("mlp70b", M, s0.N, s0.K, s0.group, r, us1, "scalar",
                                 {"ec_overhead_time_frac": round(us1 / us0 - 1.0, 4), "plain_us_same_arena": round(us0, 2)}))
        del arena, L
    table["config4"] = rows4
    torch.cuda.empty_cache()
    table["mlp_gate_cost"] = mlp_gate_rows(sp, rand_layer, arena_for, steady_us, row)
    table["single_cold_launch"] = cold_launch_rows(sp, device, rand_layer, desc_of, row, gen)
    table["fused_tail"] = tail_rows(sp, device, rand_layer, desc_of, clones, gen)
    torch.cuda.empty_cache()
    table["config5"] = stack_rows(sp, device, rand_layer, desc_of, gen, hbm, tpk)
    return table


def mlp_gate_rows(sp, rand_layer, arena_for, steady_us, row):
    """The paper's MLP gate (h = 4r) against the scalar gate of the configs (reading A1): config 1, one decode and
    one prefill shape."""
    out = []
    for (name, M, N, K, group, r) in (("config1", 4, 2048, 2048, 128, 16), ("config2 gate_up", 8, 16384, 2048, 128, 32),
                                      ("config3 qkv", 256, 6144, 4096, 4096, 64)):
        for gate in ("scalar", "mlp"):
            L = rand_layer(N, K, group, r, gate)
            arena, n_calls = arena_for(L, M)
            out.append(row(name, M, N, K, group, r, steady_us(M, arena, n_calls), gate))
            del arena, L
    return out


def tail_rows(sp, device, rand_layer, desc_of, clones, gen):
    """the layer with the residual add + next-layer RMSNorm fused into its epilogue (spear_w4_ec_gemm_tail) against
    the layer alone, on the two projections of configs[1] that write the residual stream (o, down), M = 8, steady state."""
    import torch
    out = []
    stream = torch.cuda.Stream()
    for (name, N, K) in (("o", 2048, 2048), ("down", 2048, 8192)):
        M, r = 8, 32
        L = rand_layer(N, K, 128, r)
        arena = clones(L, max(2, -(-(512 << 20) // (N * K // 2))))
        x = torch.randn(M, K, device=device, generator=gen).half()
        y = torch.empty(M, N, dtype=torch.float16, device=device)
        res = torch.randn(M, N, device=device, generator=gen).half()
        gw = torch.ones(N, dtype=torch.float16, device=device)
        hn = torch.empty(M, N, dtype=torch.float16, device=device)
        ds = [desc_of(C) for C in arena]
        us = {}
        for mode in ("layer", "layer+tail"):
            def body():
                for i in range(64):
                    C = arena[i % len(arena)]
                    if mode == "layer":
                        sp.w4_ec_gemm_ex(x, C["pw"], C["A"], C["B"], ds[i % len(arena)], y=y)
                    else:
                        sp.w4_ec_gemm_tail(x, C["pw"], C["A"], C["B"], ds[i % len(arena)], res, gw, 1e-5, y=y, h_out=hn)
            with torch.cuda.stream(stream):
                body()
                torch.cuda.synchronize()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=stream):
                    body()
                g.replay()
                torch.cuda.synchronize()
                ts = []
                for _ in range(5):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(stream)
                    g.replay()
                    e1.record(stream)
                    e1.synchronize()
                    ts.append(e0.elapsed_time(e1) * 1e3 / 64)
            us[mode] = sorted(ts)[2]
        out.append({"name": f"config2 {name}", "M": M, "N": N, "K": K, "r": r, "us_layer": round(us["layer"], 2),
                    "us_layer_plus_fused_tail": round(us["layer+tail"], 2),
                    "tail_overhead_time_frac": round(us["layer+tail"] / us["layer"] - 1.0, 4)})
        del arena, L
    return out


def cold_launch_rows(sp, device, rand_layer, desc_of, row, gen):
    """SURVEY.md 8(d) regime 2: ONE call after the L2 has been flushed by a 256 MB write; median of 15."""
    import torch
    out = []
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=device)
    for (name, M, N, K, group, r) in (("config2 o", 1, 2048, 2048, 128, 32), ("config2 gate_up", 8, 16384, 2048, 128, 32),
                                      ("config3 gate_up", 16, 28672, 4096, 4096, 64)):
        L = rand_layer(N, K, group, r)
        x = torch.randn(M, K, device=device, generator=gen).half()
        y = torch.empty(M, N, dtype=torch.float16, device=device)
        d = desc_of(L)
        ts = []
        for i in range(18):
            flush.fill_(i & 0xff)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            sp.w4_ec_gemm_ex(x, L["pw"], L["A"], L["B"], d, y=y)
            e1.record()
            e1.synchronize()
            if i >= 3:
                ts.append(e0.elapsed_time(e1) * 1e3)
        out.append(row(name, M, N, K, group, r, sorted(ts)[len(ts) // 2]))
        del L
    return out


def stack_rows(sp, device, rand_layer, desc_of, gen, hbm, tpk):
    """configs[4]: the 64-call projection stack as ONE spear_w4_ec_gemm_batch captured in ONE CUDA graph (reading A11), with the
    ECs on o / down of layers {0, 1, 14, 15} and with no EC at all; the stack's own weights (579 MB) exceed L2."""
    import torch
    from workloads import algorithmic_flops
    from workloads.configs import stack_shapes
    out = []
    for M in (64, 2048):
        shapes = stack_shapes(M)
        layers = [rand_layer(s.N, s.K, s.group, s.r) for s in shapes]
        xs = [torch.randn(M, s.K, device=device, generator=gen).half() for s in shapes]
        ys = [torch.empty(M, s.N, dtype=torch.float16, device=device) for s in shapes]
        for with_ec in (False, True):
            ds = [desc_of(L) if with_ec else sp.make_desc(gate="none") for L in layers]
            batch = sp.Batch([(x, L["pw"], L.get("A") if with_ec else None, L.get("B") if with_ec else None, d, y)
                              for x, L, d, y in zip(xs, layers, ds, ys)])
            st = torch.cuda.Stream()
            with torch.cuda.stream(st):
                sp.w4_ec_gemm_batch(batch, stream=st)
                torch.cuda.synchronize()
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=st):
                    sp.w4_ec_gemm_batch(batch, stream=st)
                g.replay()
                torch.cuda.synchronize()
                ts = []
                for _ in range(5):
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(st)
                    g.replay()
                    e1.record(st)
                    e1.synchronize()
                    ts.append(e0.elapsed_time(e1) * 1e3)
            us = sorted(ts)[len(ts) // 2]
            by = sum(algorithmic_bytes(M, s.N, s.K, s.group, s.r if with_ec else 0, "scalar") for s in shapes)
            fl = sum(algorithmic_flops(M, s.N, s.K, s.group, s.r if with_ec else 0, "scalar") for s in shapes)
            t_meas = sum(max(algorithmic_bytes(M, s.N, s.K, s.group, s.r if with_ec else 0, "scalar") / (hbm * 1e3),
                             algorithmic_flops(M, s.N, s.K, s.group, s.r if with_ec else 0, "scalar") / (tpk * 1e6)) for s in shapes)
            t_nom = sum(max(algorithmic_bytes(M, s.N, s.K, s.group, s.r if with_ec else 0, "scalar") / (NOMINAL_HBM_GBS * 1e3),
                            algorithmic_flops(M, s.N, s.K, s.group, s.r if with_ec else 0, "scalar") / (NOMINAL_TFLOPS * 1e6)) for s in shapes)
            out.append({"name": "16-layer stack, 64 calls, one batch in one CUDA graph", "M": M, "ec_on_8_calls": with_ec,
                        "us": round(us, 1), "gbs": round(by / us * 1e-3, 1), "tflops": round(fl / us * 1e-6, 2),
                        "sum_t_roof_measured_us": round(t_meas, 1), "frac_of_measured_roofline": round(t_meas / us, 4),
                        "frac_of_nominal_roofline": round(t_nom / us, 4)})
        del layers, xs, ys
        torch.cuda.empty_cache()
    return out


# ------------------------------------------------------------------------------------------------
# oracle legs (the only places bench.py executes oracle/): cpu_baseline and --impl reference
# ------------------------------------------------------------------------------------------------
def _oracle_pass(layers):
    """One oracle pass (dequantise + forward, fp64) over prepared LayerInputs; returns seconds."""
    import oracle
    t0 = time.perf_counter()
    for li in layers:
        oracle.forward_layer(li)
    return time.perf_counter() - t0


def _sample_layers(which):
    shapes = step_shapes()
    if which == "step":
        sel = [s for M in TOKENS for s in shapes[M]]
    elif which == "m1":
        sel = list(shapes[1])
    else:
        sel = [s for s in shapes[1] if s.name == "o"]
    layers = [make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar") for s in sel]
    nbytes = sum(algorithmic_bytes(s.M, s.N, s.K, s.group, s.r, "scalar") for s in sel)
    return layers, nbytes, sel


SAMPLE_TEXT = {"step": "the full step once: 12 layer calls (dequantise to fp64 + naive fp64 GEMM + gate + EC)",
               "m1": "the four projections at M=1 (dequantise to fp64 + naive fp64 GEMM + gate + EC)",
               "o": "the o projection (2048x2048) at M=1"}


def cpu_baseline_sample():
    import oracle
    oracle.build()
    layers, nbytes, _ = _sample_layers("step")
    _oracle_pass(layers[:1])                      # page in / thread pool start
    t = _oracle_pass(layers)
    return {"value": round(nbytes / t / 1e9, 4), "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": SAMPLE_TEXT["step"] + f"; {t:.2f} s wall", "seconds": round(t, 3)}


def run_reference(args, rank, world):
    if rank != 0:
        return
    import oracle
    oracle.build()
    # bounded sample per step, sized so warmup + steps ends within a few minutes
    layers, nbytes, _ = _sample_layers("m1")
    t_probe = _oracle_pass(layers)
    which = "m1"
    if t_probe * (args.steps + args.warmup) > 150.0:
        which = "o"
        layers, nbytes, _ = _sample_layers("o")
    for _ in range(args.warmup):
        _oracle_pass(layers)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        _oracle_pass(layers)
    t = (time.perf_counter() - t0) / args.steps
    v = round(nbytes / t / 1e9, 4)
    out = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": world, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": round(t * 1e3, 4), "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded, workloads/)",
           "config": {"workload": "BASELINE.json configs[1] (bounded sample per step: " + SAMPLE_TEXT[which] + ")",
                      "bytes_per_step": nbytes},
           "cpu_baseline": {"value": v, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                            "sample": SAMPLE_TEXT[which]},
           "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-table", action="store_true", help="skip the per-config result table (configs key)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuda" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_cuda(args, rank, world)


if __name__ == "__main__":
    main()
