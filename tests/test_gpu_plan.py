"""S9 on the GPU: spear_plan measures the valid variants of a problem, records the fastest, spear_plan_query
returns it, the table survives save / load, and the planned variant still matches the oracle."""
import os
import numpy as np
import pytest

import oracle
from workloads import make_layer

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sp():
    import paper_2606_11244_b200 as sp
    sp.init()
    return sp


def test_plan_decode_times_fused_and_split(sp, tmp_path):
    chosen, us = sp.plan(8, 2048, 2048, 32, 128, gate="scalar")
    # every decode arm is a candidate and is timed: ring kernel fused / split, row-strip kernel; the fastest is recorded
    assert chosen in (sp.VARIANT_STREAM_FUSED, sp.VARIANT_STREAM_SPLIT, sp.VARIANT_ROWS, sp.VARIANT_LSTREAM)
    assert us[sp.VARIANT_STREAM_FUSED] > 0 and us[sp.VARIANT_STREAM_SPLIT] > 0 and us[sp.VARIANT_ROWS] > 0
    assert us[chosen] == min(t for t in us if t > 0)
    assert sp.plan_query(8, 2048, 2048, 32, 128, gate="scalar") == chosen
    # the MLP gate has no fused decode arm: the plan must fall on the split one
    chosen_mlp, us_mlp = sp.plan(8, 2048, 2048, 32, 128, gate="mlp", gate_hidden=128)
    assert chosen_mlp in (sp.VARIANT_STREAM_SPLIT, sp.VARIANT_ROWS) and us_mlp[sp.VARIANT_STREAM_FUSED] < 0      # both go through the EC pre-kernel
    path = str(tmp_path / "plan.txt")
    sp.plan_save(path)
    txt = open(path).read()
    assert "8 2048 2048 32 128" in txt
    sp.plan_load(path)
    assert sp.plan_query(8, 2048, 2048, 32, 128, gate="scalar") == chosen


def test_plan_crossover_shapes(sp):
    # M <= 16: the decode kernels and the tcgen05 kernel are all valid; 17..64 tokens: the tcgen05 arms and the strip kernel's
    # 32-token form, never the ring kernel; above 64 tokens only the tcgen05 arms
    chosen, us = sp.plan(16, 4096, 4096, 64, 4096, gate="scalar")
    assert us[sp.VARIANT_TC_FUSED] > 0 and us[sp.VARIANT_STREAM_FUSED] > 0 and us[sp.VARIANT_ROWS] > 0
    chosen64, us64 = sp.plan(64, 2048, 2048, 32, 128, gate="scalar")
    assert chosen64 in (sp.VARIANT_TC_FUSED, sp.VARIANT_TC_SPLIT, sp.VARIANT_ROWS) and us64[sp.VARIANT_STREAM_FUSED] < 0
    assert us64[sp.VARIANT_TC_FUSED] > 0 and us64[sp.VARIANT_TC_SPLIT] > 0 and us64[sp.VARIANT_ROWS] > 0
    assert us64[chosen64] == min(t for t in us64 if t > 0)
    chosen96, us96 = sp.plan(96, 2048, 2048, 32, 128, gate="scalar")
    assert chosen96 in (sp.VARIANT_TC_FUSED, sp.VARIANT_TC_SPLIT) and us96[sp.VARIANT_ROWS] < 0 and us96[sp.VARIANT_STREAM_FUSED] < 0


def test_planned_variant_matches_oracle(sp):
    import torch
    from paper_2606_11244_b200 import harness as h
    li = make_layer(1700, 16, 512, 1024, 128, 16, gate="scalar")
    sp.plan(li.M, li.N, li.K, li.r, li.group, gate="scalar")
    y, _ = h.run_layer(h.upload_layer(li), h.dev(li.x))          # AUTO -> the planned variant
    torch.cuda.synchronize()
    ref = oracle.forward_layer(li)["y"]
    rms = float(np.sqrt(np.mean(ref ** 2)))
    assert float(np.max(np.abs(y.cpu().numpy().astype(np.float64) - ref))) <= 1e-2 * rms


def test_lut_measure_feeds_the_chunk_selector(sp):
    """SURVEY.md 8(f)4 end to end on the device: spear_lut_measure fills l_W4 / l_EC of one layer type from the library's own
    timings, the LUT built from them agrees with the oracle's linear scan."""
    from oracle import sched_oracle as so
    grid = [1, 16, 64, 256]
    w4, ec = sp.lut_measure(grid, 1024, 1024, 128, 32, gate="scalar")
    assert len(w4) == len(ec) == 4 and all(t > 0 for t in w4 + ec)
    assert all(e >= 0.5 * w for w, e in zip(w4, ec)), "an EC layer cannot be much faster than the plain one"
    assert max(w4) < 5000 and max(ec) < 5000, "microseconds, not another unit"
    lut = sp.Lut(grid, [w4], [ec])
    types, sel = [0] * 8, [True, False] * 4
    # a table entry is reproduced at its grid point (after the running maximum both sides apply)
    mw, me = so.monotone(w4), so.monotone(ec)
    assert abs(lut.iteration_us(types, sel, 64) - 4 * (mw[2] + me[2])) <= 1e-3 * 4 * (mw[2] + me[2])
    t16 = lut.iteration_us(types, sel, 16)
    for slo_factor in (1.5, 3.0, 10.0):
        want = so.slo_chunk(grid, [w4], [ec], None, types, sel, 0, 16, 1, 512, slo_factor * t16)
        got = lut.slo_chunk(types, sel, 16, 1, 512, slo_factor * t16)
        assert got == want, (slo_factor, got, want)
