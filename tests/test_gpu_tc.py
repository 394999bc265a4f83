"""GPU parity for the tcgen05 path (SPEAR_VARIANT_TC_FUSED, M > 16): libspear.so through the C ABI
against the fp64 CPU oracle on the same seeded inputs.  Small shapes compare every element; the
BASELINE.json prefill shapes compare all N columns of a seeded row sample (each y[m][:] depends on
x[m][:] only, so sampling rows is exact -- SURVEY.md 8(c) large-shape policy)."""
import numpy as np
import pytest

import oracle
from workloads import make_layer, config_shapes

pytestmark = pytest.mark.gpu

Y_TOL = 1e-2
GATE_TOL = 1e-3
TC = 3          # SPEAR_VARIANT_TC_FUSED
STREAM = 2      # SPEAR_VARIANT_STREAM_SPLIT


@pytest.fixture(scope="module")
def sp():
    import paper_2606_11244_b200 as sp
    sp.init()
    return sp


def _h():
    from paper_2606_11244_b200 import harness
    return harness


def sample_rows(M, seed, extra=48):
    """One seeded row per 128-row block + `extra` random rows + the first and last row."""
    rng = np.random.default_rng(seed)
    rows = {0, M - 1}
    for b in range(0, M, 128):
        rows.add(int(b + rng.integers(0, min(128, M - b))))
    rows.update(int(v) for v in rng.integers(0, M, size=extra))
    return np.array(sorted(rows))


def check(li, variant=TC, rows=None, label=""):
    import torch
    h = _h()
    dl = h.upload_layer(li)
    x = h.dev(li.x)
    y, gate = h.run_layer(dl, x, variant=variant, want_gate=True)
    torch.cuda.synchronize()
    yg = y.cpu().numpy().astype(np.float64)
    ref = oracle.forward_layer(li, rows=rows)
    yr = ref["y"]
    if rows is not None:
        yg = yg[rows]
    rms = float(np.sqrt(np.mean(yr ** 2)))
    err = float(np.max(np.abs(yg - yr)))
    assert np.all(np.isfinite(yg)), label
    assert err <= Y_TOL * rms, f"{label}: max err {err:.4g} > {Y_TOL} * rms {rms:.4g}"
    if gate is not None and ref["gam"] is not None:
        gg = gate.cpu().numpy().astype(np.float64)
        if rows is not None:
            gg = gg[rows]
        assert float(np.max(np.abs(gg - ref["gam"]))) <= GATE_TOL, label
    return y


@pytest.mark.parametrize("M", [17, 32, 33, 64, 100, 128, 129, 256, 300, 520])
def test_tc_token_counts(sp, M):
    # every token-tile width (32/64/128/256), ragged tails, several panels, K not a power of two
    li = make_layer(900 + M, M, 384, 640, 128, 24, gate="scalar")
    check(li, label=f"tc M={M}")


@pytest.mark.parametrize("r", [0, 8, 16, 64, 72, 128])
@pytest.mark.parametrize("gate", ["scalar", "mlp", "none"])
def test_tc_ranks_and_gates(sp, r, gate):
    if r == 0 and gate != "scalar":
        pytest.skip("r = 0 has no gate")
    li = make_layer(1000 + r, 200, 256, 512, 128, r, gate=gate)
    check(li, label=f"tc r={r} {gate}")


@pytest.mark.parametrize("group,K", [(128, 1024), (256, 1024), (1024, 1024), (1792, 1792)])
def test_tc_groups(sp, group, K):
    li = make_layer(1100 + group, 96, 256, K, group, 16, gate="scalar")
    check(li, label=f"tc group={group}")


def test_tc_many_tiles_per_cta(sp):
    # more tiles than SMs: exercises the persistent schedule, both TMEM accumulators and ring wrap-around
    li = make_layer(1200, 1100, 6144, 256, 128, 16, gate="scalar")
    check(li, rows=sample_rows(1100, 1), label="tc many tiles")


def test_tc_matches_stream_variant(sp):
    """P11: the same M = 16 problem through the decode kernel and through the tcgen05 kernel."""
    import torch
    h = _h()
    li = make_layer(1300, 16, 512, 1024, 128, 32, gate="mlp")
    dl = h.upload_layer(li)
    x = h.dev(li.x)
    ya, _ = h.run_layer(dl, x, variant=STREAM)
    yb, _ = h.run_layer(dl, x, variant=TC)
    ref = oracle.forward_layer(li)["y"]
    rms = float(np.sqrt(np.mean(ref ** 2)))
    assert float((ya.float() - yb.float()).abs().max()) <= Y_TOL * rms


def test_tc_gate_zero_is_plain_w4(sp):
    import torch
    h = _h()
    li = make_layer(1400, 150, 256, 512, 128, 16, gate="scalar")
    plain = make_layer(1400, 150, 256, 512, 128, 0)
    y0, _ = h.run_layer(h.upload_layer(plain), h.dev(plain.x), variant=TC)
    li.b_g = -100.0
    y1, _ = h.run_layer(h.upload_layer(li), h.dev(li.x), variant=TC)
    assert torch.equal(y0, y1)


def test_tc_back_to_back(sp):
    import torch
    h = _h()
    li = make_layer(1500, 260, 384, 1024, 128, 32, gate="scalar")
    dl = h.upload_layer(li)
    x = h.dev(li.x)
    ys = [h.run_layer(dl, x, variant=TC)[0].clone() for _ in range(4)]
    torch.cuda.synchronize()
    ref = oracle.forward_layer(li)["y"]
    rms = float(np.sqrt(np.mean(ref ** 2)))
    for y in ys:
        assert float(np.max(np.abs(y.cpu().numpy().astype(np.float64) - ref))) <= Y_TOL * rms


@pytest.mark.parametrize("idx", [6, 7, 8])
def test_config3_prefill_M256(sp, idx):
    s = config_shapes(2)[idx]
    assert s.M == 256
    li = make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar")
    check(li, variant=0, rows=sample_rows(s.M, s.seed, extra=16), label=f"config3 {s.name} M=256")


@pytest.mark.parametrize("idx", [9, 11])
def test_config3_prefill_M2048(sp, idx):
    s = config_shapes(2)[idx]
    assert s.M == 2048
    li = make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar")
    check(li, variant=0, rows=sample_rows(s.M, s.seed, extra=8), label=f"config3 {s.name} M=2048")


@pytest.mark.parametrize("r", [0, 64])
def test_config4_M512(sp, r):
    s = [c for c in config_shapes(3) if c.M == 512 and c.r == r][0]
    li = make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar")
    check(li, variant=0, rows=sample_rows(s.M, s.seed, extra=8), label=f"config4 M=512 r={r}")


@pytest.mark.parametrize("name", ["L0.qkv", "L0.o", "L0.gate_up", "L0.down", "L7.down"])
def test_config5_M64(sp, name):
    s = [c for c in config_shapes(4) if c.M == 64 and c.name == name][0]
    li = make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar")
    check(li, variant=0, label=f"config5 {name} M=64")


@pytest.mark.parametrize("ksplit", [2, 3, 7])
@pytest.mark.parametrize("M,r", [(40, 0), (64, 32), (200, 72)])
def test_tc_split_k(sp, ksplit, M, r):
    """Split-K arm of the tcgen05 kernel (fp32 partial slots + last-arriver reduction), forced through the
    tuning hook; repeated calls must leave the counters clean."""
    import torch
    li = make_layer(1600 + M + ksplit, M, 384, 1792, 128, r, gate="scalar")
    sp.tune("tc_ksplit", ksplit)
    try:
        check(li, label=f"tc split-K {ksplit} M={M} r={r}")
        check(li, label=f"tc split-K {ksplit} M={M} r={r} (second call)")
    finally:
        sp.tune("tc_ksplit", 0)


@pytest.mark.parametrize("M,r,gate", [(40, 16, "scalar"), (200, 72, "mlp"), (300, 128, "scalar"), (16, 32, "none")])
def test_tc_split_variant(sp, M, r, gate):
    """SPEAR_VARIANT_TC_SPLIT: plain W4 tcgen05 GEMM, then the rank-r update as its own pass over y (rounded
    twice, reading A8) -- still inside the y tolerance, and close to the fused arm."""
    li = make_layer(1800 + M, M, 384, 640, 128, r, gate=gate)
    y_split = check(li, variant=4, label=f"tc split M={M} r={r} {gate}")
    y_fused = check(li, variant=TC, label=f"tc fused M={M} r={r} {gate}")
    ref = oracle.forward_layer(li)["y"]
    rms = float(np.sqrt(np.mean(ref ** 2)))
    assert float((y_split.float() - y_fused.float()).abs().max()) <= Y_TOL * rms


def test_config4_M4096_r64_sampled_rows(sp):
    """The prefill shape bench.py times (configs[3]: M = 4096, K = 8192, N = 28672, r = 64) at full size: all N
    columns of a seeded sample of token rows against the oracle (rows are independent, so sampling is exact)."""
    s = [c for c in config_shapes(3) if c.M == 4096 and c.r == 64][0]
    li = make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar")
    rng = np.random.default_rng(s.seed)
    rows = np.array(sorted({0, s.M - 1, 255, 256, *[int(v) for v in rng.integers(0, s.M, size=8)]}))
    check(li, variant=0, rows=rows, label="config4 M=4096 r=64")


# ---------------------------------------------------------------- the remaining BASELINE.json config shapes (north_star: "on all 5 configs")

@pytest.mark.parametrize("M,r", [(4096, 16), (4096, 128), (16384, 0), (16384, 64)])
def test_config4_large_sampled_rows(sp, M, r):
    """configs[3] at the sizes not covered above: M = 4096 with r = 16 / 128 and M = 16384 with r = 0 / 64, all N
    columns of a seeded row sample (SURVEY.md 8(c) large-shape policy: rows are independent, sampling is exact)."""
    s = [c for c in config_shapes(3) if c.M == M and c.r == r][0]
    li = make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar")
    rng = np.random.default_rng(s.seed + 1)
    rows = np.array(sorted({0, M - 1, 127, 128, M // 2, *[int(v) for v in rng.integers(0, M, size=5)]}))
    check(li, variant=0, rows=rows, label=f"config4 M={M} r={r}")


def test_config3_gate_up_M2048(sp):
    s = config_shapes(2)[10]
    assert s.M == 2048 and s.name == "gate_up"
    li = make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar")
    check(li, variant=0, rows=sample_rows(s.M, s.seed, extra=4)[::2], label="config3 gate_up M=2048")


@pytest.mark.parametrize("M", [64, 2048])
def test_config5_full_stack_one_batch_in_a_graph(sp, M):
    """configs[4]: the whole 64-call projection stack (16 layers x {qkv, o, gate_up, down}, EC r = 32 on o / down of layers
    {0, 1, 14, 15}, reading A11), issued as ONE spear_w4_ec_gemm_batch captured in a CUDA graph -- the way bench.py
    times it -- and every call compared with the oracle (all rows at M = 64, a row sample at M = 2048)."""
    import torch
    h = _h()
    shapes = [c for c in config_shapes(4) if c.M == M]
    assert len(shapes) == 64 and sum(1 for c in shapes if c.r > 0) == 8
    lis = [make_layer(c.seed, c.M, c.N, c.K, c.group, c.r, gate="scalar") for c in shapes]
    dls = [h.upload_layer(li) for li in lis]
    xs = [h.dev(li.x) for li in lis]
    ys = [torch.zeros((li.M, li.N), dtype=torch.float16, device="cuda") for li in lis]
    descs = [dl.desc() if li.r else sp.make_desc(gate="none") for dl, li in zip(dls, lis)]
    batch = sp.Batch([(x, dl.pw, dl.A if li.r else None, dl.B if li.r else None, d, y)
                      for x, dl, li, d, y in zip(xs, dls, lis, descs, ys)])
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        sp.w4_ec_gemm_batch(batch, stream=st)
        torch.cuda.synchronize()
        for y in ys:
            y.zero_()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            sp.w4_ec_gemm_batch(batch, stream=st)
        g.replay()
        torch.cuda.synchronize()
    rows = None if M == 64 else np.array([0, 700, M - 1])
    for c, li, y in zip(shapes, lis, ys):
        ref = oracle.forward_layer(li, rows=rows)["y"]
        yg = y.cpu().numpy().astype(np.float64)
        if rows is not None:
            yg = yg[rows]
        rms = float(np.sqrt(np.mean(ref ** 2)))
        assert float(np.max(np.abs(yg - ref))) <= Y_TOL * rms, c.name


@pytest.mark.parametrize("cfg,name,M", [(1, "gate_up", 8), (2, "qkv", 256)])
def test_paper_mlp_gate_on_config_shapes(sp, cfg, name, M):
    """The paper's own gate (gamma = 1 + tanh(W2 ReLU(W1 z + b1) + b2), h = 4r, reading A2) on one decode and
    one prefill shape of the configs -- the configs themselves use the scalar gate (reading A1)."""
    s = [c for c in config_shapes(cfg) if c.name == name and c.M == M][0]
    li = make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="mlp")
    rng = np.random.default_rng(3)
    li.b1 = (rng.integers(-8, 9, li.W1.shape[0]) / 16.0).astype(np.float32)      # non-zero biases: the ReLU clips
    li.b2 = (rng.integers(-4, 5, li.r) / 16.0).astype(np.float32)
    check(li, variant=0, label=f"MLP gate, config {cfg + 1} {name} M={M}")


def test_cluster_of_four_instance(sp):
    """tc_kernel<256, 4>: four CTAs share the token tile by TMA multicast (reachable through spear_tune only)."""
    li = make_layer(1900, 520, 1024, 640, 128, 24, gate="scalar")
    sp.tune("tc_cluster", 4)
    sp.tune("tc_bt", 256)
    try:
        check(li, label="cluster 4")
    finally:
        sp.tune("tc_cluster", 0)
        sp.tune("tc_bt", 0)


def test_tc_grid_and_tile_overrides(sp):
    li = make_layer(1901, 300, 512, 640, 128, 16, gate="scalar")
    for bt in (128, 256):
        sp.tune("tc_bt", bt)
        sp.tune("tc_grid", 7)
        try:
            check(li, label=f"tc_bt={bt} tc_grid=7")
        finally:
            sp.tune("tc_bt", 0)
            sp.tune("tc_grid", 0)


def test_single_call_hostio(sp):
    """spear_w4_ec_gemm_hostio: pinned host x -> device -> layer -> pinned host y on one stream."""
    import torch
    h = _h()
    for (M, N, K, r) in [(4, 512, 768, 16), (100, 384, 640, 8)]:
        li = make_layer(1950 + M, M, N, K, 128, r, gate="scalar")
        dl = h.upload_layer(li)
        xh = torch.from_numpy(li.x).pin_memory()
        yh = torch.zeros((M, N), dtype=torch.float16).pin_memory()
        xd = torch.empty((M, K), dtype=torch.float16, device="cuda")
        yd = torch.empty((M, N), dtype=torch.float16, device="cuda")
        sp.w4_ec_gemm_hostio(xh, yh, xd, yd, dl.pw, dl.A, dl.B, dl.desc())
        torch.cuda.synchronize()
        ref = oracle.forward_layer(li)["y"]
        rms = float(np.sqrt(np.mean(ref ** 2)))
        assert float(np.max(np.abs(yh.numpy().astype(np.float64) - ref))) <= Y_TOL * rms


@pytest.mark.parametrize("M,r", [(256, 32), (512, 0), (512, 64)])
def test_split_tail_of_a_partial_last_wave(sp, M, r):
    """150 panels: one more wave than the 148 SMs (M = 256, single CTAs: 150 tiles) or than the 74 CTA pairs (M = 512, clusters
    of 2: 150 cluster tiles) hold -- the 2 tiles of the last, nearly empty wave are split along K over idle CTAs (fp32 partial
    slots + last-arriver sum, also with the cluster variant and with the EC k-blocks riding on the last share).  Sampled rows
    against the oracle, with the split on and off, and twice in a row (the tile counters must come back to zero)."""
    N, K = 128 * 150, 4096
    li = make_layer(700 + M + r, M, N, K, 128, r, gate="scalar")
    rows = np.array(sorted({0, 1, M - 1, M // 2, 255, min(256, M - 1)}))
    try:
        for tail in (1, 1, 0):
            sp.tune("tc_tail", tail)
            check(li, variant=0, rows=rows, label=f"split tail={tail} M={M} r={r}")
    finally:
        sp.tune("tc_tail", 1)
