"""GPU parity of the row-strip decode kernel (csrc/rows.cu, SPEAR_VARIANT_ROWS) against the fp64 CPU oracle, through
the C ABI.  One CTA per 16 output rows over the whole of K; the EC term comes from the EC pre-kernel (any gate).
Bars: max|y - y_ref| <= 1e-2 * rms(y_ref); gate within 1e-3 (BASELINE.json north_star)."""
import numpy as np
import pytest

import oracle
from workloads import make_layer, config_shapes, with_int8_ec

pytestmark = pytest.mark.gpu

Y_TOL = 1e-2
GATE_TOL = 1e-3


@pytest.fixture(scope="module")
def sp():
    import paper_2606_11244_b200 as sp
    sp.init()
    return sp


def check(sp, li, label):
    import torch
    from paper_2606_11244_b200 import harness as h
    dl = h.upload_layer(li)
    y, gate = h.run_layer(dl, h.dev(li.x), variant=sp.VARIANT_ROWS, want_gate=True)
    torch.cuda.synchronize()
    ref = oracle.forward_layer(li)
    yg = y.cpu().numpy().astype(np.float64)
    rms = float(np.sqrt(np.mean(ref["y"] ** 2)))
    err = float(np.max(np.abs(yg - ref["y"])))
    assert np.all(np.isfinite(yg)), label
    assert err <= Y_TOL * rms, f"{label}: max err {err:.4g} > {Y_TOL} * rms {rms:.4g}"
    if gate is not None and ref["gam"] is not None:
        gerr = float(np.max(np.abs(gate.cpu().numpy().astype(np.float64) - ref["gam"])))
        assert gerr <= GATE_TOL, f"{label}: gate err {gerr:.3g}"


def test_config1(sp):
    s = config_shapes(0)[0]
    check(sp, make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar"), "config 1")
    check(sp, make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="mlp"), "config 1, the paper's MLP gate")


@pytest.mark.parametrize("idx", range(12))
def test_config2_every_shape(sp, idx):
    s = config_shapes(1)[idx]
    check(sp, make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar"), f"config 2 {s.name} M={s.M}")


@pytest.mark.parametrize("name,M", [("qkv", 1), ("down", 16), ("gate_up", 1)])
def test_config3_per_channel(sp, name, M):
    s = [c for c in config_shapes(2) if c.name == name and c.M == M][0]
    check(sp, make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar"), f"config 3 {name} M={M}")      # group == K


@pytest.mark.parametrize("M", [1, 2, 3, 5, 8, 9, 11, 13, 16])
def test_ragged_token_counts(sp, M):
    # K = 640: ten 64-column k-tiles over eight warps (a ragged batch), three panels
    check(sp, make_layer(340 + M, M, 384, 640, 128, 24, gate="scalar"), f"M={M}")


@pytest.mark.parametrize("r,gate", [(0, "none"), (8, "scalar"), (16, "none"), (64, "mlp"), (128, "scalar")])
def test_ranks_and_gates(sp, r, gate):
    check(sp, make_layer(360 + r, 7, 512, 1024, 128, r, gate=gate), f"r={r} gate={gate}")


@pytest.mark.parametrize("group,K", [(256, 1024), (384, 768), (1024, 1024), (128, 128), (1792, 1792), (128, 4608)])
def test_group_sizes_and_k_tails(sp, group, K):
    check(sp, make_layer(370, 4, 256, K, group, 8, gate="scalar"), f"group={group} K={K}")


@pytest.mark.parametrize("M", [4, 16])
def test_int8_ec_factors(sp, M):
    li = with_int8_ec(make_layer(380 + M, M, 2048, 2048, 128, 32, gate="scalar"))
    check(sp, li, f"INT8 EC M={M}")


@pytest.mark.parametrize("rows_ec", [0, 1, 2])
@pytest.mark.parametrize("shape", [(8, 2048, 2048, 128, 32, "scalar"), (16, 3072, 2048, 128, 32, "scalar"), (1, 512, 8192, 128, 128, "scalar"),
                                   (13, 384, 640, 128, 24, "none"), (5, 256, 128, 128, 8, "scalar"), (16, 6144, 4096, 4096, 64, "scalar")])
def test_both_ec_arms(sp, rows_ec, shape):
    """The row-strip kernel's EC for the scalar / none gate has two arms (spear_tune "rows_ec"): z recomputed by every cluster inside
    the layer kernel (0), once by the one-cluster pre-kernel ecz_cluster_kernel that the layer kernel overlaps (1), or as eight partial
    z parked in the workspace by 8 independent pre-kernel CTAs and summed + gated by the layer kernel (2, the default).  All, on
    shapes that cover ragged tokens, one k-tile per CTA of the cluster (K = 128 ... 640), r = 128, per-channel scales."""
    M, N, K, group, r, gate = shape
    sp.tune("rows_ec", rows_ec)
    try:
        check(sp, make_layer(400 + M + r, M, N, K, group, r, gate=gate), f"rows_ec={rows_ec} {shape}")
        check(sp, with_int8_ec(make_layer(401 + M + r, M, N, K, group, r, gate=gate)), f"rows_ec={rows_ec} int8 {shape}")
    finally:
        sp.tune("rows_ec", 2)


def test_stream_ordered_in_a_graph(sp):
    """Back-to-back calls in one CUDA graph (programmatic dependent launch between them), replayed."""
    import torch
    from paper_2606_11244_b200 import harness as h
    lis = [make_layer(390 + i, 8, 2048, 2048, 128, 32, gate="scalar") for i in range(4)]
    dls = [h.upload_layer(li) for li in lis]
    xs = [h.dev(li.x) for li in lis]
    ys = [torch.zeros((8, 2048), dtype=torch.float16, device="cuda:0") for _ in lis]
    ds = [dl.desc(variant=sp.VARIANT_ROWS) for dl in dls]

    def step():
        for x, dl, d, y in zip(xs, dls, ds, ys):
            sp.w4_ec_gemm_ex(x, dl.pw, dl.A, dl.B, d, y=y)

    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        step()
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            step()
        for y in ys:
            y.zero_()
        for _ in range(20):
            g.replay()
    torch.cuda.synchronize()
    for li, y in zip(lis, ys):
        ref = oracle.forward_layer(li)["y"]
        rms = float(np.sqrt(np.mean(ref ** 2)))
        assert float(np.max(np.abs(y.cpu().numpy().astype(np.float64) - ref))) <= Y_TOL * rms


@pytest.mark.parametrize("M", [17, 31, 32, 33, 48, 64])
@pytest.mark.parametrize("shape", [(3072, 2048, 128, 32, "scalar"), (2048, 8192, 128, 32, "scalar"), (384, 640, 128, 24, "mlp"),
                                   (256, 1792, 1792, 0, "none"), (512, 1024, 256, 128, "none")])
def test_mid_token_counts(sp, M, shape):
    """The 32-token form of the strip kernel (17..64 tokens; u as fp16 from the M > 16 EC pre-pass): config-5-sized layers, ragged
    token blocks, K not a multiple of 512, per-channel scales, every gate, r = 0 and r = 128."""
    N, K, group, r, gate = shape
    check(sp, make_layer(500 + M + r, M, N, K, group, r, gate=gate), f"mid-M M={M} {shape}")


def test_mid_token_counts_refuse_int8_when_forced_and_fall_back_on_auto(sp):
    import torch
    from paper_2606_11244_b200 import harness as h
    li = with_int8_ec(make_layer(560, 40, 512, 1024, 128, 16, gate="scalar"))
    dl = h.upload_layer(li)
    with pytest.raises(sp.SpearError):
        h.run_layer(dl, h.dev(li.x), variant=sp.VARIANT_ROWS)
    y, _ = h.run_layer(dl, h.dev(li.x))                # AUTO serves it (tcgen05 path with the factors dequantised to fp16 scratch)
    torch.cuda.synchronize()
    ref = oracle.forward_layer(li)["y"]
    assert float(np.max(np.abs(y.cpu().numpy().astype(np.float64) - ref))) <= Y_TOL * float(np.sqrt(np.mean(ref ** 2)))
