"""GPU parity: libspear.so (through the C ABI) against the fp64 CPU oracle, element by element, on
the same seeded inputs.  Bars (BASELINE.json north_star): packed bytes and dequantised fp16
bit-exact; max|y - y_ref| <= 1e-2 * rms(y_ref); gate within 1e-3 absolute."""
import numpy as np
import pytest

import oracle
from workloads import make_layer, config_shapes

pytestmark = pytest.mark.gpu

Y_TOL = 1e-2      # x rms(y_ref)
GATE_TOL = 1e-3   # absolute


@pytest.fixture(scope="module")
def sp():
    import paper_2606_11244_b200 as sp
    sp.init()
    return sp


def _harness():
    from paper_2606_11244_b200 import harness
    return harness


def check_layer(li, variant=0, rows=None, use_14arg=False, label=""):
    """Runs the layer on the GPU and compares against the oracle (all rows, or the given rows)."""
    import torch
    h = _harness()
    dl = h.upload_layer(li)
    x = h.dev(li.x)
    y, gate = h.run_layer(dl, x, variant=variant, want_gate=True, use_14arg=use_14arg)
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
        gerr = float(np.max(np.abs(gg - ref["gam"])))
        assert gerr <= GATE_TOL, f"{label}: gate err {gerr:.3g}"
    return err / rms


# ---------------------------------------------------------------- S0: pack / unpack / dequant, bit-exact

@pytest.mark.parametrize("N,K,group", [(128, 128, 128), (256, 384, 128), (384, 512, 256), (2048, 2048, 128),
                                       (256, 1792, 1792), (3072, 2048, 128)])
def test_pack_bit_exact(sp, N, K, group):
    import torch
    h = _harness()
    li = make_layer(11 + N + K, 1, N, K, group, 0)
    pw = sp.pack_w4(h.dev(li.codes), h.dev(li.scales), group)
    wq_ref, sc_ref = oracle.pack_w4(li.codes, li.scales, group)
    assert np.array_equal(pw.wq.cpu().numpy().view(np.uint32), wq_ref)
    assert np.array_equal(pw.scales.cpu().numpy().view(np.uint16), sc_ref.view(np.uint16))
    assert np.array_equal(sp.unpack_w4(pw).cpu().numpy(), li.codes)
    dq = sp.dequant_w4(pw).cpu().numpy()
    assert np.array_equal(dq.view(np.uint16), oracle.dequant16(li.codes, li.scales, group).view(np.uint16))


def test_pack_structured_codes(sp):
    h = _harness()
    N, K = 256, 256
    n, k = np.meshgrid(np.arange(N), np.arange(K), indexing="ij")
    codes = ((n + k) & 15).astype(np.uint8)
    scales = np.full((N, 2), 1.0, np.float16)
    pw = sp.pack_w4(h.dev(codes), h.dev(scales), 128)
    wq_ref, _ = oracle.pack_w4(codes, scales, 128)
    assert np.array_equal(pw.wq.cpu().numpy().view(np.uint32), wq_ref)
    # a single non-8 nibble walking through one tile
    for (nn, kk) in [(0, 0), (7, 63), (8, 64), (127, 127), (128, 1), (200, 255), (15, 9)]:
        c = np.full((N, K), 8, np.uint8)
        c[nn, kk] = 3
        pw = sp.pack_w4(h.dev(c), h.dev(scales), 128)
        assert np.array_equal(sp.unpack_w4(pw).cpu().numpy(), c)
        ref, _ = oracle.pack_w4(c, scales, 128)
        assert np.array_equal(pw.wq.cpu().numpy().view(np.uint32), ref)


def test_pack_rejects_bad_code(sp):
    h = _harness()
    c = np.full((128, 128), 8, np.uint8)
    c[5, 77] = 16
    with pytest.raises(sp.SpearError) as e:
        sp.pack_w4(h.dev(c), h.dev(np.ones((128, 1), np.float16)), 128)
    assert e.value.status == -1


def test_dequant_all_codes_and_scales(sp):
    """P7 on the GPU: every code x scales incl. 1e-3, 1, powers of two, full-mantissa values."""
    h = _harness()
    N, K = 128, 128
    scales = np.array([1e-3, 1.0, 0.5, 2.0, 0.02, 0.0123, 1.9990234375, 6.1e-5] * 16, np.float16).reshape(N, 1)
    codes = ((np.arange(N)[:, None] + np.arange(K)[None, :]) & 15).astype(np.uint8)
    pw = sp.pack_w4(h.dev(codes), h.dev(scales), 128)
    dq = sp.dequant_w4(pw).cpu().numpy()
    assert np.array_equal(dq.view(np.uint16), oracle.dequant16(codes, scales, 128).view(np.uint16))


# ---------------------------------------------------------------- decode path (M <= 16)

def test_config1_scalar_gate(sp):
    s = config_shapes(0)[0]
    li = make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar")
    check_layer(li, label="config1")
    check_layer(li, use_14arg=True, label="config1/14arg")


def test_config1_mlp_gate(sp):
    s = config_shapes(0)[0]
    for hh in (None, 2 * s.r, s.r):
        li = make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="mlp", h=hh)
        check_layer(li, label=f"config1/mlp h={hh}")


@pytest.mark.parametrize("M", [1, 2, 3, 5, 8, 9, 13, 16])
@pytest.mark.parametrize("gate", ["scalar", "mlp", "none"])
def test_decode_small_shapes(sp, M, gate):
    # several panels / chunks, ragged token counts, K not a power of two
    li = make_layer(100 + M, M, 384, 640, 128, 24, gate=gate)
    check_layer(li, label=f"decode M={M} {gate}")


@pytest.mark.parametrize("r", [0, 8, 16, 32, 64, 128])
def test_decode_ranks(sp, r):
    li = make_layer(200 + r, 7, 512, 1024, 128, r, gate="scalar")
    check_layer(li, label=f"decode r={r}")


@pytest.mark.parametrize("group,K", [(128, 1024), (256, 1024), (1024, 1024), (1792, 1792)])
def test_decode_groups(sp, group, K):
    li = make_layer(300 + group, 4, 256, K, group, 16, gate="scalar")
    check_layer(li, label=f"decode group={group}")


@pytest.mark.parametrize("idx", range(12))
def test_config2_llama1b_decode(sp, idx):
    s = config_shapes(1)[idx]
    li = make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar")
    check_layer(li, label=f"config2 {s.name} M={s.M}")


@pytest.mark.parametrize("idx", range(12))
def test_config2_plain_w4_every_shape(sp, idx):
    """The plain-W4 leg of the bench step (r = 0), every call, through AUTO: row-strip kernel on qkv / o / down (M <= 8),
    ring kernel on gate_up and down at M = 16."""
    s = config_shapes(1)[idx]
    li = make_layer(s.seed, s.M, s.N, s.K, s.group, 0, gate="none")
    check_layer(li, label=f"config2 plain {s.name} M={s.M}")


@pytest.mark.parametrize("idx", [0, 1, 2, 3, 4, 5])
def test_config3_per_channel_decode(sp, idx):
    s = config_shapes(2)[idx]       # M = 1 and 16, per-channel scales (group = K)
    li = make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar")
    check_layer(li, label=f"config3 {s.name} M={s.M}")


# ---------------------------------------------------------------- invariants on the GPU (P2, P6)

def test_gate_zero_or_A_zero_is_plain_w4(sp):
    import torch
    h = _harness()
    li = make_layer(77, 6, 256, 512, 128, 16, gate="scalar")
    plain = make_layer(77, 6, 256, 512, 128, 0)
    y0, _ = h.run_layer(h.upload_layer(plain), h.dev(plain.x))
    li.b_g = -100.0                                   # sigmoid(-100 + small) == 0 in fp32
    y1, g1 = h.run_layer(h.upload_layer(li), h.dev(li.x), want_gate=True)
    assert float(g1.abs().max()) < 1e-30
    assert torch.equal(y0, y1)
    li.b_g = 0.0
    li.A = np.zeros_like(li.A)
    y2, _ = h.run_layer(h.upload_layer(li), h.dev(li.x))
    assert torch.equal(y0, y2)


def test_token_permutation_equivariance(sp):
    import torch
    h = _harness()
    li = make_layer(78, 8, 256, 512, 128, 16, gate="mlp")
    dl = h.upload_layer(li)
    x = h.dev(li.x)
    perm = torch.tensor([3, 0, 7, 1, 6, 2, 5, 4], device=x.device)
    y, g = h.run_layer(dl, x, want_gate=True)
    yp, gp = h.run_layer(dl, x[perm].contiguous(), want_gate=True)
    assert torch.allclose(yp.float(), y[perm].float(), atol=2e-2, rtol=2e-3)
    assert torch.allclose(gp, g[perm], atol=1e-5)


def test_back_to_back_calls_leave_workspace_clean(sp):
    """The library's counters / z accumulators must be zero again after every call."""
    import torch
    h = _harness()
    li = make_layer(79, 16, 384, 2048, 128, 32, gate="scalar")
    dl = h.upload_layer(li)
    x = h.dev(li.x)
    ys = [h.run_layer(dl, x)[0].clone() for _ in range(5)]
    torch.cuda.synchronize()
    ref = oracle.forward_layer(li)["y"]
    rms = float(np.sqrt(np.mean(ref ** 2)))
    for y in ys:
        # z is reduced with fp32 red.add, so the last bit may differ run to run; a dirty workspace
        # (stale z, counters) would be off by whole EC terms
        assert float(np.max(np.abs(y.cpu().numpy().astype(np.float64) - ref))) <= Y_TOL * rms
        assert float((y.float() - ys[0].float()).abs().max()) <= 1e-3 * rms


def test_errors(sp):
    import torch
    h = _harness()
    li = make_layer(80, 4, 128, 128, 128, 8, gate="scalar")
    dl = h.upload_layer(li)
    x = h.dev(li.x)
    with pytest.raises(sp.SpearError) as e:      # r not a multiple of 8
        sp.w4_ec_gemm(x, dl.pw, dl.A[:4].contiguous(), dl.B[:, :4].contiguous(), dl.w_g, dl.b_g)
    assert e.value.status == -2
    with pytest.raises(sp.SpearError) as e:      # missing gate weights
        sp.w4_ec_gemm(x, dl.pw, dl.A, dl.B, None, None)
    assert e.value.status == -1


# ---------------------------------------------------------------- fused vs split EC on the decode path (S9 arms)

@pytest.mark.parametrize("variant", [1, 2])      # SPEAR_VARIANT_STREAM_FUSED, SPEAR_VARIANT_STREAM_SPLIT
@pytest.mark.parametrize("M,N,K,r,gate", [(1, 256, 512, 8, "scalar"), (4, 2048, 2048, 16, "scalar"),
                                          (16, 384, 640, 24, "none"), (9, 3072, 2048, 32, "scalar"),
                                          (16, 2048, 8192, 128, "scalar"), (3, 128, 128, 64, "scalar")])
def test_decode_fused_and_split(sp, variant, M, N, K, r, gate):
    li = make_layer(400 + M + r, M, N, K, 128, r, gate=gate)
    check_layer(li, variant=variant, label=f"variant {variant} M={M} r={r} {gate}")


def test_fused_variant_rejects_mlp_gate(sp):
    h = _harness()
    li = make_layer(81, 4, 128, 128, 128, 8, gate="mlp")
    with pytest.raises(sp.SpearError) as e:
        h.run_layer(h.upload_layer(li), h.dev(li.x), variant=1)
    assert e.value.status == -2


def test_fused_back_to_back_leaves_workspace_clean(sp):
    import torch
    h = _harness()
    li = make_layer(82, 16, 384, 2048, 128, 32, gate="scalar")
    dl = h.upload_layer(li)
    x = h.dev(li.x)
    ys = [h.run_layer(dl, x, variant=1)[0].clone() for _ in range(6)]
    torch.cuda.synchronize()
    ref = oracle.forward_layer(li)["y"]
    rms = float(np.sqrt(np.mean(ref ** 2)))
    for y in ys:
        assert float(np.max(np.abs(y.cpu().numpy().astype(np.float64) - ref))) <= Y_TOL * rms


# ---------------------------------------------------------------- batch of independent calls (concurrent lanes)

def test_batch_matches_oracle_and_single_calls(sp):
    """spear_w4_ec_gemm_batch over mixed shapes / token counts (decode, mid-M, plain and EC): each call
    must equal the oracle, also inside a CUDA graph replayed several times."""
    import torch
    h = _harness()
    specs = [(1, 256, 512, 16, "scalar"), (16, 384, 640, 24, "scalar"), (8, 2048, 2048, 0, "scalar"),
             (4, 512, 1024, 32, "mlp"), (40, 256, 512, 16, "scalar"), (3, 128, 128, 8, "none"), (16, 3072, 2048, 32, "scalar")]
    lis = [make_layer(500 + i, M, N, K, 128, r, gate=g) for i, (M, N, K, r, g) in enumerate(specs)]
    dls = [h.upload_layer(li) for li in lis]
    xs = [h.dev(li.x) for li in lis]
    ys = [torch.zeros((li.M, li.N), dtype=torch.float16, device="cuda:0") for li in lis]
    batch = sp.Batch([(x, dl.pw, dl.A, dl.B, dl.desc(), y) for x, dl, y in zip(xs, dls, ys)])
    sp.w4_ec_gemm_batch(batch)
    torch.cuda.synchronize()
    refs = [oracle.forward_layer(li)["y"] for li in lis]

    def verify(tag):
        for li, y, ref in zip(lis, ys, refs):
            rms = float(np.sqrt(np.mean(ref ** 2)))
            err = float(np.max(np.abs(y.cpu().numpy().astype(np.float64) - ref)))
            assert err <= Y_TOL * rms, f"{tag}: M={li.M} N={li.N} r={li.r}: {err:.4g} > {Y_TOL} * {rms:.4g}"
    verify("eager")
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            sp.w4_ec_gemm_batch(batch)
        for y in ys:
            y.zero_()
        for _ in range(3):
            g.replay()
    torch.cuda.synchronize()
    verify("graph")


def test_batch_hostio_matches_oracle(sp):
    """spear_w4_ec_gemm_batch_hostio: pinned-host x in, pinned-host y out, per call, on the lanes."""
    import torch
    h = _harness()
    specs = [(1, 256, 512, 16, "scalar"), (16, 384, 640, 24, "scalar"), (40, 256, 512, 16, "scalar"), (8, 2048, 2048, 0, "scalar")]
    lis = [make_layer(600 + i, M, N, K, 128, r, gate=g) for i, (M, N, K, r, g) in enumerate(specs)]
    dls = [h.upload_layer(li) for li in lis]
    xs = [torch.zeros((li.M, li.K), dtype=torch.float16, device="cuda:0") for li in lis]      # staging buffers
    ys = [torch.zeros((li.M, li.N), dtype=torch.float16, device="cuda:0") for li in lis]
    xh = [torch.from_numpy(li.x).pin_memory() for li in lis]
    yh = [torch.zeros((li.M, li.N), dtype=torch.float16).pin_memory() for li in lis]
    batch = sp.Batch([(x, dl.pw, dl.A, dl.B, dl.desc(), y) for x, dl, y in zip(xs, dls, ys)])
    sp.w4_ec_gemm_batch_hostio(batch, xh, yh)
    torch.cuda.synchronize()
    for li, y in zip(lis, yh):
        ref = oracle.forward_layer(li)["y"]
        rms = float(np.sqrt(np.mean(ref ** 2)))
        assert float(np.max(np.abs(y.numpy().astype(np.float64) - ref))) <= Y_TOL * rms


# ---------------------------------------------------------------- degenerate sizes

@pytest.mark.parametrize("M,N,K,group,r,gate", [
    (1, 128, 128, 128, 8, "scalar"),       # one unit, one CTA: the device-wide EC arrive / wait with a grid of 1
    (16, 128, 128, 128, 128, "scalar"),    # maximum rank on the smallest layer
    (5, 128, 1152, 128, 16, "scalar"),     # odd chunk count: the panel's tail unit holds a single chunk
    (16, 256, 1152, 384, 24, "none"),      # group of three chunks: a unit's two chunks fall in different groups
    (2, 128, 128, 128, 0, "scalar"),       # plain W4, smallest
    (9, 18432, 256, 128, 8, "scalar"),     # more panels than CTAs, whole panels per CTA
])
@pytest.mark.parametrize("variant", [0, 2, 3])
def test_degenerate_shapes(sp, M, N, K, group, r, gate, variant):
    li = make_layer(700 + M + N + K, M, N, K, group, r, gate=gate)
    check_layer(li, variant=variant, label=f"degenerate M={M} N={N} K={K} g={group} r={r} v={variant}")


def test_empty_and_misaligned_inputs_are_rejected(sp):
    """Edge cases of the boundary: no tokens, a misaligned activation pointer, an unsupported shape."""
    import torch
    h = _harness()
    li = make_layer(90, 4, 128, 128, 128, 0)
    dl = h.upload_layer(li)
    with pytest.raises(sp.SpearError) as e:                      # M = 0
        sp.w4_ec_gemm(torch.empty((0, 128), dtype=torch.float16, device="cuda:0"), dl.pw)
    assert e.value.status == -1
    buf = torch.zeros(4 * 128 + 8, dtype=torch.float16, device="cuda:0")
    x_mis = buf[1:1 + 4 * 128].view(4, 128)                      # 2 bytes off a 16-byte boundary
    assert x_mis.data_ptr() % 16 != 0
    with pytest.raises(sp.SpearError) as e:
        sp.w4_ec_gemm(x_mis, dl.pw)
    assert e.value.status == -1
    with pytest.raises(sp.SpearError) as e:                      # K not a multiple of 128
        sp.pack_w4(torch.zeros((128, 64), dtype=torch.uint8, device="cuda:0"),
                   torch.ones((128, 1), dtype=torch.float16, device="cuda:0"), 64)
    assert e.value.status == -2


def test_config2_step_in_the_bench_launch_configuration(sp):
    """The 12 calls of BASELINE.json configs[1] issued exactly as bench.py times them: ONE
    spear_w4_ec_gemm_batch (lanes, shallow-ring instance, ~8 units per CTA), captured in a CUDA graph and replayed;
    every call against the oracle, every output element."""
    import torch
    h = _harness()
    shapes = config_shapes(1)
    lis = [make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar") for s in shapes]
    dls = [h.upload_layer(li) for li in lis]
    xs = [h.dev(li.x) for li in lis]
    ys = [torch.zeros((li.M, li.N), dtype=torch.float16, device="cuda:0") for li in lis]
    batch = sp.Batch([(x, dl.pw, dl.A, dl.B, dl.desc(), y) for x, dl, y in zip(xs, dls, ys)])
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        sp.w4_ec_gemm_batch(batch)
        torch.cuda.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=st):
            sp.w4_ec_gemm_batch(batch)
        for y in ys:
            y.zero_()
        for _ in range(5):
            g.replay()
    torch.cuda.synchronize()
    for s, li, y in zip(shapes, lis, ys):
        ref = oracle.forward_layer(li)["y"]
        rms = float(np.sqrt(np.mean(ref ** 2)))
        err = float(np.max(np.abs(y.cpu().numpy().astype(np.float64) - ref)))
        assert err <= Y_TOL * rms, f"config2 {s.name} M={s.M} in the batch: {err:.4g} > {Y_TOL} * {rms:.4g}"


# ---------------------------------------------------------------- INT8 EC factors

@pytest.mark.parametrize("idx", [0, 1, 2, 3, 6, 9, 10, 11])
def test_int8_ec_config2(sp, idx):
    """configs[1] shapes with the EC factors stored INT8 per-channel symmetric: the GPU reads the int8 codes directly
    (fused decode kernel) and must match the oracle's spo_forward_q8 within the usual bars."""
    from workloads import with_int8_ec
    s = config_shapes(1)[idx]
    li = with_int8_ec(make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar"))
    check_layer(li, label=f"int8 EC config2 {s.name} M={s.M}")


def test_int8_ec_config1_and_variants(sp):
    from workloads import with_int8_ec
    s = config_shapes(0)[0]
    li = with_int8_ec(make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar"))
    check_layer(li, variant=1, label="int8 EC config1 fused")
    check_layer(li, variant=2, label="int8 EC config1 split")
    lm = with_int8_ec(make_layer(77, 5, 512, 1024, 128, 24, gate="mlp"))
    check_layer(lm, label="int8 EC, MLP gate (split arm)")
    ln = with_int8_ec(make_layer(78, 16, 384, 640, 128, 128, gate="none", alpha=0.75))
    check_layer(ln, label="int8 EC, r = 128, gate none")


@pytest.mark.parametrize("M", [40, 300])
def test_int8_ec_prefill_path(sp, M):
    """M > 16: the factors are dequantised to an fp16 scratch (one rounding) and take the tcgen05 path."""
    from workloads import with_int8_ec
    li = with_int8_ec(make_layer(79 + M, M, 384, 640, 128, 24, gate="scalar"))
    check_layer(li, label=f"int8 EC M={M}")


# ---------------------------------------------------------------- fused post-EC tail

def check_tail(li, variant=0, rows=None, label=""):
    """Layer + residual add + next-layer RMSNorm against the oracle (spo_forward + spo_tail)."""
    import torch
    import paper_2606_11244_b200 as sp
    h = _harness()
    rng = np.random.default_rng(li.seed + 99)
    res = (rng.standard_normal((li.M, li.N)) * 4.0).astype(np.float16)
    gw = rng.uniform(0.5, 1.5, li.N).astype(np.float16)
    eps = 1e-5
    dl = h.upload_layer(li)
    y, hn = sp.w4_ec_gemm_tail(h.dev(li.x), dl.pw, dl.A, dl.B, dl.desc(variant=variant), h.dev(res), h.dev(gw), eps)
    torch.cuda.synchronize()
    ref = oracle.forward_layer(li)
    s_ref, h_ref = oracle.tail(ref["y"], res, gw, eps)
    for name, got, want in (("residual stream", y, s_ref), ("rmsnorm", hn, h_ref)):
        g64 = got.cpu().numpy().astype(np.float64)
        rms = float(np.sqrt(np.mean(want ** 2)))
        err = float(np.max(np.abs(g64 - want)))
        assert err <= Y_TOL * rms, f"{label} {name}: max err {err:.4g} > {Y_TOL} * rms {rms:.4g}"


@pytest.mark.parametrize("idx", [0, 2, 3, 5, 7, 8, 10, 11])
def test_fused_tail_config2(sp, idx):
    s = config_shapes(1)[idx]
    check_tail(make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar"), label=f"tail config2 {s.name} M={s.M}")


def test_fused_tail_variants_and_back_to_back(sp):
    li = make_layer(300, 7, 1024, 768, 128, 16, gate="scalar")
    for v in (1, 2, 5, 3):          # fused in the decode epilogue (1, 2); layer + row kernel (layer-stream, tcgen05)
        check_tail(li, variant=v, label=f"tail variant {v}")
        check_tail(li, variant=v, label=f"tail variant {v} again")       # the tail state must come back clean
    check_tail(make_layer(301, 3, 256, 256, 128, 0), label="tail r=0")
    check_tail(make_layer(302, 16, 128 * 19, 256, 128, 8, gate="mlp"), label="tail mlp, more panels than CTAs have units")
    check_tail(make_layer(303, 100, 384, 640, 128, 8, gate="scalar"), label="tail M=100 (tcgen05 + row kernel)")


def test_fused_tail_in_place_residual(sp):
    """The residual stream may be updated in place (residual == y)."""
    import torch
    import paper_2606_11244_b200 as sp_
    h = _harness()
    li = make_layer(304, 5, 512, 512, 128, 8, gate="scalar")
    rng = np.random.default_rng(1)
    res = (rng.standard_normal((5, 512)) * 3).astype(np.float16)
    gw = np.ones(512, np.float16)
    dl = h.upload_layer(li)
    stream = h.dev(res)
    y, hn = sp_.w4_ec_gemm_tail(h.dev(li.x), dl.pw, dl.A, dl.B, dl.desc(), stream, h.dev(gw), 1e-5, y=stream)
    torch.cuda.synchronize()
    s_ref, h_ref = oracle.tail(oracle.forward_layer(li)["y"], res, gw, 1e-5)
    assert float(np.max(np.abs(y.cpu().numpy().astype(np.float64) - s_ref))) <= Y_TOL * float(np.sqrt(np.mean(s_ref ** 2)))
    assert float(np.max(np.abs(hn.cpu().numpy().astype(np.float64) - h_ref))) <= Y_TOL * float(np.sqrt(np.mean(h_ref ** 2)))


def test_fused_tail_in_place_is_refused_where_the_tail_is_not_fused(sp):
    """residual == y only works where one thread reads residual[m][n] and writes y[m][n] (the weight-stream epilogue).
    The two-kernel arms store y first and would then add the layer to itself: they must refuse, not return 2 * layer."""
    import torch
    import paper_2606_11244_b200 as sp_
    h = _harness()
    gw = h.dev(np.ones(512, np.float16))
    for M, variant in ((5, sp_.VARIANT_ROWS), (5, sp_.VARIANT_LSTREAM), (40, sp_.VARIANT_AUTO)):
        li = make_layer(305 + M, M, 512, 512, 128, 8, gate="scalar")
        dl = h.upload_layer(li)
        res = np.full((M, 512), 3.0, np.float16)
        stream = h.dev(res)
        with pytest.raises(sp_.SpearError):
            sp_.w4_ec_gemm_tail(h.dev(li.x), dl.pw, dl.A, dl.B, dl.desc(variant=variant), stream, gw, 1e-5, y=stream)
        torch.cuda.synchronize()
        assert np.array_equal(stream.cpu().numpy(), res), "a refused call must not touch the residual stream"
        # ... and the same call out of place is served, and right
        y, hn = sp_.w4_ec_gemm_tail(h.dev(li.x), dl.pw, dl.A, dl.B, dl.desc(variant=variant), stream, gw, 1e-5)
        torch.cuda.synchronize()
        s_ref, h_ref = oracle.tail(oracle.forward_layer(li)["y"], res, np.ones(512, np.float16), 1e-5)
        assert float(np.max(np.abs(y.cpu().numpy().astype(np.float64) - s_ref))) <= Y_TOL * float(np.sqrt(np.mean(s_ref ** 2)))
        assert float(np.max(np.abs(hn.cpu().numpy().astype(np.float64) - h_ref))) <= Y_TOL * float(np.sqrt(np.mean(h_ref ** 2)))


def test_config2_step_stream_ordered_as_bench_headline(sp):
    """The headline leg of bench.py: the 12 calls of BASELINE.json configs[1] one after the other on one stream
    (spear_w4_ec_gemm_ex, AUTO dispatch: row-strip kernel on qkv / o, deep-ring weight-stream kernel on gate_up / down, PDL-chained),
    captured in a CUDA graph and replayed; every call, every output element against the oracle."""
    import torch
    h = _harness()
    shapes = config_shapes(1)
    lis = [make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar") for s in shapes]
    dls = [h.upload_layer(li) for li in lis]
    xs = [h.dev(li.x) for li in lis]
    ys = [torch.zeros((li.M, li.N), dtype=torch.float16, device="cuda:0") for li in lis]
    ds = [dl.desc() for dl in dls]

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
        for _ in range(5):
            g.replay()
    torch.cuda.synchronize()
    for s, li, y in zip(shapes, lis, ys):
        ref = oracle.forward_layer(li)["y"]
        rms = float(np.sqrt(np.mean(ref ** 2)))
        err = float(np.max(np.abs(y.cpu().numpy().astype(np.float64) - ref)))
        assert err <= Y_TOL * rms, f"config2 {s.name} M={s.M} stream-ordered: {err:.4g} > {Y_TOL} * {rms:.4g}"


def test_stream_ordered_step_replay_stress(sp):
    """5000 back-to-back replays of the headline step (row-strip kernel behind its one-cluster EC pre-kernel, cooperative ring
    kernel with the fused EC, all PDL-chained): every replay must finish, the workspace state (z buffers, epoch word, split-K
    and panel counters) must come back clean every time, and the last results must still match the oracle."""
    import torch
    h = _harness()
    shapes = config_shapes(1)
    lis = [make_layer(s.seed, s.M, s.N, s.K, s.group, s.r, gate="scalar") for s in shapes]
    dls = [h.upload_layer(li) for li in lis]
    xs = [h.dev(li.x) for li in lis]
    ys = [torch.zeros((li.M, li.N), dtype=torch.float16, device="cuda:0") for li in lis]
    ds = [dl.desc() for dl in dls]

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
        for _ in range(5000):
            g.replay()
        torch.cuda.synchronize()
        snap = [y.clone() for y in ys]
        for y in ys:
            y.zero_()
        g.replay()
        torch.cuda.synchronize()
    for s, li, y, y0 in zip(shapes, lis, ys, snap):
        ref = oracle.forward_layer(li)["y"]
        rms = float(np.sqrt(np.mean(ref ** 2)))
        for lab, t in (("after 5000 replays", y0), ("replay 5001 into zeroed y", y)):
            err = float(np.max(np.abs(t.cpu().numpy().astype(np.float64) - ref)))
            assert err <= Y_TOL * rms, f"{s.name} M={s.M} {lab}: {err:.4g} > {Y_TOL} * {rms:.4g}"


@pytest.mark.parametrize("shape", [(8, 2048, 8192, 128, 32), (16, 2048, 8192, 128, 0), (1, 6144, 4096, 4096, 64), (16, 4096, 14336, 14336, 64),
                                   (5, 1280, 1792, 128, 16), (8, 384, 7168, 128, 8), (16, 2432, 4608, 256, 24)])
@pytest.mark.parametrize("knob", [("stream_aligned", 0), ("stream_aligned", 1), ("stream_grid", 37), ("stream_grid", 101)])
def test_ring_kernel_partitions(sp, shape, knob):
    """The ring kernel's result must not depend on how the units are cut over CTAs: panel-aligned equal parts (default when a layer has
    fewer panels than SMs), the even stream-K split (stream_aligned = 0), and two odd forced grids whose CTAs straddle panels with
    ragged first / last segments -- with and without the EC (whose B slab follows the segment that starts a panel)."""
    M, N, K, group, r = shape
    li = make_layer(800 + M + r, M, N, K, group, r, gate="scalar")
    sp.tune(knob[0], knob[1])
    try:
        check_layer(li, variant=1 if r else 2, label=f"{knob} {shape}")
    finally:
        sp.tune("stream_aligned", 1)
        sp.tune("stream_grid", 0)
