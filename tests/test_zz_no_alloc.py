"""spear_w4_ec_gemm_noalloc: the decode layer with its scratch in a static device array (csrc/noalloc.cu), for callers
that cannot call cudaMalloc.  Collected last on purpose (the suite runs with pytest -x: a failure here hides nothing).

Checked against the existing path (spear_w4_ec_gemm_ex, AUTO) on the same inputs, two calls in a row that share the static
array -- the second with another M, rank and gate, so that stale z / u of the first would show -- within the tolerance of
the other GPU tests (1e-2 * rms(y)); both also against the fp64 oracle.  Also: sizes beyond the stated maxima are refused
with a message that names the limit, and the free device memory does not move across a call."""
import numpy as np
import pytest

import oracle
from workloads import make_layer, with_int8_ec

pytestmark = pytest.mark.gpu

Y_TOL = 1e-2


@pytest.fixture(scope="module")
def sp():
    import paper_2606_11244_b200 as sp
    sp.init()          # for the reference path and the packing; the entry point under test never needs it
    return sp


def _pair(sp, li):
    """(y of the no-alloc entry point, y of the existing path, oracle y) for one layer."""
    import torch
    from paper_2606_11244_b200 import harness as h
    dl = h.upload_layer(li)
    x = h.dev(li.x)
    y_new = torch.zeros((li.M, li.N), dtype=torch.float16, device="cuda:0")
    sp.w4_ec_gemm_noalloc(x, dl.pw, dl.A, dl.B, dl.desc(), y=y_new)
    y_old = sp.w4_ec_gemm_ex(x, dl.pw, dl.A, dl.B, dl.desc())
    torch.cuda.synchronize()
    return y_new.cpu().numpy().astype(np.float64), y_old.cpu().numpy().astype(np.float64), oracle.forward_layer(li)["y"]


def _check(y_new, y_old, ref, label):
    rms = float(np.sqrt(np.mean(ref ** 2)))
    assert np.all(np.isfinite(y_new)), label
    assert float(np.max(np.abs(y_new - y_old))) <= Y_TOL * rms, f"{label}: differs from the existing path"
    assert float(np.max(np.abs(y_new - ref))) <= Y_TOL * rms, f"{label}: differs from the oracle"


def test_two_calls_in_a_row_match_the_existing_path(sp):
    # first call: full-size scratch use (M = 16, r = 128, scalar gate: z column r carries the gate's pre-activation)
    a = make_layer(901, 16, 512, 1024, 128, 128, gate="scalar")
    _check(*_pair(sp, a), "call 1 (M=16 r=128 scalar)")
    # second call right behind it on the same array: fewer tokens, lower rank, the paper's MLP gate, alpha != 1
    b = make_layer(902, 5, 384, 640, 128, 24, gate="mlp", alpha=0.75)
    _check(*_pair(sp, b), "call 2 (M=5 r=24 mlp)")
    # and the cases with no / other scratch use: plain W4, gate none, INT8 factors
    _check(*_pair(sp, make_layer(903, 3, 256, 768, 384, 0)), "call 3 (plain W4)")
    _check(*_pair(sp, with_int8_ec(make_layer(904, 8, 2048, 2048, 128, 32, gate="scalar"))), "call 4 (INT8 EC)")
    _check(*_pair(sp, make_layer(905, 9, 256, 256, 128, 16, gate="none")), "call 5 (gate none)")


def test_same_call_repeated_is_stable_and_allocates_nothing(sp):
    import torch
    from paper_2606_11244_b200 import harness as h
    li = make_layer(906, 8, 2048, 2048, 128, 32, gate="scalar")
    dl = h.upload_layer(li)
    x = h.dev(li.x)
    d = dl.desc()
    y = torch.zeros((8, 2048), dtype=torch.float16, device="cuda:0")
    sp.w4_ec_gemm_noalloc(x, dl.pw, dl.A, dl.B, d, y=y)          # first call: kernels get loaded, the symbol address is taken
    torch.cuda.synchronize()
    first = y.clone()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(50):
        sp.w4_ec_gemm_noalloc(x, dl.pw, dl.A, dl.B, d, y=y)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, f"free device memory moved by {free0 - free1} bytes across 50 calls"
    ref = oracle.forward_layer(li)["y"]
    rms = float(np.sqrt(np.mean(ref ** 2)))
    assert float(np.max(np.abs(y.cpu().numpy().astype(np.float64) - ref))) <= Y_TOL * rms
    # fp32 red.add order may differ between runs: equal within rounding, not necessarily bit for bit
    assert float((y.float() - first.float()).abs().max()) <= Y_TOL * rms


def test_sizes_beyond_the_static_scratch_are_refused(sp):
    import torch
    from paper_2606_11244_b200 import harness as h
    li = make_layer(907, 17, 256, 256, 128, 8, gate="scalar")          # M = 17 > 16
    dl = h.upload_layer(li)
    y = torch.full((17, 256), 7.0, dtype=torch.float16, device="cuda:0")
    with pytest.raises(sp.SpearError) as e:
        sp.w4_ec_gemm_noalloc(h.dev(li.x), dl.pw, dl.A, dl.B, dl.desc(), y=y)
    assert "maximum of 16 tokens" in str(e.value)
    torch.cuda.synchronize()
    assert bool((y == 7.0).all()), "a refused call must not write y"
    # r = 136 > 128 (the existing path refuses it too; here the message names the scratch limit)
    A = torch.zeros((136, 256), dtype=torch.float16, device="cuda:0")
    B = torch.zeros((256, 136), dtype=torch.float16, device="cuda:0")
    x = torch.zeros((4, 256), dtype=torch.float16, device="cuda:0")
    with pytest.raises(sp.SpearError) as e:
        sp.w4_ec_gemm_noalloc(x, dl.pw, A, B, sp.make_desc(gate="none"), y=torch.zeros((4, 256), dtype=torch.float16, device="cuda:0"))
    assert "maximum rank 128" in str(e.value)
