"""Device-side plumbing shared by the GPU tests, smoke() and bench.py: uploads a
workloads.LayerInputs (host numpy, canonical layouts) to the GPU, packs the weights through
spear_pack_w4 and calls the layer through the C ABI.  No arithmetic of the method lives here and
nothing from oracle/ is imported.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import Optional

import numpy as np
import torch

from . import (EcDesc, PackedW4, VARIANT_AUTO, make_desc, pack_w4, w4_ec_gemm, w4_ec_gemm_ex)


def dev(a: Optional[np.ndarray], device="cuda:0"):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(device)


@dataclass
class DeviceLayer:
    """One layer's parameters resident in HBM (packed weights + EC factors + gate)."""
    pw: PackedW4
    M: int
    N: int
    K: int
    r: int
    group: int
    gate: str
    alpha: float
    A: Optional[torch.Tensor] = None
    B: Optional[torch.Tensor] = None
    w_g: Optional[torch.Tensor] = None
    b_g: Optional[torch.Tensor] = None
    W1: Optional[torch.Tensor] = None
    b1: Optional[torch.Tensor] = None
    W2: Optional[torch.Tensor] = None
    b2: Optional[torch.Tensor] = None
    A_scale: Optional[torch.Tensor] = None     # INT8 EC factors: A / B are int8, one fp16 scale per row
    B_scale: Optional[torch.Tensor] = None

    def desc(self, gate_out=None, variant=VARIANT_AUTO) -> EcDesc:
        return make_desc(gate=self.gate if self.r > 0 else "none", alpha=self.alpha, w_g=self.w_g, b_g=self.b_g,
                         W1=self.W1, b1=self.b1, W2=self.W2, b2=self.b2, gate_out=gate_out, variant=variant,
                         A_scale=self.A_scale, B_scale=self.B_scale)


def upload_layer(li, device="cuda:0") -> DeviceLayer:
    codes = dev(li.codes, device)
    scales = dev(li.scales, device)
    pw = pack_w4(codes, scales, li.group)
    dl = DeviceLayer(pw=pw, M=li.M, N=li.N, K=li.K, r=li.r, group=li.group, gate=li.gate, alpha=li.alpha)
    if li.r > 0:
        dl.A, dl.B = dev(li.A, device), dev(li.B, device)
        if getattr(li, "A_scale", None) is not None:
            dl.A_scale, dl.B_scale = dev(li.A_scale, device), dev(li.B_scale, device)
        if li.gate == "scalar":
            dl.w_g = dev(li.w_g, device)
            dl.b_g = torch.tensor([li.b_g], dtype=torch.float32, device=device)
        elif li.gate == "mlp":
            dl.W1, dl.W2 = dev(li.W1, device), dev(li.W2, device)
            dl.b1, dl.b2 = dev(li.b1, device), dev(li.b2, device)
    return dl


def run_layer(dl: DeviceLayer, x: torch.Tensor, variant=VARIANT_AUTO, want_gate=False, y=None, use_14arg=False):
    """Returns (y fp16 [M][N], gate fp32 or None)."""
    M = x.shape[0]
    if use_14arg:
        assert dl.r == 0 or (dl.gate == "scalar" and dl.alpha == 1.0)
        y = w4_ec_gemm(x, dl.pw, dl.A, dl.B, dl.w_g, dl.b_g, y=y)
        return y, None
    gate_out = None
    if want_gate and dl.r > 0 and dl.gate != "none":
        shape = (M, dl.r) if dl.gate == "mlp" else (M,)
        gate_out = torch.zeros(shape, dtype=torch.float32, device=x.device)
    y = w4_ec_gemm_ex(x, dl.pw, dl.A, dl.B, dl.desc(gate_out=gate_out, variant=variant), y=y)
    return y, gate_out
