"""The five BASELINE.json configs as shape lists, plus the algorithmic
byte/flop counts of SURVEY.md 8(d).  Shapes only; no method arithmetic."""
from __future__ import annotations

from dataclasses import dataclass
from typing import List


@dataclass(frozen=True)
class LayerShape:
    name: str
    M: int
    N: int
    K: int
    group: int
    r: int
    gate: str = "scalar"
    seed: int = 0


def _llama1b(M, r, group=128, seed=2):
    return [
        LayerShape("qkv", M, 3072, 2048, group, r, seed=seed),
        LayerShape("o", M, 2048, 2048, group, r, seed=seed + 100),
        LayerShape("gate_up", M, 16384, 2048, group, r, seed=seed + 200),
        LayerShape("down", M, 2048, 8192, group, r, seed=seed + 300),
    ]


def config_shapes(idx: int) -> List[LayerShape]:
    """idx is the 0-based position in BASELINE.json `configs`."""
    if idx == 0:
        return [LayerShape("cfg1", 4, 2048, 2048, 128, 16, seed=0)]
    if idx == 1:
        out = []
        for M in (1, 8, 16):
            out += _llama1b(M, 32, seed=2 + M)
        return out
    if idx == 2:
        out = []
        for M in (1, 16, 256, 2048):
            out += [
                LayerShape("qkv", M, 6144, 4096, 4096, 64, seed=3000 + M),
                LayerShape("gate_up", M, 28672, 4096, 4096, 64, seed=3100 + M),
                LayerShape("down", M, 4096, 14336, 14336, 64, seed=3200 + M),
            ]
        return out
    if idx == 3:
        out = []
        for M in (512, 4096, 16384):
            for r in (0, 16, 64, 128):
                out.append(LayerShape("mlp70b", M, 28672, 8192, 128, r, seed=4000 + M + r))
        return out
    if idx == 4:
        out = []
        for M in (64, 2048):
            out += stack_shapes(M)
        return out
    raise IndexError(idx)


EC_LAYERS = (0, 1, 14, 15)   # reading A11: ECs on o/down of these layers only


def stack_shapes(M: int) -> List[LayerShape]:
    """Config 5: 16 layers x {qkv, o, gate_up, down}, 64 independent calls."""
    out = []
    for layer in range(16):
        for name, N, K in (("qkv", 3072, 2048), ("o", 2048, 2048),
                           ("gate_up", 16384, 2048), ("down", 2048, 8192)):
            r = 32 if (layer in EC_LAYERS and name in ("o", "down")) else 0
            out.append(LayerShape(f"L{layer}.{name}", M, N, K, 128, r,
                                  seed=5000 + 10 * layer + len(out) % 4 + M))
    return out


CONFIGS = [config_shapes(i) for i in range(5)]


def algorithmic_bytes(M, N, K, group, r, gate="scalar", h=0, ec_int8=False) -> int:
    """bytes_W4 + bytes_EC of SURVEY.md 8(d) (what the method must move); ec_int8: INT8 factors + their fp16 row scales."""
    G = K // group
    b = N * K // 2 + 2 * N * G + 2 * M * K + 2 * M * N
    if r > 0:
        b += (r * (K + N) + 2 * (r + N)) if ec_int8 else 2 * r * (K + N)
        if gate == "scalar":
            b += 2 * K + 4
        elif gate == "mlp":
            b += 2 * 2 * r * h + 4 * (h + r)
    return b


def algorithmic_flops(M, N, K, group, r, gate="scalar", h=0) -> int:
    f = 2 * M * N * K
    if r > 0:
        f += 2 * M * r * (K + N)
        if gate == "scalar":
            f += 2 * M * K
        elif gate == "mlp":
            f += 4 * M * r * h
    return f
