"""Counter-based seeded generators (SURVEY.md 8(d) "Synthetic inputs").

Every element of every tensor is a pure function of (seed, tensor tag, index),
so any slice can be regenerated independently of order or thread count:

    u64(i) = splitmix64(seed*0x9E3779B97F4A7C15 + tag*0xD1B54A32D192ED03 + i)
    U(i)   = ((u64 >> 11) + 0.5) * 2**-53                      in (0, 1)
    N(i)   = sqrt(-2 ln U(2i)) * cos(2 pi U(2i+1))             Box-Muller
    code(i)= u64 >> 60                                         uniform 0..15

Values are drawn in fp64 and rounded once (round-to-nearest-even) to fp16.
The distributions follow BASELINE.json `configs` under readings A9/A10 of
SURVEY.md 8(c): the second argument of N(0, s) is a standard deviation.

No arithmetic of the SPEAR layer lives here (no dequantisation, no GEMM, no
gate): this module is shared by the oracle-side and the CUDA-side callers.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_GOLD = 0x9E3779B97F4A7C15
_TAGMUL = 0xD1B54A32D192ED03

# tensor tags (fixed; part of the recipe)
TAGS = {
    "codes": 1, "scales": 2, "x": 3, "A": 4, "B": 5, "w_g": 6,
    "W1": 7, "W2": 8, "outlier_perm": 9, "b1": 10, "b2": 11, "misc": 12,
}


def splitmix64(x: np.ndarray) -> np.ndarray:
    """Vectorised splitmix64 finaliser on uint64 (wrap-around arithmetic)."""
    x = np.asarray(x, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = x + np.uint64(_GOLD)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def _base(seed: int, tag: int) -> np.uint64:
    return np.uint64((seed * _GOLD + tag * _TAGMUL) & 0xFFFFFFFFFFFFFFFF)


def _u64(seed: int, tag: int, start: int, count: int) -> np.ndarray:
    idx = np.arange(start, start + count, dtype=np.uint64)
    with np.errstate(over="ignore"):
        return splitmix64(idx + _base(seed, tag))


_CHUNK = 1 << 24


def uniform_f64(seed: int, tag: int, count: int, start: int = 0) -> np.ndarray:
    out = np.empty(count, dtype=np.float64)
    for o in range(0, count, _CHUNK):
        n = min(_CHUNK, count - o)
        u = _u64(seed, tag, start + o, n)
        out[o:o + n] = ((u >> np.uint64(11)).astype(np.float64) + 0.5) * (2.0 ** -53)
    return out


def normal_f64(seed: int, tag: int, count: int) -> np.ndarray:
    """Standard normals; element i uses counters 2i and 2i+1."""
    out = np.empty(count, dtype=np.float64)
    for o in range(0, count, _CHUNK // 2):
        n = min(_CHUNK // 2, count - o)
        u = uniform_f64(seed, tag, 2 * n, start=2 * o)
        out[o:o + n] = np.sqrt(-2.0 * np.log(u[0::2])) * np.cos(2.0 * np.pi * u[1::2])
    return out


def codes_uniform(seed: int, tag: int, count: int) -> np.ndarray:
    out = np.empty(count, dtype=np.uint8)
    for o in range(0, count, _CHUNK):
        n = min(_CHUNK, count - o)
        out[o:o + n] = (_u64(seed, tag, o, n) >> np.uint64(60)).astype(np.uint8)
    return out


@dataclass
class LayerInputs:
    """Canonical (unpacked) inputs of one layer call; every array is host numpy.

    Layouts (row-major, contiguous): x[M][K] f16, codes[N][K] u8,
    scales[N][K/group] f16, A[r][K] f16, B[N][r] f16, w_g[K] f16, b_g f32 scalar,
    W1[h][r] f16, b1[h] f32, W2[r][h] f16, b2[r] f32.
    """
    M: int
    N: int
    K: int
    r: int
    group: int
    seed: int
    gate: str                      # "scalar" | "mlp" | "none"
    h: int
    alpha: float
    codes: np.ndarray
    scales: np.ndarray
    x: np.ndarray
    A: Optional[np.ndarray] = None
    B: Optional[np.ndarray] = None
    w_g: Optional[np.ndarray] = None
    b_g: float = 0.0
    W1: Optional[np.ndarray] = None
    b1: Optional[np.ndarray] = None
    W2: Optional[np.ndarray] = None
    b2: Optional[np.ndarray] = None
    A_scale: Optional[np.ndarray] = None      # INT8 EC factors: A is int8 [r][K] with one fp16 scale per row
    B_scale: Optional[np.ndarray] = None      # B is int8 [N][r] with one fp16 scale per row (output channel)
    outlier_channels: np.ndarray = field(default_factory=lambda: np.zeros(0, np.int64))


def _f16(a: np.ndarray) -> np.ndarray:
    return np.ascontiguousarray(a.astype(np.float16))


def make_x(seed: int, M: int, K: int):
    """x ~ N(0,1) with round(0.01*K) outlier channels scaled x20 (reading A10)."""
    n_out = int(round(0.01 * K))
    perm_key = uniform_f64(seed, TAGS["outlier_perm"], K)
    chans = np.argsort(perm_key, kind="stable")[:n_out].astype(np.int64)
    x = normal_f64(seed, TAGS["x"], M * K).reshape(M, K)
    x[:, chans] *= 20.0
    return _f16(x), chans


def make_layer(seed: int, M: int, N: int, K: int, group: int, r: int,
               gate: str = "scalar", h: Optional[int] = None,
               alpha: float = 1.0) -> LayerInputs:
    """One layer call's inputs with the distributions BASELINE.json states."""
    assert K % group == 0 and gate in ("scalar", "mlp", "none")
    G = K // group
    codes = codes_uniform(seed, TAGS["codes"], N * K).reshape(N, K)
    scales = _f16(np.abs(0.02 * normal_f64(seed, TAGS["scales"], N * G)) + 1e-3).reshape(N, G)
    x, chans = make_x(seed, M, K)
    li = LayerInputs(M=M, N=N, K=K, r=r, group=group, seed=seed, gate=gate,
                     h=0, alpha=alpha, codes=codes, scales=scales, x=x,
                     outlier_channels=chans)
    if r > 0:
        li.A = _f16(normal_f64(seed, TAGS["A"], r * K) / np.sqrt(K)).reshape(r, K)
        li.B = _f16(normal_f64(seed, TAGS["B"], N * r) / np.sqrt(r)).reshape(N, r)
        if gate == "scalar":
            li.w_g = _f16(normal_f64(seed, TAGS["w_g"], K) / np.sqrt(K))
            li.b_g = 0.0
        elif gate == "mlp":
            hh = 4 * r if h is None else h
            li.h = hh
            li.W1 = _f16(normal_f64(seed, TAGS["W1"], hh * r) / np.sqrt(r)).reshape(hh, r)
            li.W2 = _f16(normal_f64(seed, TAGS["W2"], r * hh) / np.sqrt(hh)).reshape(r, hh)
            li.b1 = np.zeros(hh, np.float32)
            li.b2 = np.zeros(r, np.float32)
    return li


def with_int8_ec(li: LayerInputs) -> LayerInputs:
    """The same layer with its EC factors stored the way the paper stores them after calibration: "INT8 per-channel
    symmetric".  Input preparation only: per row, scale = fp16(max|v| / 127), code = clamp(round-half-even
    (v / scale), -127, 127).  The quantised factors (code * scale) are the layer's EC from here on -- the oracle and the
    GPU both consume the int8 codes and the fp16 scales."""
    import copy
    assert li.r > 0 and li.A.dtype == np.float16
    out = copy.copy(li)

    def q(mat):
        m = mat.astype(np.float64)
        s = np.max(np.abs(m), axis=1) / 127.0
        s = np.where(s > 0, s, 1.0).astype(np.float16)
        codes = np.clip(np.rint(m / s.astype(np.float64)[:, None]), -127, 127).astype(np.int8)
        return np.ascontiguousarray(codes), np.ascontiguousarray(s)

    out.A, out.A_scale = q(li.A)
    out.B, out.B_scale = q(li.B)
    return out
