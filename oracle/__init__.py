"""CPU oracle for the SPEAR W4A16 + gated-EC layer -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
reference legs may import this package.  The product (paper_2606_11244_b200)
never does, and this package never imports the product.

The arithmetic lives in spear_oracle.c (plain C, fp64, written from PAPER.md
Eq. 2-4 :96-:114 and the layout document in DESIGN.md); this file is the
ctypes/numpy marshalling around it and builds the shared object with gcc when
it is missing or stale.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "spear_oracle.c")
_SO = os.path.join(_HERE, "libspear_oracle.so")

GATE_SCALAR, GATE_MLP, GATE_NONE = 0, 1, 2
_GATE = {"scalar": GATE_SCALAR, "mlp": GATE_MLP, "none": GATE_NONE}


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp, no -ffast-math."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _SO)
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.spo_f16_to_f64.restype = ctypes.c_double
        L.spo_f16_to_f64.argtypes = [ctypes.c_uint16]
        L.spo_f64_to_f16.restype = ctypes.c_uint16
        L.spo_f64_to_f16.argtypes = [ctypes.c_double]
        L.spo_num_threads.restype = ctypes.c_int
        L.spo_forward.restype = ctypes.c_int
        L.spo_forward.argtypes = [ctypes.c_void_p] * 4 + [ctypes.c_int, ctypes.c_int, ctypes.c_double] + \
            [ctypes.c_void_p] * 5 + [ctypes.c_double] + [ctypes.c_int] * 4 + [ctypes.c_void_p] * 4
        L.spo_tail.restype = ctypes.c_int
        L.spo_tail.argtypes = [ctypes.c_void_p] * 3 + [ctypes.c_double, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
        L.spo_forward_q8.restype = ctypes.c_int
        L.spo_forward_q8.argtypes = [ctypes.c_void_p] * 6 + [ctypes.c_int, ctypes.c_int, ctypes.c_double] + \
            [ctypes.c_void_p] * 5 + [ctypes.c_double] + [ctypes.c_int] * 4 + [ctypes.c_void_p] * 4
        for name in ("spo_dequant", "spo_dequant16"):
            f = getattr(L, name)
            f.restype = ctypes.c_int
            f.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                          ctypes.c_void_p]
        L.spo_pack_w4.restype = ctypes.c_int
        L.spo_pack_w4.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int,
                                  ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
        L.spo_unpack_w4.restype = ctypes.c_int
        L.spo_unpack_w4.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_void_p]
        L.spo_rtn_quantise.restype = None
        L.spo_rtn_quantise.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                       ctypes.c_void_p, ctypes.c_void_p]
        L.spo_f16_to_f64_array.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t]
        L.spo_f64_to_f16_array.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_size_t]
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().spo_num_threads())


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _bits(a: Optional[np.ndarray]) -> Optional[np.ndarray]:
    """fp16 array -> contiguous uint16 bit patterns (a view, no arithmetic)."""
    if a is None:
        return None
    assert a.dtype == np.float16, a.dtype
    return np.ascontiguousarray(a).view(np.uint16)


def f16_to_f64(a: np.ndarray) -> np.ndarray:
    b = _bits(a)
    out = np.empty(b.shape, np.float64)
    lib().spo_f16_to_f64_array(_p(b), _p(out), b.size)
    return out


def f64_to_f16(a: np.ndarray) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float64)
    out = np.empty(a.shape, np.uint16)
    lib().spo_f64_to_f16_array(_p(a), _p(out), a.size)
    return out.view(np.float16)


def dequant(codes: np.ndarray, scales: np.ndarray, group: int) -> np.ndarray:
    """O1: What[n][k] = (q - 8) * s[n][k/group], fp64."""
    N, K = codes.shape
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    out = np.empty((N, K), np.float64)
    rc = lib().spo_dequant(_p(codes), _p(_bits(scales)), N, K, group, _p(out))
    if rc:
        raise ValueError("code > 15")
    return out


def dequant16(codes: np.ndarray, scales: np.ndarray, group: int) -> np.ndarray:
    """Q3: RN-even fp16 of O1."""
    N, K = codes.shape
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    out = np.empty((N, K), np.uint16)
    rc = lib().spo_dequant16(_p(codes), _p(_bits(scales)), N, K, group, _p(out))
    if rc:
        raise ValueError("code > 15")
    return out.view(np.float16)


def forward(x, What, A=None, B=None, gate="scalar", alpha=1.0, w_g=None, b_g=0.0,
            W1=None, b1=None, W2=None, b2=None, A_scale=None, B_scale=None):
    """O2..O6 on fp16 inputs (numpy float16 arrays) and an fp64 What from dequant().

    Returns dict(y, ybase, z, gam) in fp64; gam is [M][r] for the MLP gate, [M]
    for the scalar gate, None otherwise.
    """
    M, K = x.shape
    N = What.shape[0]
    assert What.shape == (N, K) and What.dtype == np.float64
    r = 0 if A is None else A.shape[0]
    h = 0 if W1 is None else W1.shape[0]
    What = np.ascontiguousarray(What)
    y = np.empty((M, N), np.float64)
    ybase = np.empty((M, N), np.float64)
    z = np.zeros((M, max(r, 1)), np.float64)
    gam = np.zeros((M, max(r, 1)), np.float64)
    b1c = None if b1 is None else np.ascontiguousarray(b1, dtype=np.float32)
    b2c = None if b2 is None else np.ascontiguousarray(b2, dtype=np.float32)
    if A is not None and A.dtype == np.int8:       # INT8 per-channel symmetric EC factors
        assert B.dtype == np.int8 and A_scale is not None and B_scale is not None
        assert A_scale.shape == (r,) and B_scale.shape == (N,)
        rc = lib().spo_forward_q8(_p(_bits(x)), _p(What), _p(np.ascontiguousarray(A)), _p(_bits(A_scale)),
                                  _p(np.ascontiguousarray(B)), _p(_bits(B_scale)),
                                  _GATE[gate], h, float(alpha),
                                  _p(_bits(W1)), _p(b1c), _p(_bits(W2)), _p(b2c),
                                  _p(_bits(w_g)), float(b_g), M, N, K, r,
                                  _p(y), _p(ybase), _p(z), _p(gam))
    else:
        rc = lib().spo_forward(_p(_bits(x)), _p(What), _p(_bits(A)), _p(_bits(B)),
                               _GATE[gate], h, float(alpha),
                               _p(_bits(W1)), _p(b1c), _p(_bits(W2)), _p(b2c),
                               _p(_bits(w_g)), float(b_g), M, N, K, r,
                               _p(y), _p(ybase), _p(z), _p(gam))
    if rc:
        raise ValueError("spo_forward: bad arguments")
    out = {"y": y, "ybase": ybase, "z": None, "gam": None}
    if r > 0:
        out["z"] = z[:, :r]
        if gate == "mlp":
            out["gam"] = gam[:, :r]
        elif gate == "scalar":
            out["gam"] = gam[:, 0].copy()
    return out


def forward_layer(li, rows=None):
    """Convenience: run the oracle on a workloads.LayerInputs (optionally on a
    subset of token rows -- each y[m][:] depends on x[m][:] only)."""
    What = dequant(li.codes, li.scales, li.group)
    x = li.x if rows is None else np.ascontiguousarray(li.x[rows])
    if li.r == 0:
        return forward(x, What, gate="none")
    return forward(x, What, li.A, li.B, gate=li.gate, alpha=li.alpha, w_g=li.w_g, b_g=li.b_g,
                   W1=li.W1, b1=li.b1, W2=li.W2, b2=li.b2,
                   A_scale=getattr(li, "A_scale", None), B_scale=getattr(li, "B_scale", None))


def tail(y: np.ndarray, residual: np.ndarray, rms_weight: np.ndarray, eps: float):
    """T1 / T2: returns (s = residual + y, h = RMSNorm(s) * weight), fp64."""
    M, N = y.shape
    y = np.ascontiguousarray(y, dtype=np.float64)
    s = np.empty((M, N), np.float64)
    h = np.empty((M, N), np.float64)
    rc = lib().spo_tail(_p(y), _p(_bits(residual)), _p(_bits(rms_weight)), float(eps), M, N, _p(s), _p(h))
    if rc:
        raise ValueError("spo_tail: bad arguments")
    return s, h


def pack_w4(codes: np.ndarray, scales: np.ndarray, group: int):
    """Q1: packed layout from the layout document. Returns (wq uint32[N*K/8], scales_packed f16)."""
    N, K = codes.shape
    codes = np.ascontiguousarray(codes, dtype=np.uint8)
    wq = np.empty(N * K // 8, np.uint32)
    sp = np.empty(N * (K // group), np.uint16)
    rc = lib().spo_pack_w4(_p(codes), _p(_bits(scales)), N, K, group, _p(wq), _p(sp))
    if rc == -1:
        raise ValueError("code > 15")
    if rc:
        raise ValueError("unsupported shape for the packed layout")
    return wq, sp.view(np.float16)


def unpack_w4(wq: np.ndarray, N: int, K: int) -> np.ndarray:
    wq = np.ascontiguousarray(wq, dtype=np.uint32)
    codes = np.empty((N, K), np.uint8)
    rc = lib().spo_unpack_w4(_p(wq), N, K, _p(codes))
    if rc:
        raise ValueError("unsupported shape for the packed layout")
    return codes


def rtn_quantise(W: np.ndarray, group: int):
    """A5 (test-only): returns (codes u8[N][K], scales f16[N][K/group])."""
    W = np.ascontiguousarray(W, dtype=np.float64)
    N, K = W.shape
    codes = np.empty((N, K), np.uint8)
    scales = np.empty((N, K // group), np.uint16)
    lib().spo_rtn_quantise(_p(W), N, K, group, _p(codes), _p(scales))
    return codes, scales.view(np.float16)
