"""paper_2606_11244_b200 -- thin Python binding of libspear.so (include/spear.h).

Argument marshalling only: every step of the SPEAR W4A16 + gated-EC layer (PAPER.md:107-110,
Eq. 3) runs in the CUDA kernels behind the C ABI.  torch is used for device memory and streams.
There is no CPU path: importing works without a GPU (so the symbol table can be checked), but
every compute call needs the library and a CUDA device and raises otherwise.
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass
from typing import Optional

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libspear.so")

GATE_SCALAR_SIGMOID, GATE_MLP, GATE_NONE = 0, 1, 2
GATE_KINDS = {"scalar": GATE_SCALAR_SIGMOID, "mlp": GATE_MLP, "none": GATE_NONE}
VARIANT_AUTO, VARIANT_STREAM_FUSED, VARIANT_STREAM_SPLIT, VARIANT_TC_FUSED, VARIANT_TC_SPLIT, VARIANT_LSTREAM, VARIANT_ROWS = range(7)
VARIANT_COUNT = 7
VARIANT_NAMES = ["auto", "stream_fused", "stream_split", "tc_fused", "tc_split", "lstream", "rows"]

EXPORTS = [
    "spear_pack_w4_sizes", "spear_pack_w4", "spear_unpack_w4", "spear_dequant_w4",
    "spear_w4_ec_gemm", "spear_w4_ec_gemm_ex", "spear_w4_ec_gemm_hostio", "spear_w4_ec_gemm_tail", "spear_w4_ec_gemm_noalloc", "spear_w4_ec_gemm_batch", "spear_w4_ec_gemm_batch_hostio",
    "spear_workspace_bytes", "spear_init", "spear_memory_bytes", "spear_plan", "spear_plan_save", "spear_plan_load",
    "spear_plan_query", "spear_plan_batch", "spear_lut_create", "spear_lut_destroy", "spear_lut_iteration_us",
    "spear_slo_chunk", "spear_lut_measure", "spear_tune", "spear_last_error", "spear_launch_count",
]


class SpearError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"libspear status {status}: {msg}")
        self.status = status


class EcDesc(ctypes.Structure):
    """struct spear_ec_desc of include/spear.h."""
    _fields_ = [
        ("gate_kind", ctypes.c_int), ("gate_hidden", ctypes.c_int), ("alpha", ctypes.c_float),
        ("W1", ctypes.c_void_p), ("b1", ctypes.c_void_p), ("W2", ctypes.c_void_p), ("b2", ctypes.c_void_p),
        ("w_g", ctypes.c_void_p), ("b_g", ctypes.c_void_p), ("gate_out", ctypes.c_void_p),
        ("workspace", ctypes.c_void_p), ("workspace_bytes", ctypes.c_size_t), ("force_variant", ctypes.c_int),
        ("ec_dtype", ctypes.c_int), ("A_scale", ctypes.c_void_p), ("B_scale", ctypes.c_void_p),
    ]


class TailDesc(ctypes.Structure):
    """struct spear_tail_desc of include/spear.h."""
    _fields_ = [("residual", ctypes.c_void_p), ("rms_weight", ctypes.c_void_p), ("eps", ctypes.c_float), ("h_out", ctypes.c_void_p)]


class Call(ctypes.Structure):
    """struct spear_call of include/spear.h (one entry of spear_w4_ec_gemm_batch)."""
    _fields_ = [
        ("x", ctypes.c_void_p), ("Wq", ctypes.c_void_p), ("scales", ctypes.c_void_p), ("A", ctypes.c_void_p),
        ("B", ctypes.c_void_p), ("ec", ctypes.POINTER(EcDesc)), ("y", ctypes.c_void_p),
        ("M", ctypes.c_int), ("N", ctypes.c_int), ("K", ctypes.c_int), ("r", ctypes.c_int), ("group", ctypes.c_int),
    ]


class HostIO(ctypes.Structure):
    """struct spear_host_io of include/spear.h."""
    _fields_ = [("x_host", ctypes.c_void_p), ("y_host", ctypes.c_void_p)]


_lib = None


def lib():
    """Loads libspear.so; raises (loudly) if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_11244_b200.build` "
                              "(there is no fallback path)")
        L = ctypes.CDLL(LIB_PATH)
        vp, ci = ctypes.c_void_p, ctypes.c_int
        L.spear_pack_w4_sizes.argtypes = [ci, ci, ci, ctypes.POINTER(ctypes.c_size_t), ctypes.POINTER(ctypes.c_size_t)]
        L.spear_pack_w4.argtypes = [vp, vp, vp, vp, ci, ci, ci, vp]
        L.spear_unpack_w4.argtypes = [vp, vp, ci, ci, ci, vp]
        L.spear_dequant_w4.argtypes = [vp, vp, vp, ci, ci, ci, vp]
        L.spear_w4_ec_gemm.argtypes = [vp] * 8 + [ci] * 5 + [vp]
        L.spear_w4_ec_gemm_ex.argtypes = [vp] * 5 + [ctypes.POINTER(EcDesc), vp] + [ci] * 5 + [vp]
        L.spear_w4_ec_gemm_noalloc.argtypes = [vp] * 5 + [ctypes.POINTER(EcDesc), vp] + [ci] * 5 + [vp]
        L.spear_w4_ec_gemm_tail.argtypes = [vp] * 5 + [ctypes.POINTER(EcDesc), ctypes.POINTER(TailDesc), vp] + [ci] * 5 + [vp]
        L.spear_w4_ec_gemm_batch.argtypes = [ctypes.POINTER(Call), ci, vp]
        L.spear_w4_ec_gemm_batch_hostio.argtypes = [ctypes.POINTER(Call), ctypes.POINTER(HostIO), ci, vp]
        L.spear_w4_ec_gemm_hostio.argtypes = [vp] * 8 + [ctypes.POINTER(EcDesc)] + [ci] * 5 + [vp]
        L.spear_workspace_bytes.argtypes = [ci] * 5 + [ctypes.POINTER(ctypes.c_size_t)]
        L.spear_init.argtypes = []
        L.spear_memory_bytes.argtypes = [ctypes.POINTER(ctypes.c_size_t)]
        L.spear_plan.argtypes = [ci] * 7 + [ctypes.POINTER(ci), ctypes.POINTER(ctypes.c_float), vp]
        L.spear_plan_save.argtypes = [ctypes.c_char_p]
        L.spear_plan_load.argtypes = [ctypes.c_char_p]
        L.spear_plan_query.argtypes = [ci] * 6 + [ctypes.POINTER(ci)]
        L.spear_plan_batch.argtypes = [ctypes.POINTER(Call), ci, ctypes.POINTER(ci), ctypes.POINTER(ctypes.c_float), vp]
        fp = ctypes.POINTER(ctypes.c_float)
        L.spear_lut_create.argtypes = [ctypes.POINTER(ci), ci, ci, fp, fp, fp, ctypes.POINTER(vp)]
        L.spear_lut_destroy.argtypes = [vp]
        L.spear_lut_destroy.restype = None
        L.spear_lut_iteration_us.argtypes = [vp, ctypes.POINTER(ci), ctypes.c_char_p, ci, ci, ci, ctypes.POINTER(ctypes.c_double)]
        L.spear_slo_chunk.argtypes = [vp, ctypes.POINTER(ci), ctypes.c_char_p, ci, ci, ci, ci, ci, ctypes.c_double, ctypes.POINTER(ci)]
        L.spear_lut_measure.argtypes = [ctypes.POINTER(ci), ci, ci, ci, ci, ci, ci, ci, fp, fp, vp]
        L.spear_tune.argtypes = [ctypes.c_char_p, ci]
        L.spear_last_error.restype = ctypes.c_char_p
        L.spear_launch_count.restype = ctypes.c_ulonglong
        for name in EXPORTS:
            if name not in ("spear_last_error", "spear_launch_count", "spear_lut_destroy"):
                getattr(L, name).restype = ci
        _lib = L
    return _lib


def _check(rc: int):
    if rc != 0:
        raise SpearError(rc, lib().spear_last_error().decode())


def _ptr(t) -> Optional[int]:
    return None if t is None else t.data_ptr()


def _stream(stream) -> Optional[int]:
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return s.cuda_stream or None


def init():
    _check(lib().spear_init())


def launch_count() -> int:
    return int(lib().spear_launch_count())


def tune(key: str, value: int):
    _check(lib().spear_tune(key.encode(), int(value)))


def pack_w4_sizes(N: int, K: int, group: int):
    a, b = ctypes.c_size_t(), ctypes.c_size_t()
    _check(lib().spear_pack_w4_sizes(N, K, group, ctypes.byref(a), ctypes.byref(b)))
    return a.value, b.value


@dataclass
class PackedW4:
    """Opaque packed weights of one layer (SPW4 layout) on the device."""
    wq: "torch.Tensor"        # uint8 [N*K/2]
    scales: "torch.Tensor"    # float16 [N*K/group] (packed order)
    N: int
    K: int
    group: int


def pack_w4(codes, scales, group: int, stream=None) -> PackedW4:
    """spear_pack_w4: codes uint8 [N][K] in 0..15, scales float16 [N][K/group] (device tensors)."""
    import torch
    N, K = codes.shape
    assert codes.dtype == torch.uint8 and codes.is_cuda and codes.is_contiguous()
    assert scales.dtype == torch.float16 and scales.is_cuda and scales.is_contiguous()
    wb, sb = pack_w4_sizes(N, K, group)
    wq = torch.empty(wb, dtype=torch.uint8, device=codes.device)
    sp = torch.empty(sb // 2, dtype=torch.float16, device=codes.device)
    _check(lib().spear_pack_w4(_ptr(codes), _ptr(scales), _ptr(wq), _ptr(sp), N, K, group, _stream(stream)))
    return PackedW4(wq, sp, N, K, group)


def unpack_w4(pw: PackedW4, stream=None):
    import torch
    out = torch.empty((pw.N, pw.K), dtype=torch.uint8, device=pw.wq.device)
    _check(lib().spear_unpack_w4(_ptr(pw.wq), _ptr(out), pw.N, pw.K, pw.group, _stream(stream)))
    return out


def dequant_w4(pw: PackedW4, stream=None):
    import torch
    out = torch.empty((pw.N, pw.K), dtype=torch.float16, device=pw.wq.device)
    _check(lib().spear_dequant_w4(_ptr(pw.wq), _ptr(pw.scales), _ptr(out), pw.N, pw.K, pw.group, _stream(stream)))
    return out


def w4_ec_gemm(x, pw: PackedW4, A=None, B=None, gate_w=None, gate_b=None, y=None, stream=None):
    """spear_w4_ec_gemm (the 14-argument call of BASELINE.json): scalar sigmoid gate, alpha = 1."""
    import torch
    M, K = x.shape
    assert K == pw.K and x.dtype == torch.float16 and x.is_contiguous()
    r = 0 if A is None else A.shape[0]
    if y is None:
        y = torch.empty((M, pw.N), dtype=torch.float16, device=x.device)
    _check(lib().spear_w4_ec_gemm(_ptr(x), _ptr(pw.wq), _ptr(pw.scales), _ptr(A), _ptr(B), _ptr(gate_w),
                                  _ptr(gate_b), _ptr(y), M, pw.N, K, r, pw.group, _stream(stream)))
    return y


def make_desc(gate="scalar", alpha=1.0, w_g=None, b_g=None, W1=None, b1=None, W2=None, b2=None,
              gate_out=None, workspace=None, variant=VARIANT_AUTO, A_scale=None, B_scale=None) -> EcDesc:
    d = EcDesc()
    d.gate_kind = GATE_KINDS[gate] if isinstance(gate, str) else int(gate)
    d.gate_hidden = 0 if W1 is None else int(W1.shape[0])
    d.alpha = float(alpha)
    d.W1, d.b1, d.W2, d.b2 = _ptr(W1), _ptr(b1), _ptr(W2), _ptr(b2)
    d.w_g, d.b_g, d.gate_out = _ptr(w_g), _ptr(b_g), _ptr(gate_out)
    d.workspace = _ptr(workspace)
    d.workspace_bytes = 0 if workspace is None else workspace.numel() * workspace.element_size()
    d.force_variant = int(variant)
    d.ec_dtype = 0 if A_scale is None else 1          # SPEAR_EC_INT8: A / B are int8 with one fp16 scale per row
    d.A_scale, d.B_scale = _ptr(A_scale), _ptr(B_scale)
    return d


def w4_ec_gemm_ex(x, pw: PackedW4, A=None, B=None, desc: Optional[EcDesc] = None, y=None, stream=None):
    """spear_w4_ec_gemm_ex: the paper's MLP gate, alpha, gate_out, forced variants."""
    import torch
    M, K = x.shape
    assert K == pw.K and x.dtype == torch.float16 and x.is_contiguous()
    r = 0 if A is None else A.shape[0]
    if desc is None:
        desc = make_desc(gate="none")
    if y is None:
        y = torch.empty((M, pw.N), dtype=torch.float16, device=x.device)
    _check(lib().spear_w4_ec_gemm_ex(_ptr(x), _ptr(pw.wq), _ptr(pw.scales), _ptr(A), _ptr(B),
                                     ctypes.byref(desc), _ptr(y), M, pw.N, K, r, pw.group, _stream(stream)))
    return y


def w4_ec_gemm_noalloc(x, pw: PackedW4, A=None, B=None, desc: Optional[EcDesc] = None, y=None, stream=None):
    """spear_w4_ec_gemm_noalloc: the decode layer (M <= 16, r <= 128) with its scratch in a static device array: the call
    allocates nothing.  y must be passed by a caller that may not allocate; it is created here only when omitted."""
    import torch
    M, K = x.shape
    assert K == pw.K and x.dtype == torch.float16 and x.is_contiguous()
    r = 0 if A is None else A.shape[0]
    if desc is None:
        desc = make_desc(gate="none")
    if y is None:
        y = torch.empty((M, pw.N), dtype=torch.float16, device=x.device)
    _check(lib().spear_w4_ec_gemm_noalloc(_ptr(x), _ptr(pw.wq), _ptr(pw.scales), _ptr(A), _ptr(B),
                                          ctypes.byref(desc), _ptr(y), M, pw.N, K, r, pw.group, _stream(stream)))
    return y


def w4_ec_gemm_tail(x, pw: PackedW4, A, B, desc: Optional[EcDesc], residual, rms_weight, eps, y=None, h_out=None, stream=None):
    """spear_w4_ec_gemm_tail: the layer + residual add + next-layer RMSNorm; returns (y, h_out)."""
    import torch
    M, K = x.shape
    r = 0 if A is None else A.shape[0]
    if desc is None:
        desc = make_desc(gate="none")
    if y is None:
        y = torch.empty((M, pw.N), dtype=torch.float16, device=x.device)
    if h_out is None:
        h_out = torch.empty((M, pw.N), dtype=torch.float16, device=x.device)
    t = TailDesc()
    t.residual, t.rms_weight, t.eps, t.h_out = _ptr(residual), _ptr(rms_weight), float(eps), _ptr(h_out)
    _check(lib().spear_w4_ec_gemm_tail(_ptr(x), _ptr(pw.wq), _ptr(pw.scales), _ptr(A), _ptr(B), ctypes.byref(desc), ctypes.byref(t),
                                       _ptr(y), M, pw.N, K, r, pw.group, _stream(stream)))
    return y, h_out


def w4_ec_gemm_hostio(x_host, y_host, x_dev, y_dev, pw: PackedW4, A=None, B=None,
                      desc: Optional[EcDesc] = None, stream=None):
    """spear_w4_ec_gemm_hostio: x from (pinned) host memory, y back to host, on `stream`."""
    M, K = x_host.shape
    r = 0 if A is None else A.shape[0]
    if desc is None:
        desc = make_desc(gate="none")
    _check(lib().spear_w4_ec_gemm_hostio(_ptr(x_host), _ptr(y_host), _ptr(x_dev), _ptr(y_dev), _ptr(pw.wq),
                                         _ptr(pw.scales), _ptr(A), _ptr(B), ctypes.byref(desc),
                                         M, pw.N, K, r, pw.group, _stream(stream)))


class Batch:
    """A prepared array of spear_call entries (keeps the descriptors and tensors it points to alive)."""

    def __init__(self, entries):
        """entries: iterable of (x, pw, A, B, desc, y) with device tensors; desc may be None when A is None."""
        entries = list(entries)
        self.keep = entries
        self.n = len(entries)
        self.calls = (Call * self.n)()
        for c, (x, pw, A, B, desc, y) in zip(self.calls, entries):
            M, K = x.shape
            assert K == pw.K and y.shape == (M, pw.N)
            c.x, c.Wq, c.scales, c.A, c.B, c.y = _ptr(x), _ptr(pw.wq), _ptr(pw.scales), _ptr(A), _ptr(B), _ptr(y)
            c.ec = ctypes.pointer(desc) if desc is not None else None
            c.M, c.N, c.K, c.r, c.group = M, pw.N, K, (0 if A is None else A.shape[0]), pw.group


def w4_ec_gemm_batch_hostio(batch: Batch, x_hosts, y_hosts, stream=None):
    """spear_w4_ec_gemm_batch_hostio: per call, x from (pinned) host memory and y back to host, on the lanes."""
    assert len(x_hosts) == batch.n and len(y_hosts) == batch.n
    io = (HostIO * batch.n)()
    for e, xh, yh in zip(io, x_hosts, y_hosts):
        e.x_host, e.y_host = _ptr(xh), _ptr(yh)
    _check(lib().spear_w4_ec_gemm_batch_hostio(batch.calls, io, batch.n, _stream(stream)))


def w4_ec_gemm_batch(batch: Batch, stream=None):
    """spear_w4_ec_gemm_batch: independent layer calls, run concurrently on the library's lanes."""
    _check(lib().spear_w4_ec_gemm_batch(batch.calls, batch.n, _stream(stream)))


def workspace_bytes(M, N, K, r, group) -> int:
    b = ctypes.c_size_t()
    _check(lib().spear_workspace_bytes(M, N, K, r, group, ctypes.byref(b)))
    return b.value


def plan(M, N, K, r, group, gate="scalar", gate_hidden=0, stream=None):
    """spear_plan: measures the valid variants, records and returns (chosen, [us per variant])."""
    chosen = ctypes.c_int()
    times = (ctypes.c_float * VARIANT_COUNT)()
    _check(lib().spear_plan(M, N, K, r, group, GATE_KINDS[gate], gate_hidden, ctypes.byref(chosen), times,
                            _stream(stream)))
    return chosen.value, [float(t) for t in times]


def plan_batch(batch, stream=None):
    """spear_plan_batch: times lanes / sequential kernels vs ONE layer-stream launch for this batch; returns (chosen, [us, us])."""
    chosen = ctypes.c_int(-1)
    times = (ctypes.c_float * 2)()
    _check(lib().spear_plan_batch(batch.calls, batch.n, ctypes.byref(chosen), times, _stream(stream)))
    return chosen.value, [float(t) for t in times]


def plan_query(M, N, K, r, group, gate="scalar") -> int:
    v = ctypes.c_int()
    _check(lib().spear_plan_query(M, N, K, r, group, GATE_KINDS[gate], ctypes.byref(v)))
    return v.value


def plan_save(path: str):
    _check(lib().spear_plan_save(path.encode()))


def plan_load(path: str):
    _check(lib().spear_plan_load(path.encode()))


# ---- PAPER.md 4.3: latency tables and SLO-constrained chunk selection (host only; marshalling only) -------------
class Lut:
    """spear_lut: l_W4 / l_EC tables per layer type on a sparse M grid (+ optional attention table), microseconds."""

    def __init__(self, M_grid, lat_w4_us, lat_ec_us, lat_attn_us=None):
        n = len(M_grid)
        n_types = len(lat_w4_us)
        assert len(lat_ec_us) == n_types and all(len(r) == n for r in list(lat_w4_us) + list(lat_ec_us))
        grid = (ctypes.c_int * n)(*[int(v) for v in M_grid])
        flat = lambda rows: (ctypes.c_float * (n_types * n))(*[float(v) for r in rows for v in r])
        attn = None if lat_attn_us is None else (ctypes.c_float * n)(*[float(v) for v in lat_attn_us])
        self._h = ctypes.c_void_p()
        _check(lib().spear_lut_create(grid, n, n_types, flat(lat_w4_us), flat(lat_ec_us), attn, ctypes.byref(self._h)))

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.spear_lut_destroy(self._h)
            self._h = None

    @staticmethod
    def _modules(module_type, selected):
        n = len(module_type)
        types = (ctypes.c_int * n)(*[int(t) for t in module_type])
        sel = None if selected is None else bytes(bytearray(1 if s else 0 for s in selected))
        return types, sel, n

    def iteration_us(self, module_type, selected, M, n_attn_layers=0) -> float:
        types, sel, n = self._modules(module_type, selected)
        out = ctypes.c_double()
        _check(lib().spear_lut_iteration_us(self._h, types, sel, n, n_attn_layers, int(M), ctypes.byref(out)))
        return out.value

    def slo_chunk(self, module_type, selected, d, c_min, c_max, t_slo_us, n_attn_layers=0) -> int:
        types, sel, n = self._modules(module_type, selected)
        c = ctypes.c_int()
        _check(lib().spear_slo_chunk(self._h, types, sel, n, n_attn_layers, int(d), int(c_min), int(c_max),
                                     float(t_slo_us), ctypes.byref(c)))
        return c.value


def lut_measure(M_grid, N, K, group, r, gate="scalar", gate_hidden=0, stream=None):
    """spear_lut_measure: (l_W4 row, l_EC row) of one layer type, measured on the device with spear_plan."""
    n = len(M_grid)
    grid = (ctypes.c_int * n)(*[int(v) for v in M_grid])
    w4, ec = (ctypes.c_float * n)(), (ctypes.c_float * n)()
    _check(lib().spear_lut_measure(grid, n, N, K, group, r, GATE_KINDS[gate], gate_hidden, w4, ec, _stream(stream)))
    return [float(v) for v in w4], [float(v) for v in ec]
