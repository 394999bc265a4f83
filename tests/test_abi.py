"""CPU-side checks of the boundary: libspear.so builds, loads and exports every symbol that
include/spear.h declares; argument errors are reported without a GPU.  No compute calls here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def spear():
    from paper_2606_11244_b200 import build as b
    b.build()
    import paper_2606_11244_b200 as sp
    sp.lib()
    return sp


def _declared():
    src = open(os.path.join(ROOT, "include", "spear.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(spear_[a-z0-9_]+)\s*\(", src)))


def test_header_symbols_all_exported(spear):
    names = _declared()
    assert "spear_w4_ec_gemm" in names and "spear_pack_w4" in names and "spear_plan" in names
    L = ctypes.CDLL(spear.LIB_PATH)
    for n in names:
        assert hasattr(L, n), f"{n} declared in spear.h but not exported"
    assert sorted(spear.EXPORTS) == names


def test_ec_desc_layout_matches_header(spear):
    # 2 ints + float + pad, 7 pointers, void* + size_t, 2 ints (force_variant, ec_dtype), 2 pointers (INT8 EC scales)
    assert ctypes.sizeof(spear.EcDesc) == 16 + 7 * 8 + 16 + 8 + 16
    assert spear.EcDesc.W1.offset == 16 and spear.EcDesc.force_variant.offset == 88
    assert spear.EcDesc.ec_dtype.offset == 92 and spear.EcDesc.A_scale.offset == 96 and spear.EcDesc.B_scale.offset == 104
    assert ctypes.sizeof(spear.TailDesc) == 32 and spear.TailDesc.h_out.offset == 24


def test_sizes_and_shape_errors_need_no_gpu(spear):
    wb, sb = spear.pack_w4_sizes(2048, 2048, 128)
    assert wb == 2048 * 2048 // 2 and sb == 2048 * 16 * 2
    wb, sb = spear.pack_w4_sizes(4096, 14336, 14336)
    assert wb == 4096 * 14336 // 2 and sb == 4096 * 2
    with pytest.raises(spear.SpearError) as e:
        spear.pack_w4_sizes(100, 2048, 128)
    assert e.value.status == -2
    with pytest.raises(spear.SpearError) as e:
        spear.pack_w4_sizes(128, 2048, 96)
    assert e.value.status == -2
    with pytest.raises(spear.SpearError) as e:
        spear.pack_w4_sizes(0, 2048, 128)
    assert e.value.status == -1


def test_no_cpu_fallback(spear):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(spear.SpearError) as e:
        spear.init()
    assert e.value.status == -3   # SPEAR_ECUDA: the library refuses to run without a device


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_11244_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(import oracle|from oracle)\b", txt, flags=re.M), f
                assert "spear_oracle" not in txt and "libspear_oracle" not in txt, f
    osrc = open(os.path.join(ROOT, "oracle", "spear_oracle.c")).read() + open(os.path.join(ROOT, "oracle", "__init__.py")).read()
    assert "paper_2606_11244_b200" not in osrc.replace("(paper_2606_11244_b200)", "")


def test_plan_table_file_roundtrip_and_heuristics_without_gpu(tmp_path):
    """Host logic of S9 that needs no device: the plan file format, and the heuristic AUTO falls back on."""
    import ctypes
    L = ctypes.CDLL(os.path.join(ROOT, "paper_2606_11244_b200", "libspear.so"))
    L.spear_plan_query.argtypes = [ctypes.c_int] * 6 + [ctypes.POINTER(ctypes.c_int)]
    L.spear_plan_load.argtypes = [ctypes.c_char_p]
    L.spear_plan_save.argtypes = [ctypes.c_char_p]
    v = ctypes.c_int()

    def query(M, N, K, r, group, gate):
        assert L.spear_plan_query(M, N, K, r, group, gate, ctypes.byref(v)) == 0
        return v.value
    # heuristics (api.cu heuristic_variant; variants: 1 stream fused, 2 stream split, 3 tcgen05, 6 row-strip).
    # Decode, M <= 16: the row-strip kernel on latency-bound layers -- up to 4 MiB of int4 whatever M, the EC or the gate ...
    assert query(4, 2048, 2048, 16, 128, 0) == 6
    assert query(4, 2048, 2048, 16, 128, 1) == 6          # MLP gate: EC pre-kernel + row-strip kernel
    assert query(4, 2048, 2048, 0, 128, 0) == 6
    assert query(16, 3072, 2048, 32, 128, 0) == 6         # 3 MiB, M = 16
    # ... and nothing above 4 MiB (down 2048 x 8192 = 8 MiB), whatever M or the EC
    assert query(8, 2048, 8192, 0, 128, 0) == 2
    assert query(16, 2048, 8192, 0, 128, 0) == 2
    assert query(8, 2048, 8192, 32, 128, 0) == 1
    assert query(8, 4096, 2048, 0, 128, 0) == 6           # exactly 4 MiB
    assert query(8, 4224, 2048, 0, 128, 0) == 2           # just above
    # the ring kernel for everything larger: fused unless the MLP gate (then, and for r = 0, the split arm)
    assert query(8, 16384, 2048, 32, 128, 0) == 1
    assert query(8, 16384, 2048, 32, 128, 1) == 2
    assert query(8, 16384, 2048, 0, 128, 0) == 2
    # 17..64 tokens: the strip kernel's 32-token form up to 4 MiB of int4, the tcgen05 kernel otherwise and above 64 tokens
    assert query(64, 2048, 2048, 32, 128, 0) == 6
    assert query(17, 2048, 2048, 0, 128, 0) == 6
    assert query(64, 4096, 2048, 0, 128, 0) == 6          # exactly 4 MiB
    assert query(64, 2048, 8192, 32, 128, 0) == 3         # 8 MiB
    assert query(65, 2048, 2048, 32, 128, 0) == 3         # above 64 tokens
    assert query(2048, 2048, 2048, 0, 128, 0) == 3
    # a hand-written table overrides them and survives save -> load
    src = tmp_path / "plan.txt"
    src.write_text("# spear plan v1\n4 2048 2048 16 128 0 2 17.2 16.5 26.4 32.2 -1\n64 2048 2048 32 128 0 4 -1 -1 30.0 28.0 -1\n")
    assert L.spear_plan_load(str(src).encode()) == 0
    assert query(4, 2048, 2048, 16, 128, 0) == 2
    assert query(64, 2048, 2048, 32, 128, 0) == 4
    out = tmp_path / "saved.txt"
    assert L.spear_plan_save(str(out).encode()) == 0
    txt = out.read_text()
    assert "4 2048 2048 16 128 0 2" in txt and "64 2048 2048 32 128 0 4" in txt
    bad = tmp_path / "bad.txt"
    bad.write_text("1 2 3\n")
    assert L.spear_plan_load(str(bad).encode()) == -1


def test_variant_names_cover_every_variant_of_the_header():
    """The binding's variant table must follow include/spear.h (a stale list broke plan_configs when ROWS was added)."""
    import re
    import paper_2606_11244_b200 as sp
    hdr = open(os.path.join(ROOT, "include", "spear.h")).read()
    enum = dict((m.group(1), int(m.group(2))) for m in re.finditer(r"SPEAR_VARIANT_([A-Z_]+)\s*=\s*(\d+)", hdr))
    count = enum.pop("COUNT")
    assert sp.VARIANT_COUNT == count == len(sp.VARIANT_NAMES)
    for name, value in enum.items():
        assert sp.VARIANT_NAMES[value] == name.lower(), (name, value)
        assert getattr(sp, "VARIANT_" + name) == value
