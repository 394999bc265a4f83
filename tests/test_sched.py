"""PAPER.md 4.3 (:231-:237): latency look-up tables, the online aggregator T_S(M) and the SLO-constrained chunk selection.
CPU only: the oracle (oracle/sched_oracle.py, a linear scan in exact rationals) is pinned to a hand-computed example and
to its own invariants; the product (csrc/sched.cu through the C ABI, binary search) is compared with the oracle on the
example and on a seeded synthetic Poisson arrival trace (the paper replays ShareGPT requests, :274 -- not available and
not recreated here; the trace only supplies (d, T_SLO, c_max) triples)."""
import json
import os
from fractions import Fraction

import numpy as np
import pytest

from oracle import sched_oracle as so

GOLD = os.path.join(os.path.dirname(__file__), "golden", "slo_chunk_worked_example.json")


def gold():
    with open(GOLD) as f:
        return json.load(f)


# ---------------------------------------------------------------- oracle pins

def test_oracle_worked_example():
    g = gold()
    args = (g["grid"], g["lat_w4"], g["lat_ec"], g["lat_attn"], g["module_type"], g["selected"], g["n_attn"])
    for M, want in g["T"].items():
        assert abs(float(so.iteration_us(*args, int(M))) - want) < 1e-9, M
    assert so.iteration_us(*args, 8) == Fraction(*g["T_8_fraction"])
    for c in g["chunks"]:
        assert so.slo_chunk(*args, c["d"], c["c_min"], c["c_max"], c["t_slo"]) == c["c"], c


def test_oracle_interpolation_against_numpy_and_selection_semantics():
    rng = np.random.default_rng(0)
    grid = [1, 4, 16, 64, 256, 1024]
    w4 = np.sort(rng.uniform(5, 500, (3, 6)), axis=1)
    ec = w4 * rng.uniform(1.0, 1.3, (3, 6))
    ec = np.maximum.accumulate(ec, axis=1)
    types = [0, 1, 2, 1, 0]
    sel = [1, 0, 1, 0, 0]
    for M in (1, 2, 5, 16, 100, 700, 1024):
        want = sum(np.interp(M, grid, (ec if s else w4)[t]) for t, s in zip(types, sel))
        assert abs(float(so.iteration_us(grid, w4.tolist(), ec.tolist(), None, types, sel, 0, M)) - want) < 1e-9
    # selecting a module never makes the iteration cheaper (l_EC >= l_W4 here), deselecting everything gives the backbone
    t_none = so.iteration_us(grid, w4.tolist(), ec.tolist(), None, types, None, 0, 100)
    t_sel = so.iteration_us(grid, w4.tolist(), ec.tolist(), None, types, sel, 0, 100)
    assert t_sel >= t_none
    assert t_none == sum(so.interp(grid, w4[t].tolist(), 100) for t in types)


def test_oracle_monotone_and_scan_properties():
    rng = np.random.default_rng(1)
    grid = [1, 8, 32, 128, 512]
    w4 = rng.uniform(5, 300, (2, 5)).tolist()          # NOT sorted: the running maximum must repair it
    ec = rng.uniform(5, 300, (2, 5)).tolist()
    types, sel = [0, 1, 1, 0], [1, 1, 0, 0]
    T = [so.iteration_us(grid, w4, ec, None, types, sel, 0, M) for M in range(0, 600)]
    assert all(b >= a for a, b in zip(T, T[1:]))        # T_S monotone
    for t_slo in (50.0, 400.0, 900.0, 5000.0):
        c = so.slo_chunk(grid, w4, ec, None, types, sel, 0, 4, 1, 512, t_slo)
        if c:
            assert T[4] + T[c] <= Fraction(t_slo)
            assert c == 512 or T[4] + T[c + 1] > Fraction(t_slo)      # maximal
        else:
            assert T[4] + T[1] > Fraction(t_slo)


# ---------------------------------------------------------------- product (C ABI, binary search) against the oracle

@pytest.fixture(scope="module")
def sp():
    import paper_2606_11244_b200 as sp
    return sp


def test_product_worked_example(sp):
    g = gold()
    lut = sp.Lut(g["grid"], g["lat_w4"], g["lat_ec"], g["lat_attn"])
    for M, want in g["T"].items():
        assert abs(lut.iteration_us(g["module_type"], g["selected"], int(M), g["n_attn"]) - want) < 1e-6, M
    for c in g["chunks"]:
        assert lut.slo_chunk(g["module_type"], g["selected"], c["d"], c["c_min"], c["c_max"], c["t_slo"], g["n_attn"]) == c["c"]


def test_product_matches_the_linear_scan_on_a_synthetic_poisson_trace(sp):
    """Seeded synthetic serving trace: per scheduling step the number of decode tokens in flight d follows a Poisson
    process of arrivals and departures; T_SLO and c_max vary.  The binary search must return the scan's answer."""
    rng = np.random.default_rng(2026)
    grid = [1, 2, 4, 8, 16, 32, 64, 128, 256, 512, 1024, 2048]
    base = np.array([9.0, 9.2, 9.5, 10.0, 11.0, 14.0, 21.0, 38.0, 70.0, 135.0, 265.0, 520.0])     # a decode-to-prefill shaped curve
    w4 = np.stack([base * s for s in (1.0, 0.7, 5.0, 2.6)])
    ec = w4 * np.array([[1.08], [1.12], [1.05], [1.07]]) + 1.5
    attn = base * 0.4
    n_layers = 6
    types = [t for _ in range(n_layers) for t in (0, 1, 2, 3)]
    sel = [1 if (l in (0, 1, 5) and t in (1, 3)) else 0 for l in range(n_layers) for t in (0, 1, 2, 3)]
    lut = sp.Lut(grid, w4.tolist(), ec.tolist(), attn.tolist())
    d = 0
    for step in range(30):
        d = max(0, d + int(rng.poisson(1.6)) - int(rng.poisson(1.5)))
        t_slo = float(rng.choice([1500.0, 3000.0, 9000.0]))
        c_max = int(rng.choice([128, 256, 768]))
        want = so.slo_chunk(grid, w4.tolist(), ec.tolist(), attn.tolist(), types, sel, n_layers, d, 16, c_max, t_slo)
        got = lut.slo_chunk(types, sel, d, 16, c_max, t_slo, n_layers)
        t_want = float(so.iteration_us(grid, w4.tolist(), ec.tolist(), attn.tolist(), types, sel, n_layers, d))
        assert abs(lut.iteration_us(types, sel, d, n_layers) - t_want) <= 1e-6 * max(1.0, t_want)
        assert got == want, (step, d, t_slo, c_max)


def test_product_argument_errors(sp):
    with pytest.raises(sp.SpearError):
        sp.Lut([4, 2], [[1, 2]], [[1, 2]])
    lut = sp.Lut([1, 16], [[1, 2]], [[1, 2]])
    with pytest.raises(sp.SpearError):
        lut.iteration_us([3], None, 8)
    with pytest.raises(sp.SpearError):
        lut.slo_chunk([0], None, 0, 8, 4, 10.0)
