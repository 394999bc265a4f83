"""CPU oracle for the paper's latency tables and SLO-constrained chunk selection -- TEST INFRASTRUCTURE ONLY.

Plain Python, written from PAPER.md section 4.3 (:231-:237); shares no code with csrc/sched.cu.

  T_S(M) = sum over linear layers m of (l_EC if m in S else l_W4)[type(m)](M) + n_attn * l_attn(M)      (:231)
           with "linear interpolation ... for unseen M" (:231) between the grid points of the offline tables
  chunk  = the largest c in [c_min, c_max] with T_S(d) + T_S(c) <= T_SLO                                 (:235)
           -- found here by the plain linear scan over every c (the paper's binary search, :237, is the
           product's job; it must agree with the scan whenever T_S is monotone)

Readings: T_S(0) = 0 (no tokens, no iteration); below the first grid point the first entry;
above the last grid point the last segment extended; a table entry smaller than its predecessor is raised to it
before use (running maximum), so that T_S is monotone as :237 assumes.
"""
from fractions import Fraction


def monotone(row):
    out, cur = [], 0.0
    for v in row:
        v = float(v)
        if not v >= 0.0:
            v = 0.0
        cur = max(cur, v) if out else v
        out.append(cur)
    return out


def interp(grid, row, M):
    """Piecewise-linear table value at token count M (exact rational arithmetic on the float entries)."""
    if M <= 0:
        return Fraction(0)
    if M <= grid[0] or len(grid) == 1:
        return Fraction(row[0])
    hi = next((i for i, g in enumerate(grid) if g > M), len(grid) - 1)
    lo = hi - 1
    t = Fraction(M - grid[lo], grid[hi] - grid[lo])
    return Fraction(row[lo]) + t * (Fraction(row[hi]) - Fraction(row[lo]))


def iteration_us(grid, lat_w4, lat_ec, lat_attn, module_type, selected, n_attn, M):
    if M <= 0:
        return Fraction(0)
    w4 = [monotone(r) for r in lat_w4]
    ec = [monotone(r) for r in lat_ec]
    attn = monotone(lat_attn) if lat_attn is not None else [0.0] * len(grid)
    t = Fraction(0)
    for m, ty in enumerate(module_type):
        t += interp(grid, (ec if (selected is not None and selected[m]) else w4)[ty], M)
    return t + n_attn * interp(grid, attn, M)


def slo_chunk(grid, lat_w4, lat_ec, lat_attn, module_type, selected, n_attn, d, c_min, c_max, t_slo_us):
    """Linear scan: the largest feasible c, 0 when none is."""
    td = iteration_us(grid, lat_w4, lat_ec, lat_attn, module_type, selected, n_attn, d)
    best = 0
    for c in range(c_min, c_max + 1):
        if td + iteration_us(grid, lat_w4, lat_ec, lat_attn, module_type, selected, n_attn, c) <= Fraction(t_slo_us):
            best = c
    return best
