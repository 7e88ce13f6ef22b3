"""Independent brute-force checker used to pin the oracle.

Different language (Python) and data structure (a sparse dict keyed by (pad, time)) from the oracle's dense
C arrays, and different formulations of every rule:
  * "earlier neighbour" is decided by Python's lexicographic tuple order on (pad, time), not by a listed
    offset set;
  * the peak rule is "the centre is the FIRST maximum of the 3x3 window in that order";
  * the gate cell of an outer-ring cell is found by arg-min Euclidean distance to the peak among the
    inner cells 8-adjacent to it (no sgn() arithmetic);
  * qTot is gathered arm-by-arm from the open inner cells, not tested per outer cell.
It imports neither oracle/ nor the product package.
"""
from fractions import Fraction
import math


def _get(cells, P, T, p, t):
    if p < 0 or p >= P or t < 0 or t >= T:
        return 0
    return cells.get((p, t), 0)


def is_peak(cells, P, T, p, t, q_peak_min=4):
    q = _get(cells, P, T, p, t)
    if q < q_peak_min:
        return False
    window = []
    for pp in (p - 1, p, p + 1):
        for tt in (t - 1, t, t + 1):
            window.append(((pp, tt), _get(cells, P, T, pp, tt)))
    window.sort(key=lambda kv: kv[0])
    best = max(v for _, v in window)
    first = next(k for k, v in window if v == best)
    return first == (p, t)


def gate_cell(dp, dt):
    """Inner cell gating outer-ring cell (dp,dt): nearest to the peak among 8-adjacent inner cells."""
    assert max(abs(dp), abs(dt)) == 2
    cand = []
    for ip in (-1, 0, 1):
        for it in (-1, 0, 1):
            if (ip, it) == (0, 0):
                continue
            if max(abs(ip - dp), abs(it - dt)) == 1:
                cand.append((ip * ip + it * it, (ip, it)))
    cand.sort()
    assert len(cand) == 1 or cand[0][0] < cand[1][0], "gate must be unique"
    return cand[0][1]


def arms():
    """inner cell -> list of the outer cells it gates."""
    a = {}
    for dp in range(-2, 3):
        for dt in range(-2, 3):
            if max(abs(dp), abs(dt)) == 2:
                a.setdefault(gate_cell(dp, dt), []).append((dp, dt))
    return a


_ARMS = arms()


def counted_cells(cells, P, T, p, t, q_inner_gate=2):
    """List of (dp, dt, charge) entering the cluster at peak (p,t): gather-by-gate formulation."""
    out = []
    for ip in (-1, 0, 1):
        for it in (-1, 0, 1):
            c = _get(cells, P, T, p + ip, t + it)
            out.append((ip, it, c))
            if (ip, it) != (0, 0) and c >= q_inner_gate:
                for (dp, dt) in _ARMS[(ip, it)]:
                    out.append((dp, dt, _get(cells, P, T, p + dp, t + dt)))
    return out


def cluster_at(cells, P, T, p, t, q_inner_gate=2):
    cc = counted_cells(cells, P, T, p, t, q_inner_gate)
    S0 = sum(c for _, _, c in cc)
    S1p = sum(c * dp for dp, _, c in cc)
    S1t = sum(c * dt for _, dt, c in cc)
    S2p = sum(c * dp * dp for dp, _, c in cc)
    S2t = sum(c * dt * dt for _, dt, c in cc)
    return S0, S1p, S1t, S2p, S2t


def moments_from_sums(p, t, S0, S1p, S1t, S2p, S2t):
    """Exact rational mean / variance, returned as Python floats (rounded once)."""
    mp, mt = Fraction(S1p, S0), Fraction(S1t, S0)
    vp = Fraction(S2p, S0) - mp * mp
    vt = Fraction(S2t, S0) - mt * mt
    return (float(p + mp), float(t + mt),
            math.sqrt(float(max(vp, 0))), math.sqrt(float(max(vt, 0))))


def find_clusters(cells, P, T, q_peak_min=4, q_inner_gate=2):
    """All clusters of one plane in (pad,time) order:
    list of (pad, time, qmax, S0, S1p, S1t, S2p, S2t)."""
    out = []
    for (p, t) in sorted(cells.keys()):
        if cells[(p, t)] == 0:
            continue
        if is_peak(cells, P, T, p, t, q_peak_min):
            out.append((p, t, cells[(p, t)]) + cluster_at(cells, P, T, p, t, q_inner_gate))
    return out


# ---- variants (DESIGN.md §3 V1..V3), formulated differently from the oracle ---------------
F_EDGE_PAD, F_EDGE_TIME, F_SINGLE_PAD, F_SINGLE_TIME, F_SATURATED = 1, 2, 4, 8, 16


def cluster_flags(cells, P, T, p, t, q_inner_gate=2, q_saturation=0):
    """V1 by enumeration: EDGE_* iff some cell of the 5x5 window falls outside the plane in that coordinate;
    SINGLE_* iff the set of pads / time bins that contributed charge is just the peak's own."""
    fl = 0
    window = [(p + dp, t + dt) for dp in range(-2, 3) for dt in range(-2, 3)]
    if any(pp < 0 or pp >= P for pp, _ in window):
        fl |= F_EDGE_PAD
    if any(tt < 0 or tt >= T for _, tt in window):
        fl |= F_EDGE_TIME
    cc = [(dp, dt) for dp, dt, c in counted_cells(cells, P, T, p, t, q_inner_gate) if c > 0]
    if {dp for dp, _ in cc} <= {0}:
        fl |= F_SINGLE_PAD
    if {dt for _, dt in cc} <= {0}:
        fl |= F_SINGLE_TIME
    if q_saturation and cells[(p, t)] >= q_saturation:
        fl |= F_SATURATED
    return fl


def find_clusters_variants(cells, P, T, q_peak_min=4, q_inner_gate=2, q_tot_min=0, q_saturation=0,
                           cut_single_pad=False, cut_single_time=False):
    """V2/V3: the base list, each entry with its flags appended, minus the entries that fail a cut."""
    out = []
    for c in find_clusters(cells, P, T, q_peak_min, q_inner_gate):
        fl = cluster_flags(cells, P, T, c[0], c[1], q_inner_gate, q_saturation)
        if c[3] < q_tot_min:
            continue
        if (cut_single_pad and fl & F_SINGLE_PAD) or (cut_single_time and fl & F_SINGLE_TIME):
            continue
        out.append(c + (fl,))
    return out


# ---- V4 charge sharing (DESIGN.md §3 V4), formulated differently from the oracle ------------------------------------
F_SHARED = 32


def find_clusters_shared(cells, P, T, q_peak_min=4, q_inner_gate=2, q_tot_min=0, q_saturation=0,
                         cut_single_pad=False, cut_single_time=False):
    """V4 by enumeration of the cluster list (no peak-charge map, no box sum): the weight of cluster k on a cell is
    qmax_k over the summed qmax of the listed clusters whose peak lies within Chebyshev distance 2 of the cell; the
    share is the floor of an exact Fraction.  Entries: (pad, time, qmax, qtot, S0', S1p', S1t', S2p', S2t', flags)."""
    base = find_clusters_variants(cells, P, T, q_peak_min, q_inner_gate, q_tot_min, q_saturation,
                                  cut_single_pad, cut_single_time)
    out = []
    for (p, t, qmax, _S0, _a, _b, _c, _d, fl) in base:
        sums = [0, 0, 0, 0, 0]
        shared = False
        for dp, dt, c in counted_cells(cells, P, T, p, t, q_inner_gate):
            x = (p + dp, t + dt)
            claim = sum(k[2] for k in base if max(abs(k[0] - x[0]), abs(k[1] - x[1])) <= 2)
            if c > 0 and claim != qmax:
                shared = True
            share = math.floor(Fraction(64 * c * qmax, claim))
            for i, w in enumerate((1, dp, dt, dp * dp, dt * dt)):
                sums[i] += share * w
        qtot = math.floor(Fraction(sums[0], 64) + Fraction(1, 2))
        out.append((p, t, qmax, qtot) + tuple(sums) + (fl | (F_SHARED if shared else 0),))
    return out


def moments_from_shared_sums(p, t, S0, S1p, S1t, S2p, S2t):
    """moments_from_sums with V4's degenerate case: all shares rounded to zero -> the peak's position, sigmas 0."""
    if S0 == 0:
        return float(p), float(t), 0.0, 0.0
    return moments_from_sums(p, t, S0, S1p, S1t, S2p, S2t)
