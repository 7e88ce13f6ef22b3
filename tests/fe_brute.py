"""Independent restatement of TPC-FE v1 (include/tpc_fe.h) for checking the C oracle: another language, another
order of evaluation (the common-mode values of all time bins first, as one masked numpy reduction; then every pad line
on its own, start to end), exact rationals for the two roundings.  Test infrastructure; small inputs only."""
from fractions import Fraction
import math

import numpy as np


def half_up(fr):
    return math.floor(fr + Fraction(1, 2))


def filter_plane(raw, ped4, P, zs_threshold, cm_quiet4, cm_min_pads, it_decay_shift, it_kappa_shift):
    """raw [T, W] uint16, ped4 [W] -> list of (pad, time, q), pad-major."""
    T = raw.shape[0]
    x = 4 * raw[:, :P].astype(np.int64) - ped4[:P].astype(np.int64)[None, :]
    quiet = np.abs(x) <= cm_quiet4
    n = quiet.sum(axis=1)
    s = np.where(quiet, x, 0).sum(axis=1)
    cm = [half_up(Fraction(int(s[t]), int(n[t]))) if n[t] >= cm_min_pads else 0 for t in range(T)]
    out = []
    for p in range(P):
        S = 0
        for t in range(T):
            z = int(x[t, p]) - cm[t] + S // 4096
            q = min(half_up(Fraction(z, 4)), 65535)
            kept = q >= zs_threshold
            S = S - S // (1 << it_decay_shift)
            if kept:
                out.append((p, t, q))
                if it_kappa_shift:
                    S += q << (14 - it_kappa_shift)
    return out


def run(raw, ped4, n_sectors, n_rows, max_pads, n_time, npads=None, **prm):
    res = []
    for pl in range(n_sectors * n_rows):
        P = int(npads[pl % n_rows]) if npads is not None else max_pads
        for (p, t, q) in filter_plane(raw[pl], ped4[pl], P, **prm):
            res.append((pl // n_rows, pl % n_rows, p, t, q))
    return res
