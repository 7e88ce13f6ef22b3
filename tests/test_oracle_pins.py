"""Pins for the CPU oracle (-m "not gpu").  Each test checks the oracle against something other than itself:
hand-evaluated grids (tests/golden/worked_examples.txt), a brute-force sparse-dict checker (tests/brute.py),
library routines on special cases (numpy argmax, box sums, weighted moments), closed forms and invariants.
Citations: SURVEY.md §8(c) E1..E15, P1..P7, I1..I9 (definition: BASELINE.json:north_star; step: PAPER.md:57).
"""
import os

import numpy as np
import pytest

from oracle import oracle as orc
import brute

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "worked_examples.txt")


def parse_golden(path=GOLDEN):
    ex, cur = [], None
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        tag, rest = line[0], line[1:].split()
        if tag == "E":
            cur = {"name": rest[0], "digits": [], "clusters": []}
            ex.append(cur)
        elif tag == "D":
            cur["digits"].append(tuple(int(x) for x in rest))
        elif tag == "C":
            cur["clusters"].append(tuple(int(x) for x in rest))
    return ex


EXAMPLES = parse_golden()


def run_plane(cells, P=12, T=12, **kw):
    d = orc.make_digits(cells)
    return orc.run(d, 1, 1, P, T, **kw)


def check_against_sums(clusters, expected):
    """expected: list of (pad,time,qmax,S0,S1p,S1t,S2p,S2t).  Integers exact; floats to 1 ulp of float32."""
    assert len(clusters) == len(expected)
    for c, e in zip(clusters, expected):
        p, t, qmax, S0, S1p, S1t, S2p, S2t = e
        assert (int(c["pad"]), int(c["time"]), int(c["qmax"]), int(c["qtot"])) == (p, t, qmax, S0)
        assert int(c["flags"]) == 0 and int(c["rsv"]) == 0
        pm, tm, sp, stime = brute.moments_from_sums(p, t, S0, S1p, S1t, S2p, S2t)
        for got, want in ((c["pad_mean"], pm), (c["time_mean"], tm), (c["sigma_pad"], sp), (c["sigma_time"], stime)):
            w32 = np.float32(want)
            assert abs(float(got) - float(w32)) <= float(np.spacing(w32)), (got, want)


def test_golden_file_has_all_examples():
    names = [e["name"].split("_")[0] for e in EXAMPLES]
    assert names == ["E1", "E2", "E3", "E4a", "E4b", "E4c", "E5", "E6", "E7", "E8", "E9", "E10",
                     "E11", "E12", "E13", "E14", "E15"]


@pytest.mark.parametrize("ex", EXAMPLES, ids=[e["name"] for e in EXAMPLES])
def test_worked_example(ex):
    clusters, st = run_plane(ex["digits"])
    assert st["n_clusters"] == len(ex["clusters"]) and st["n_bad_digits"] == 0
    check_against_sums(clusters, ex["clusters"])


def test_printed_values_of_survey_table():
    """Decimal values printed in SURVEY.md §8(c) for E2, E4c, E11, E12, E14 (closed forms)."""
    by = {e["name"].split("_")[0]: e for e in EXAMPLES}
    c, _ = run_plane(by["E2"]["digits"])
    assert float(c[0]["pad_mean"]) == 5.375 and abs(float(c[0]["sigma_pad"]) - np.sqrt(0.234375)) < 1e-7
    c, _ = run_plane(by["E4c"]["digits"])
    assert int(c[0]["qtot"]) == 15 and abs(float(c[0]["time_mean"]) - 7.2) < 1e-6
    c, _ = run_plane(by["E11"]["digits"])
    assert float(c[0]["sigma_pad"]) == 1.0 and float(c[0]["sigma_time"]) == 1.0 and int(c[0]["qtot"]) == 256
    c, _ = run_plane(by["E12"]["digits"])
    assert float(c[0]["sigma_pad"]) == 1.0 and abs(float(c[0]["sigma_time"]) - np.sqrt(0.5)) < 1e-7
    c, _ = run_plane(by["E14"]["digits"])
    assert abs(float(c[0]["sigma_pad"]) - 0.016571481) < 2e-9


# ---- P1: peak rule == numpy.argmax first-occurrence on the 3x3 window -------------------------------------

def test_peak_rule_equals_argmax_exhaustive():
    """All 4^9 windows over {0,3,4,5}: centre is a peak iff q>=4 and argmax(window.ravel())==4."""
    vals = np.array([0, 3, 4, 5], dtype=np.uint16)
    idx = np.arange(4 ** 9)
    # pack the windows into planes, spaced 4 apart so that windows do not touch
    per_row, T = 64, 64 * 4 + 2
    n = idx.size
    rows_per_plane = 60
    win = vals[(idx[:, None] // 4 ** np.arange(9)[None, :]) % 4]          # [n, 9] pad-major/time-minor
    want_peak = (win[:, 4] >= 4) & (np.argmax(win, axis=1) == 4)
    n_planes = (n + per_row * rows_per_plane - 1) // (per_row * rows_per_plane)
    dig = []
    for k in range(n):
        plane, rem = divmod(k, per_row * rows_per_plane)
        wr, wc = divmod(rem, per_row)
        p0, t0 = 1 + 4 * wr, 1 + 4 * wc
        for j in range(9):
            if win[k, j]:
                dig.append((plane, p0 + j // 3 - 1, t0 + j % 3 - 1, int(win[k, j])))
    d = np.zeros(len(dig), dtype=orc.DIGIT)
    arr = np.array(dig, dtype=np.int64)
    d["sector"] = 0
    d["row"] = arr[:, 0]
    d["pad"] = arr[:, 1]
    d["time"] = arr[:, 2]
    d["charge"] = arr[:, 3]
    Pp = 4 * rows_per_plane + 2
    clusters, st = orc.run(d, 1, n_planes, Pp, T)
    # a window's neighbours may also be peaks (centre is not the only candidate): look only at centres
    got = np.zeros(n, dtype=bool)
    cr, cp, ct = clusters["row"].astype(np.int64), clusters["pad"].astype(np.int64), clusters["time"].astype(np.int64)
    centre = ((cp - 1) % 4 == 0) & ((ct - 1) % 4 == 0)
    k = cr[centre] * per_row * rows_per_plane + ((cp[centre] - 1) // 4) * per_row + (ct[centre] - 1) // 4
    got[k] = True
    assert np.array_equal(got, want_peak)


def random_cells(rng, P, T, n, alphabet):
    cells = {}
    for _ in range(n):
        cells[(int(rng.integers(P)), int(rng.integers(T)))] = int(rng.choice(alphabet))
    return cells


@pytest.mark.parametrize("alphabet,fill", [((3, 4, 5, 9), 14), ((1, 2, 4, 7, 7, 30), 20), ((4,), 18),
                                           ((1, 2, 3, 65535, 65534), 16)])
def test_brute_force_random_tiny_grids(alphabet, fill):
    """Oracle == brute-force checker (peaks, qMax, qTot, all five sums via floats) on many 6x6 grids."""
    rng = np.random.default_rng(1234 + fill)
    P = T = 6
    n_grids = 3000
    digs = []
    expected = []
    for gidx in range(n_grids):
        cells = random_cells(rng, P, T, fill, alphabet)
        exp = brute.find_clusters(cells, P, T)
        expected.append(exp)
        for (p, t), q in cells.items():
            digs.append((gidx // 200, gidx % 200, p, t, q))
    arr = np.array(digs, dtype=np.int64)
    d = np.zeros(arr.shape[0], dtype=orc.DIGIT)
    d["sector"], d["row"], d["pad"], d["time"], d["charge"] = arr.T
    rng.shuffle(d)                                            # any input order (I1 / R12)
    clusters, st = orc.run(d, n_grids // 200, 200, P, T)
    assert st["n_clusters"] == sum(len(e) for e in expected)
    pos = 0
    for gidx, exp in enumerate(expected):
        got = clusters[pos:pos + len(exp)]
        pos += len(exp)
        assert np.all(got["sector"] == gidx // 200) and np.all(got["row"] == gidx % 200)
        check_against_sums(got, exp)


# ---- P2: gate table ----------------------------------------------------------------------------------------

def test_gate_table_single_outer_cells():
    """32 grids: peak 10 at (5,5), one outer-ring cell of 3, its gate cell (by arg-min distance) 2 or 1."""
    for dp in range(-2, 3):
        for dt in range(-2, 3):
            if max(abs(dp), abs(dt)) != 2:
                continue
            gp, gt = brute.gate_cell(dp, dt)
            for gate_q, expect in ((2, 15), (1, 11)):
                cells = [(5, 5, 10), (5 + gp, 5 + gt, gate_q), (5 + dp, 5 + dt, 3)]
                c, _ = run_plane(cells)
                assert len(c) == 1 and int(c[0]["qtot"]) == expect, (dp, dt, gate_q)
                # every OTHER inner cell open must not open this outer cell
                others = [(5, 5, 10), (5 + dp, 5 + dt, 3)]
                for ip in (-1, 0, 1):
                    for it in (-1, 0, 1):
                        if (ip, it) not in ((0, 0), (gp, gt)):
                            others.append((5 + ip, 5 + it, 2))
                c, _ = run_plane(others)
                assert int(c[0]["qtot"]) == 10 + 2 * 7, (dp, dt)


# ---- P3: qTot special cases that reduce to box sums -------------------------------------------------------

def box_sum(a, k):
    r = k // 2
    pad = np.pad(a.astype(np.int64), r)
    out = np.zeros(a.shape, dtype=np.int64)
    for i in range(k):
        for j in range(k):
            out += pad[i:i + a.shape[0], j:j + a.shape[1]]
    return out


def random_plane(rng, P, T, occ, qmax=200):
    a = np.zeros((P, T), dtype=np.uint16)
    m = rng.random((P, T)) < occ
    a[m] = rng.integers(1, qmax, size=int(m.sum()))
    return a


def plane_to_digits(a, sector=0, row=0):
    p, t = np.nonzero(a)
    d = np.zeros(p.size, dtype=orc.DIGIT)
    d["sector"], d["row"], d["pad"], d["time"], d["charge"] = sector, row, p, t, a[p, t]
    return d


def test_qtot_all_gates_open_is_box5_and_closed_is_box3():
    rng = np.random.default_rng(7)
    a = random_plane(rng, 40, 90, 0.2)
    d = plane_to_digits(a)
    c5, _ = orc.run(d, 1, 1, 40, 90, q_inner_gate=0)
    c3, _ = orc.run(d, 1, 1, 40, 90, q_inner_gate=65535)
    cd, _ = orc.run(d, 1, 1, 40, 90)
    assert len(c5) == len(c3) == len(cd) > 50
    b5, b3 = box_sum(a, 5), box_sum(a, 3)
    p, t = c5["pad"].astype(int), c5["time"].astype(int)
    assert np.array_equal(c5["qtot"].astype(np.int64), b5[p, t])
    assert np.array_equal(c3["qtot"].astype(np.int64), b3[p, t])
    # bounds: qMax <= box3 <= qTot <= box5
    assert np.all(cd["qmax"] <= cd["qtot"])
    assert np.all(b3[p, t] <= cd["qtot"]) and np.all(cd["qtot"] <= b5[p, t])
    # peak positions == argmax-first-occurrence rule evaluated with numpy on the dense plane
    padded = np.pad(a, 1)
    win = np.stack([padded[i:i + 40, j:j + 90] for i in range(3) for j in range(3)], axis=-1)
    is_peak = (a >= 4) & (np.argmax(win, axis=-1) == 4)
    pp, tt = np.nonzero(is_peak)
    assert np.array_equal(pp, p) and np.array_equal(tt, t)


def test_moments_all_gates_open_equal_numpy_weighted_moments():
    rng = np.random.default_rng(11)
    a = random_plane(rng, 30, 60, 0.25, qmax=1000)
    d = plane_to_digits(a)
    c, _ = orc.run(d, 1, 1, 30, 60, q_inner_gate=0)
    padded = np.pad(a, 2).astype(np.float64)
    for k in range(len(c)):
        p, t = int(c[k]["pad"]), int(c[k]["time"])
        w = padded[p:p + 5, t:t + 5]
        pads = np.arange(p - 2, p + 3, dtype=np.float64)
        times = np.arange(t - 2, t + 3, dtype=np.float64)
        mp = np.average(pads, weights=w.sum(axis=1))
        mt = np.average(times, weights=w.sum(axis=0))
        sp = np.sqrt(np.cov(pads, aweights=w.sum(axis=1), ddof=0))
        stime = np.sqrt(np.cov(times, aweights=w.sum(axis=0), ddof=0))
        assert abs(float(c[k]["pad_mean"]) - mp) <= 2e-6 * max(1, abs(mp))
        assert abs(float(c[k]["time_mean"]) - mt) <= 2e-6 * max(1, abs(mt))
        assert abs(float(c[k]["sigma_pad"]) - sp) <= 1e-5
        assert abs(float(c[k]["sigma_time"]) - stime) <= 1e-5


def test_max_charge_everywhere_is_exact():
    """P5: all 25 cells = 65535: sums stay below 2^24; one peak (rectangular plateau), qTot = 25*65535."""
    cells = [(p, t, 65535) for p in range(3, 8) for t in range(3, 8)]
    c, st = run_plane(cells)
    assert st["n_clusters"] == 1
    assert (int(c[0]["pad"]), int(c[0]["time"])) == (3, 3)
    assert int(c[0]["qtot"]) == 9 * 65535            # window of (3,3) covers pads 3..5, times 3..5
    cells = [(p, t, 65534) for p in range(3, 8) for t in range(3, 8) if (p, t) != (5, 5)] + [(5, 5, 65535)]
    c, st = run_plane(cells)
    # (3,3) is the first cell of the surrounding 65534 plateau and (5,5) is outside its 3x3: two peaks
    assert [(int(x["pad"]), int(x["time"])) for x in c] == [(3, 3), (5, 5)]
    assert int(c[1]["qtot"]) == 24 * 65534 + 65535 and float(c[1]["sigma_pad"]) > 1.41


@pytest.mark.parametrize("kp,kt", [(1, 2), (2, 2), (3, 5), (1, 5), (3, 1)])
def test_rectangular_plateau_has_one_peak_at_first_cell(kp, kt):
    cells = [(4 + i, 3 + j, 50) for i in range(kp) for j in range(kt)] + [(3, 3, 7), (8, 9, 2)]
    c, _ = run_plane(cells)
    peaks = [(int(x["pad"]), int(x["time"])) for x in c if int(x["qmax"]) == 50]
    assert peaks == [(4, 3)]


# ---- P6 invariants ----------------------------------------------------------------------------------------

def frame(rng, S=2, R=3, P=20, T=50, occ=0.12):
    ds = []
    for s in range(S):
        for r in range(R):
            ds.append(plane_to_digits(random_plane(rng, P, T, occ), s, r))
    return np.concatenate(ds)


def test_I1_permutation_invariance_and_P7_order():
    rng = np.random.default_rng(3)
    d = frame(rng)
    c0, s0 = orc.run(d, 2, 3, 20, 50)
    d2 = d.copy()
    rng.shuffle(d2)
    c1, s1 = orc.run(d2, 2, 3, 20, 50)
    assert s0 == s1 and c0.tobytes() == c1.tobytes()
    key = (c0["sector"].astype(np.int64) << 32) | (c0["row"].astype(np.int64) << 24) | \
          (c0["pad"].astype(np.int64) << 16) | c0["time"].astype(np.int64)
    assert np.all(np.diff(key) > 0)


def test_I2_translation():
    rng = np.random.default_rng(5)
    a = np.zeros((40, 80), dtype=np.uint16)
    a[10:25, 10:50] = random_plane(rng, 15, 40, 0.2)
    b = np.zeros_like(a)
    b[17:32, 33:73] = a[10:25, 10:50]
    ca, _ = orc.run(plane_to_digits(a), 1, 1, 40, 80)
    cb, _ = orc.run(plane_to_digits(b), 1, 1, 40, 80)
    assert len(ca) == len(cb) > 5
    for f in ("qmax", "qtot", "sigma_pad", "sigma_time"):
        assert np.array_equal(ca[f], cb[f])
    assert np.array_equal(ca["pad"] + 7, cb["pad"]) and np.array_equal(ca["time"] + 23, cb["time"])
    assert np.allclose(ca["pad_mean"] + 7, cb["pad_mean"], atol=4e-6)
    assert np.allclose(ca["time_mean"] + 23, cb["time_mean"], atol=8e-6)


def test_I3_relabel_planes_and_I7_union():
    rng = np.random.default_rng(9)
    a = plane_to_digits(random_plane(rng, 20, 50, 0.15), 0, 0)
    b = plane_to_digits(random_plane(rng, 20, 50, 0.15), 0, 0)
    ca, _ = orc.run(a, 1, 1, 20, 50)
    cb, _ = orc.run(b, 1, 1, 20, 50)
    a2, b2 = a.copy(), b.copy()
    a2["sector"], a2["row"] = 1, 2
    b2["sector"], b2["row"] = 0, 1
    cu, _ = orc.run(np.concatenate([a2, b2]), 2, 3, 20, 50)
    assert len(cu) == len(ca) + len(cb)
    first, second = cu[:len(cb)].copy(), cu[len(cb):].copy()
    assert np.all(first["sector"] == 0) and np.all(first["row"] == 1)
    assert np.all(second["sector"] == 1) and np.all(second["row"] == 2)
    first["sector"], first["row"], second["sector"], second["row"] = 0, 0, 0, 0
    assert first.tobytes() == cb.tobytes() and second.tobytes() == ca.tobytes()


def test_I4_charge_scaling():
    rng = np.random.default_rng(13)
    a = random_plane(rng, 20, 50, 0.15, qmax=100)
    c1, _ = orc.run(plane_to_digits(a), 1, 1, 20, 50)
    c3, _ = orc.run(plane_to_digits(a * 3), 1, 1, 20, 50, q_peak_min=12, q_inner_gate=6)
    assert np.array_equal(c1["pad"], c3["pad"]) and np.array_equal(c1["time"], c3["time"])
    assert np.array_equal(c1["qtot"] * 3, c3["qtot"]) and np.array_equal(c1["qmax"] * 3, c3["qmax"])
    for f in ("pad_mean", "time_mean", "sigma_pad", "sigma_time"):
        assert np.allclose(c1[f], c3[f], rtol=3e-7, atol=1e-6)


def distinct_plane(rng, P, T, occ):
    """plateau-free: all non-zero charges distinct."""
    a = np.zeros(P * T, dtype=np.uint16)
    n = int(P * T * occ)
    pos = rng.choice(P * T, size=n, replace=False)
    a[pos] = rng.permutation(np.arange(2, 2 + n)).astype(np.uint16)
    return a.reshape(P, T)


def test_I5_time_reflection_and_I6_transpose():
    rng = np.random.default_rng(17)
    a = distinct_plane(rng, 30, 30, 0.2)
    c, _ = orc.run(plane_to_digits(a), 1, 1, 30, 30)
    cr, _ = orc.run(plane_to_digits(a[:, ::-1]), 1, 1, 30, 30)
    ct, _ = orc.run(plane_to_digits(a.T), 1, 1, 30, 30)
    assert len(c) == len(cr) == len(ct) > 10
    key = lambda x, pf, tf: sorted(zip(pf.tolist(), tf.tolist(), x["qmax"].tolist(), x["qtot"].tolist()))
    assert key(c, c["pad"], c["time"]) == key(cr, cr["pad"], 29 - cr["time"].astype(int))
    assert key(c, c["pad"], c["time"]) == key(ct, ct["time"], ct["pad"])
    # means reflected / swapped, sigmas equal / swapped
    m = {(int(x["pad"]), int(x["time"])): x for x in c}
    for x in cr:
        o = m[(int(x["pad"]), 29 - int(x["time"]))]
        assert abs((29 - float(x["time_mean"])) - float(o["time_mean"])) < 1e-5
        assert abs(float(x["sigma_time"]) - float(o["sigma_time"])) < 1e-6
        assert float(x["pad_mean"]) == float(o["pad_mean"])
    for x in ct:
        o = m[(int(x["time"]), int(x["pad"]))]
        assert float(x["pad_mean"]) == float(o["time_mean"]) and float(x["sigma_pad"]) == float(o["sigma_time"])


def test_I8_threshold_above_max_and_I9_gate_monotone():
    rng = np.random.default_rng(19)
    a = random_plane(rng, 20, 50, 0.2, qmax=60)
    d = plane_to_digits(a)
    c, st = orc.run(d, 1, 1, 20, 50, q_peak_min=60)
    assert st["n_clusters"] == 0 and len(c) == 0
    prev = None
    for gate in (0, 1, 2, 5, 20, 70):
        c, _ = orc.run(d, 1, 1, 20, 50, q_inner_gate=gate)
        if prev is not None:
            assert np.array_equal(c["pad"], prev["pad"]) and np.all(c["qtot"] <= prev["qtot"])
        prev = c


# ---- contract details -------------------------------------------------------------------------------------

def test_bad_digits_are_skipped_and_counted():
    good = [(5, 7, 10), (6, 7, 6)]
    d = orc.make_digits(good + [(12, 3, 9), (3, 12, 9), (4, 4, 0)])
    extra = np.zeros(2, dtype=orc.DIGIT)
    extra[0] = (1, 0, 3, 0, 3, 9)      # sector out of range
    extra[1] = (0, 1, 3, 0, 3, 9)      # row out of range
    c, st = orc.run(np.concatenate([d, extra]), 1, 1, 12, 12)
    assert st["n_bad_digits"] == 5 and st["n_digits_used"] == 2 and st["n_clusters"] == 1
    assert int(c[0]["qtot"]) == 16


def test_npads_per_row_bounds_the_plane():
    """R19: cells with pad >= npads[row] do not exist: digits there are bad, reads give 0."""
    npads = np.array([6, 12], dtype=np.uint16)
    d0 = orc.make_digits([(5, 5, 10), (6, 5, 30)], row=0)       # pad 6 invalid in row 0
    d1 = orc.make_digits([(5, 5, 10), (6, 5, 30)], row=1)
    c, st = orc.run(np.concatenate([d0, d1]), 1, 2, 12, 12, npads=npads)
    assert st["n_bad_digits"] == 1 and st["n_clusters"] == 2
    assert (int(c[0]["row"]), int(c[0]["pad"]), int(c[0]["qtot"])) == (0, 5, 10)
    assert (int(c[1]["row"]), int(c[1]["pad"]), int(c[1]["qtot"])) == (1, 6, 40)


def test_capacity_overflow_keeps_first_clusters_in_order():
    rng = np.random.default_rng(23)
    d = frame(rng)
    full, st = orc.run(d, 2, 3, 20, 50)
    part, st2 = orc.run(d, 2, 3, 20, 50, capacity=7)
    assert st2["overflow"] == 1 and st2["n_clusters"] == st["n_clusters"] and len(part) == 7
    assert part.tobytes() == full[:7].tobytes()


def test_plane_range_run_is_slice_of_full_run():
    rng = np.random.default_rng(29)
    d = frame(rng)
    full, _ = orc.run(d, 2, 3, 20, 50)
    part, st = orc.run(d, 2, 3, 20, 50, planes=(2, 5))
    pl = full["sector"].astype(int) * 3 + full["row"].astype(int)
    assert part.tobytes() == full[(pl >= 2) & (pl < 5)].tobytes()


def test_plane_range_bad_digit_attribution_hand_example():
    """tpc_cf_oracle_run_planes on a partial plane range: which invalid digits (R11) it counts.  Hand example on a
    2-sector x 3-row x 20-pad x 50-bin geometry (planes 0..5 = sector * 3 + row), run on planes [2, 5):
      inside the range, invalid  : (0,2,p=20,t=1,q=5) pad out of range   -> plane 2, counted
                                   (1,0,p=3,t=50,q=5) time out of range  -> plane 3, counted
                                   (1,1,p=3,t=7,q=0)  zero charge        -> plane 4, counted
      outside the range, invalid : (0,0,p=25,t=1,q=5)                    -> plane 0, NOT counted
                                   (1,2,p=3,t=60,q=5)                    -> plane 5, NOT counted
      unattributable             : (2,0,..) sector out of range, (0,3,..) row out of range -> charged to the first
                                   plane of whatever range is asked (plane 2 here): counted by every range, once by
                                   the full-frame run (so counts of ranges that tile a frame need not add up)
      valid digits               : one in plane 1 (outside), one in plane 3 (inside: a single-cell cluster)
    Expected for planes [2,5): n_bad = 3 + 2 = 5, n_digits_used = 1, n_clusters = 1 (the plane-3 digit).
    Expected for the full frame: n_bad = 7, n_digits_used = 2, n_clusters = 2."""
    rows = [(0, 2, 20, 1, 5), (1, 0, 3, 50, 5), (1, 1, 3, 7, 0), (0, 0, 25, 1, 5), (1, 2, 3, 60, 5),
            (2, 0, 1, 1, 5), (0, 3, 1, 1, 5), (0, 1, 4, 4, 9), (1, 0, 6, 6, 9)]
    d = np.zeros(len(rows), dtype=orc.DIGIT)
    for i, (s, r, p, t, q) in enumerate(rows):
        d[i] = (s, r, p, 0, t, q)
    part, st = orc.run(d, 2, 3, 20, 50, planes=(2, 5))
    assert (st["n_bad_digits"], st["n_digits_used"], st["n_clusters"]) == (5, 1, 1)
    assert (int(part[0]["sector"]), int(part[0]["row"]), int(part[0]["pad"]), int(part[0]["time"])) == (1, 0, 6, 6)
    full, sf = orc.run(d, 2, 3, 20, 50)
    assert (sf["n_bad_digits"], sf["n_digits_used"], sf["n_clusters"]) == (7, 2, 2)
    # another range: its own invalid digit (plane 0) plus, again, the two unattributable ones
    a, sa = orc.run(d, 2, 3, 20, 50, planes=(0, 2))
    assert (sa["n_bad_digits"], sa["n_digits_used"], sa["n_clusters"]) == (1 + 2, 1, 1)


def test_dense_plane_matches_digits():
    rng = np.random.default_rng(31)
    a = random_plane(rng, 20, 50, 0.2)
    d = np.concatenate([plane_to_digits(a, 1, 2), plane_to_digits(random_plane(rng, 20, 50, 0.2), 0, 0)])
    assert np.array_equal(orc.dense_plane(d, 2, 3, 20, 50, 1, 2), a)
