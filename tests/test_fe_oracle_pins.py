"""Pins of the front-end filter ORACLE (oracle/tpc_fe_oracle.c, TPC-FE v1; step named in PAPER.md:57) against things
other than itself: hand-evaluated values, the identity on generated digits, a numpy special case, the exact geometric
decay of an impulse, an independent Python restatement on random inputs, invariants.  CPU only."""
import os

import numpy as np
import pytest

from datagen import gen
from oracle import fe_oracle as feo
import fe_brute

HERE = os.path.dirname(os.path.abspath(__file__))
OFF = dict(cm_min_pads=60000, it_kappa_shift=0)      # no common-mode correction, no ion-tail cancellation


def tuples(d):
    return [(int(a["sector"]), int(a["row"]), int(a["pad"]), int(a["time"]), int(a["charge"])) for a in d]


def golden():
    ex = {}
    with open(os.path.join(HERE, "golden", "fe_examples.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, p, t, q = line.split()
            ex.setdefault(k, []).append((0, 0, int(p), int(t), int(q)))
    return ex


def example_input():
    raw = np.full((1, 4, 8), 0xFFFF, dtype=np.uint16)
    raw[0, :, :3] = [[10, 10, 30], [8, 9, 12], [10, 10, 10], [10, 12, 9]]
    ped4 = np.full((1, 8), 0xFFFF, dtype=np.uint16)
    ped4[0, :3] = [40, 41, 38]
    return raw, ped4


A = dict(zs_threshold=2, cm_quiet4=8, cm_min_pads=2, it_decay_shift=1, it_kappa_shift=2)


@pytest.mark.parametrize("name,over", [("A", {}), ("B", {"it_kappa_shift": 0}), ("C", {"cm_min_pads": 3}),
                                       ("D", {"zs_threshold": 1})])
def test_hand_evaluated_examples(name, over):
    raw, ped4 = example_input()
    prm = dict(A)
    prm.update(over)
    out, st = feo.run(raw, ped4, 1, 1, 3, 4, **prm)
    assert tuples(out) == golden()[name]
    assert st == {"n_digits": len(golden()[name]), "overflow": 0}
    assert fe_brute.run(raw, ped4, 1, 1, 3, 4, **prm) == golden()[name]      # the checker reads the text the same way


@pytest.mark.parametrize("linear", [False, True])
def test_identity_on_generated_digits(linear):
    """raw = integer pedestal + charge + a common integer shift per time bin, no tail: the filter must return exactly
    the digits it was built from (pins the layout, the pedestal, the quiet-pad mean, the rounding, the threshold, the
    pad range of every row and the output order at once)."""
    c = dict(gen.CONFIGS[1])
    if linear:
        c["npads"] = "linear"
    ns, nr, mp, nt, npads = gen.geometry(c)
    d = gen.generate(c)
    d = d[d["charge"] >= 3]
    W = feo.pad_stride(mp)
    rng = np.random.default_rng(5)
    ped = rng.integers(40, 90, size=(ns * nr, W)).astype(np.int64)
    shift = rng.integers(-1, 2, size=(ns * nr, nt)).astype(np.int64)
    raw = ped[:, None, :] + shift[:, :, None]
    pl = d["sector"].astype(np.int64) * nr + d["row"]
    raw[pl, d["time"], d["pad"]] += d["charge"]
    if npads is not None:                                  # poison what lies beyond the row's pads
        for r in range(nr):
            raw[r::nr, :, int(npads[r]):] = 0xFFFF
    out, st = feo.run(raw.astype(np.uint16), (4 * ped).astype(np.uint16), ns, nr, mp, nt, npads=npads,
                      zs_threshold=2, cm_quiet4=4, cm_min_pads=8, it_decay_shift=6, it_kappa_shift=0)
    assert st["n_digits"] == d.shape[0]
    assert out.tobytes() == d.tobytes()


def test_special_case_without_cm_and_it_is_one_numpy_expression():
    rng = np.random.default_rng(11)
    ns, nr, mp, nt = 2, 3, 13, 50
    W = feo.pad_stride(mp)
    raw = rng.integers(0, 200, size=(ns * nr, nt, W)).astype(np.uint16)
    ped4 = rng.integers(200, 500, size=(ns * nr, W)).astype(np.uint16)
    thr = 7
    out, st = feo.run(raw, ped4, ns, nr, mp, nt, zs_threshold=thr, **OFF)
    q = np.floor((4.0 * raw[:, :, :mp] - ped4[:, None, :mp] + 2.0) / 4.0).astype(np.int64)
    qt = np.transpose(q, (0, 2, 1))                      # [plane, pad, time]: the output order
    pl, p, t = np.nonzero(qt >= thr)
    assert st["n_digits"] == pl.size
    assert np.array_equal(out["sector"], pl // nr) and np.array_equal(out["row"], pl % nr)
    assert np.array_equal(out["pad"], p) and np.array_equal(out["time"], t) and np.array_equal(out["charge"], qt[pl, p, t])


def test_common_mode_is_the_rounded_mean_over_quiet_pads():
    """one time bin, CM on: every pad's output moves by the exactly rounded mean of the quiet pads (Fractions)"""
    from fractions import Fraction
    import math
    rng = np.random.default_rng(3)
    for _ in range(50):
        P = int(rng.integers(3, 30))
        W = feo.pad_stride(P)
        x = rng.integers(-20, 21, size=P)
        big = rng.random(P) < 0.3
        x[big] = rng.integers(100, 400, size=int(big.sum()))
        ped4 = np.full((1, W), 400, dtype=np.uint16)
        rawv = np.full(P, 200, dtype=np.int64)             # x = 4 raw - ped4: reach every x through the pedestal
        ped4[0, :P] = (4 * rawv - x).astype(np.uint16)
        raw = np.zeros((1, 1, W), dtype=np.uint16)
        raw[0, 0, :P] = rawv
        c, m = 12, 2
        quiet = np.abs(x) <= c
        cm = math.floor(Fraction(int(x[quiet].sum()), int(quiet.sum())) + Fraction(1, 2)) if quiet.sum() >= m else 0
        want = [(0, 0, p, 0, (int(x[p]) - cm + 2) // 4) for p in range(P) if (int(x[p]) - cm + 2) // 4 >= 1]
        out, _ = feo.run(raw, ped4, 1, 1, P, 1, zs_threshold=1, cm_quiet4=c, cm_min_pads=m, it_decay_shift=3,
                         it_kappa_shift=0)
        assert tuples(out) == want


def test_impulse_tail_decays_geometrically():
    """k = 2, j = 2: a kept charge of 1024 leaves S = 2^22 for the next bin (a tail of 1024 quarter counts = the
    charge / 4), which then shrinks by exactly 3/4 per bin while it stays divisible; pad p carries a second sample
    n = p + 1 bins later whose charge must come out raised by floor(2^22 (3/4)^(n-1) / 4096) quarter counts."""
    P, T = 10, 16
    W = feo.pad_stride(P)
    ped4 = np.full((1, W), 400, dtype=np.uint16)
    raw = np.full((1, T, W), 100, dtype=np.uint16)
    raw[0, 2, :P] = 100 + 1024
    A2 = 600
    for p in range(P):
        raw[0, 2 + p + 1, p] = 100 + A2
    prm = dict(zs_threshold=500, cm_quiet4=12, cm_min_pads=60000, it_decay_shift=2)
    out, _ = feo.run(raw, ped4, 1, 1, P, T, it_kappa_shift=2, **prm)
    want = []
    for p in range(P):
        n = p + 1
        assert (2 ** 22 * 3 ** (n - 1)) % 4 ** (n - 1) == 0        # the state itself is still exact
        tail = (2 ** 22 * 3 ** (n - 1)) // 4 ** (n - 1) // 4096
        want += [(0, 0, p, 2, 1024), (0, 0, p, 2 + n, (4 * A2 + tail + 2) // 4)]
    assert tuples(out) == want
    # and without cancellation the second sample comes out unchanged
    out0, _ = feo.run(raw, ped4, 1, 1, P, T, it_kappa_shift=0, **prm)
    assert [t[4] for t in tuples(out0)] == [1024, A2] * P


@pytest.mark.parametrize("seed", range(8))
def test_against_the_independent_python_restatement(seed):
    rng = np.random.default_rng(100 + seed)
    ns, nr = int(rng.integers(1, 3)), int(rng.integers(1, 4))
    mp = int(rng.integers(1, 21))
    nt = int(rng.integers(1, 60))
    W = feo.pad_stride(mp)
    npads = rng.integers(1, mp + 1, size=nr).astype(np.uint16) if seed % 2 else None
    ped4 = rng.integers(0, 400, size=(ns * nr, W)).astype(np.uint16)
    base = rng.integers(0, 100, size=(ns * nr, nt, W))
    spikes = (rng.random((ns * nr, nt, W)) < 0.1) * rng.integers(0, 3000, size=(ns * nr, nt, W))
    raw = (base + spikes).astype(np.uint16)
    if seed == 7:
        raw[0, nt // 2:, 0] = 65535                       # saturating charge and the largest tail state
    k = int(rng.integers(1, 8))
    prm = dict(zs_threshold=int(rng.integers(1, 6)), cm_quiet4=int(rng.integers(0, 60)),
               cm_min_pads=int(rng.integers(1, 6)), it_decay_shift=k,
               it_kappa_shift=int(rng.integers(k, 15)) if seed % 3 else 0)
    out, st = feo.run(raw, ped4, ns, nr, mp, nt, npads=npads, **prm)
    want = fe_brute.run(raw, ped4, ns, nr, mp, nt, npads=npads, **prm)
    assert st["n_digits"] == len(want) and tuples(out) == want


def test_invariants_order_independence_of_planes_ignored_pads_capacity():
    rng = np.random.default_rng(9)
    ns, nr, mp, nt = 2, 4, 11, 40
    W = feo.pad_stride(mp)
    npads = np.array([11, 5, 8, 1], dtype=np.uint16)
    ped4 = rng.integers(100, 300, size=(ns * nr, W)).astype(np.uint16)
    raw = (rng.integers(20, 80, size=(ns * nr, nt, W)) + (rng.random((ns * nr, nt, W)) < 0.2) * 500).astype(np.uint16)
    prm = dict(zs_threshold=2, cm_quiet4=40, cm_min_pads=2, it_decay_shift=3, it_kappa_shift=5)
    out, st = feo.run(raw, ped4, ns, nr, mp, nt, npads=npads, **prm)
    key = ((out["sector"].astype(np.int64) * 256 + out["row"]) * 256 + out["pad"]) * 65536 + out["time"]
    assert np.all(np.diff(key) > 0) and np.all(out["rsv"] == 0) and np.all(out["charge"] >= 2)
    assert np.all(out["pad"] < npads[out["row"]])
    # planes are independent: a sub-range gives the slice
    sub, _ = feo.run(raw, ped4, ns, nr, mp, nt, npads=npads, planes=(3, 6), **prm)
    pl = out["sector"].astype(np.int64) * nr + out["row"]
    assert sub.tobytes() == out[(pl >= 3) & (pl < 6)].tobytes()
    # entries beyond the row's pads are never read
    raw2, ped2 = raw.copy(), ped4.copy()
    for r in range(nr):
        raw2[r::nr, :, int(npads[r]):] = 0xFFFF
        ped2[r::nr, int(npads[r]):] = 0
    out2, _ = feo.run(raw2, ped2, ns, nr, mp, nt, npads=npads, **prm)
    assert out2.tobytes() == out.tobytes()
    # capacity: the first records in output order, true count, overflow bit
    cut, st2 = feo.run(raw, ped4, ns, nr, mp, nt, npads=npads, capacity=10, **prm)
    assert st2 == {"n_digits": st["n_digits"], "overflow": 2} and cut.tobytes() == out[:10].tobytes()


def test_parameter_and_geometry_errors():
    raw, ped4 = example_input()
    for bad in (dict(zs_threshold=0), dict(cm_quiet4=4096), dict(cm_min_pads=0), dict(it_decay_shift=0),
                dict(it_decay_shift=16), dict(it_decay_shift=5, it_kappa_shift=4), dict(it_kappa_shift=15)):
        prm = dict(A)
        prm.update(bad)
        with pytest.raises(ValueError):
            feo.run(raw, ped4, 1, 1, 3, 4, **prm)
