"""CPU pins of the oracle's CHARGE SHARING variant (V4; SURVEY.md §8(f) NEXT #1 second half, DESIGN.md §3 V4).
Pinned by hand-evaluated grids (tests/golden/sharing_examples.txt, derivations in DESIGN.md §4 S1..S7), by the
brute-force checker's independent formulation (tests/brute.py: cluster-list enumeration and exact Fractions instead of
a peak-charge map and integer division), and by properties that hold on any input: sharing never changes which
clusters exist nor their position / qmax / flags 1..16; a cluster no other window touches is bit-identical to the
unshared run; no cell hands out more than its charge; the shared run with the flag off is the base definition."""
import os

import numpy as np
import pytest

import brute
from oracle import oracle as orc

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "sharing_examples.txt")


def parse(path=GOLDEN):
    ex, cur = [], None
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        tag, rest = line[0], line[1:].split()
        if tag == "E":
            cur = {"name": rest[0], "digits": [], "clusters": [], "v": (0, 0, 0, 0)}
            ex.append(cur)
        elif tag == "V":
            cur["v"] = tuple(int(x) for x in rest)
        elif tag == "D":
            cur["digits"].append(tuple(int(x) for x in rest))
        elif tag == "C":
            cur["clusters"].append(tuple(int(x) for x in rest))
    return ex


EXAMPLES = parse()


def share_kwargs(v, flags=True):
    q_tot_min, q_sat, csp, cst = v
    return dict(flags=orc.SHARE_CHARGE | (orc.CLUSTER_FLAGS if flags else 0) | (orc.CUT_SINGLE_PAD if csp else 0)
                | (orc.CUT_SINGLE_TIME if cst else 0), q_tot_min=q_tot_min, q_saturation=q_sat)


def check(clusters, expected):
    assert len(clusters) == len(expected)
    for c, e in zip(clusters, expected):
        p, t, qmax, qtot, S0, S1p, S1t, S2p, S2t, fl = e
        assert (int(c["pad"]), int(c["time"]), int(c["qmax"]), int(c["qtot"]), int(c["flags"])) == (p, t, qmax, qtot, fl)
        pm, tm, sp, stime = brute.moments_from_shared_sums(p, t, S0, S1p, S1t, S2p, S2t)
        for got, want in ((c["pad_mean"], pm), (c["time_mean"], tm), (c["sigma_pad"], sp), (c["sigma_time"], stime)):
            w32 = np.float32(want)
            assert abs(float(got) - float(w32)) <= float(np.spacing(w32)), (got, want)


def test_golden_file_lists_the_sharing_examples():
    assert [e["name"].split("_")[0] for e in EXAMPLES] == ["S1", "S2", "S3", "S4", "S5a", "S5b", "S6", "S7"]


@pytest.mark.parametrize("ex", EXAMPLES, ids=[e["name"] for e in EXAMPLES])
def test_sharing_worked_example(ex):
    d = orc.make_digits(ex["digits"])
    cl, st = orc.run(d, 1, 1, 12, 12, **share_kwargs(ex["v"]))
    assert st["n_clusters"] == len(ex["clusters"])
    check(cl, ex["clusters"])


@pytest.mark.parametrize("ex", EXAMPLES, ids=[e["name"] for e in EXAMPLES])
def test_sharing_worked_example_by_brute_force(ex):
    """The hand-derived lines agree with the brute-force formulation too (guards the golden file itself)."""
    cells = {(p, t): q for p, t, q in ex["digits"]}
    q_tot_min, q_sat, csp, cst = ex["v"]
    got = brute.find_clusters_shared(cells, 12, 12, 4, 2, q_tot_min, q_sat, bool(csp), bool(cst))
    assert got == ex["clusters"]


def test_e6_shares_add_up_to_the_charge_that_was_double_counted():
    """R5's example: unshared, both clusters report qtot 41 = all three cells; shared, 23 + 18 = 41."""
    d = orc.make_digits([(5, 7, 20), (5, 8, 6), (5, 9, 15)])
    base, _ = orc.run(d, 1, 1, 12, 12)
    cl, _ = orc.run(d, 1, 1, 12, 12, flags=orc.SHARE_CHARGE)
    assert base["qtot"].tolist() == [41, 41] and cl["qtot"].tolist() == [23, 18]
    assert cl["flags"].tolist() == [0, 0]                         # flags byte only on request


@pytest.mark.parametrize("seed", range(8))
def test_sharing_random_tiny_grids_against_brute_force(seed):
    rng = np.random.default_rng(300 + seed)
    P, T = int(rng.integers(3, 10)), int(rng.integers(3, 10))
    n_shared = 0
    for _ in range(60):
        m = rng.random((P, T)) < rng.choice([0.15, 0.4, 0.8])
        cells = {(int(p), int(t)): int(rng.choice([1, 2, 3, 4, 5, 7, 9, 30, 65535])) for p, t in zip(*np.nonzero(m))}
        q_tot_min = int(rng.choice([0, 0, 12, 40]))
        q_sat = int(rng.choice([0, 9, 30]))
        csp, cst = bool(rng.integers(0, 4) == 0), bool(rng.integers(0, 4) == 0)
        want = brute.find_clusters_shared(cells, P, T, 4, 2, q_tot_min, q_sat, csp, cst)
        d = orc.make_digits([(p, t, q) for (p, t), q in cells.items()])
        cl, st = orc.run(d, 1, 1, P, T, **share_kwargs((q_tot_min, q_sat, csp, cst)))
        assert st["n_clusters"] == len(want)
        check(cl, want)
        n_shared += sum(1 for w in want if w[9] & brute.F_SHARED)
    assert n_shared > 20


def _frame(cfg=4):
    from datagen import gen
    c = dict(gen.CONFIGS[cfg]); c["n_sectors"] = 1; c["n_rows"] = 3; c["n_time"] = 2048
    return gen.generate(c), gen.geometry(c)


def test_sharing_keeps_the_cluster_list_and_touches_only_overlapping_clusters():
    digits, geom = _frame()
    base, bst = orc.run(digits, *geom[:4], flags=orc.CLUSTER_FLAGS, q_saturation=200)
    sh, sst = orc.run(digits, *geom[:4], flags=orc.CLUSTER_FLAGS | orc.SHARE_CHARGE, q_saturation=200)
    assert sst == bst
    for f in ("sector", "row", "pad", "time", "qmax"):
        assert np.array_equal(sh[f], base[f])
    assert np.array_equal(sh["flags"] & 31, base["flags"])
    shared = (sh["flags"] & orc.F_SHARED) != 0
    assert 0.05 < shared.mean() < 0.95                               # config 4: 30 % close pairs
    same = sh.copy(); same["flags"] &= 31
    assert np.array_equal(same[~shared].view(np.uint8), base[~shared].view(np.uint8)), "untouched clusters are bit-identical"
    # a shared cluster gives charge away and never gains any
    assert np.all(sh["qtot"][shared] <= base["qtot"][shared]) and np.any(sh["qtot"][shared] < base["qtot"][shared])
    # SHARED is exactly "another cluster's peak within 4 pads and 4 time bins whose window holds one of my charged
    # cells"; necessary condition checked here: some other peak of the plane within +-4 / +-4
    key = lambda c: (int(c["row"]), int(c["pad"]), int(c["time"]))
    peaks = {}
    for c in sh:
        peaks.setdefault(int(c["row"]), []).append((int(c["pad"]), int(c["time"])))
    for c in sh[shared][:300]:
        r, p, t = key(c)
        assert any((pp, tt) != (p, t) and abs(pp - p) <= 4 and abs(tt - t) <= 4 for pp, tt in peaks[r])
    # without the flags request the same numbers come out with a zero flags byte
    sh0, _ = orc.run(digits, *geom[:4], flags=orc.SHARE_CHARGE, q_saturation=200)
    z = sh.copy(); z["flags"] = 0
    assert np.array_equal(sh0.view(np.uint8), z.view(np.uint8))


def test_no_cell_hands_out_more_than_its_charge():
    """Sum over clusters of qtot (in 1/64 units, from the brute-force sums) never exceeds 64 x the charge in the
    plane, and equals it when every charged cell lies in some window that lets it in (S6's middle cell: 3 x 64)."""
    rng = np.random.default_rng(7)
    for _ in range(40):
        m = rng.random((8, 8)) < 0.5
        cells = {(int(p), int(t)): int(rng.integers(1, 40)) for p, t in zip(*np.nonzero(m))}
        got = brute.find_clusters_shared(cells, 8, 8)
        per_cell = {}
        for (p, t, qmax, *_rest) in got:
            for dp, dt, c in brute.counted_cells(cells, 8, 8, p, t):
                x = (p + dp, t + dt)
                claim = sum(k[2] for k in got if max(abs(k[0] - x[0]), abs(k[1] - x[1])) <= 2)
                per_cell[x] = per_cell.get(x, 0) + (64 * c * qmax) // claim
        for x, s in per_cell.items():
            assert s <= 64 * cells.get(x, 0)
        assert sum(w[4] for w in got) == sum(per_cell.values())


def test_sharing_counts_against_capacity_like_the_base():
    digits, geom = _frame()
    full, fst = orc.run(digits, *geom[:4], flags=orc.SHARE_CHARGE)
    part, pst = orc.run(digits, *geom[:4], flags=orc.SHARE_CHARGE, capacity=10)
    assert pst["n_clusters"] == fst["n_clusters"] and pst["overflow"] == 1
    assert np.array_equal(part.view(np.uint8), full[:10].view(np.uint8))


def test_run_parallel_gives_the_single_thread_result_with_sharing():
    digits, geom = _frame()
    one, st1 = orc.run(digits, *geom[:4], flags=orc.SHARE_CHARGE | orc.CLUSTER_FLAGS)
    par, stp, _ = orc.run_parallel(digits, *geom[:4], n_threads=3, flags=orc.SHARE_CHARGE | orc.CLUSTER_FLAGS)
    assert st1["n_clusters"] == stp["n_clusters"] and np.array_equal(one.view(np.uint8), par.view(np.uint8))
