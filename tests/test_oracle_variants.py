"""CPU pins of the oracle's VARIANTS (per-cluster flags V1, cuts V2/V3).
Pinned by hand-evaluated grids (tests/golden/variant_examples.txt), by the brute-force checker's independent
formulation (tests/brute.py), and by properties: flags off => byte 0 and nothing else changes; a cut is exactly a
filter of the uncut output by the uncut output's own fields; the base definition is the variant with all knobs 0."""
import os

import numpy as np
import pytest

import brute
from oracle import oracle as orc

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "variant_examples.txt")


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


def variant_kwargs(v):
    q_tot_min, q_sat, csp, cst = v
    return dict(flags=orc.CLUSTER_FLAGS | (orc.CUT_SINGLE_PAD if csp else 0) | (orc.CUT_SINGLE_TIME if cst else 0),
                q_tot_min=q_tot_min, q_saturation=q_sat)


def check(clusters, expected):
    assert len(clusters) == len(expected)
    for c, e in zip(clusters, expected):
        p, t, qmax, S0, S1p, S1t, S2p, S2t, fl = e
        assert (int(c["pad"]), int(c["time"]), int(c["qmax"]), int(c["qtot"]), int(c["flags"])) == (p, t, qmax, S0, fl)
        pm, tm, sp, stime = brute.moments_from_sums(p, t, S0, S1p, S1t, S2p, S2t)
        for got, want in ((c["pad_mean"], pm), (c["time_mean"], tm), (c["sigma_pad"], sp), (c["sigma_time"], stime)):
            w32 = np.float32(want)
            assert abs(float(got) - float(w32)) <= float(np.spacing(w32)), (got, want)


def test_golden_file_lists_the_variant_examples():
    assert [e["name"].split("_")[0] for e in EXAMPLES] == ["V1", "V2", "V3", "V4a", "V4b", "V4c", "V5", "V6a", "V6b",
                                                            "V7", "V8", "V8b", "V9", "V10"]


@pytest.mark.parametrize("ex", EXAMPLES, ids=[e["name"] for e in EXAMPLES])
def test_variant_worked_example(ex):
    d = orc.make_digits(ex["digits"])
    cl, st = orc.run(d, 1, 1, 12, 12, **variant_kwargs(ex["v"]))
    assert st["n_clusters"] == len(ex["clusters"])
    check(cl, ex["clusters"])


@pytest.mark.parametrize("ex", EXAMPLES, ids=[e["name"] for e in EXAMPLES])
def test_variant_worked_example_by_brute_force(ex):
    """The hand-derived lines agree with the brute-force formulation too (guards the golden file itself)."""
    cells = {(p, t): q for p, t, q in ex["digits"]}
    q_tot_min, q_sat, csp, cst = ex["v"]
    got = brute.find_clusters_variants(cells, 12, 12, 4, 2, q_tot_min, q_sat, bool(csp), bool(cst))
    assert got == ex["clusters"]


@pytest.mark.parametrize("seed", range(6))
def test_variants_random_tiny_grids_against_brute_force(seed):
    rng = np.random.default_rng(100 + seed)
    P, T = int(rng.integers(3, 9)), int(rng.integers(3, 9))
    for _ in range(60):
        m = rng.random((P, T)) < rng.choice([0.15, 0.4, 0.8])
        cells = {(int(p), int(t)): int(rng.choice([1, 2, 3, 4, 5, 7, 9, 30])) for p, t in zip(*np.nonzero(m))}
        q_tot_min = int(rng.choice([0, 5, 12, 40]))
        q_sat = int(rng.choice([0, 9, 30]))
        csp, cst = bool(rng.integers(0, 2)), bool(rng.integers(0, 2))
        want = brute.find_clusters_variants(cells, P, T, 4, 2, q_tot_min, q_sat, csp, cst)
        d = orc.make_digits([(p, t, q) for (p, t), q in cells.items()])
        cl, st = orc.run(d, 1, 1, P, T, **variant_kwargs((q_tot_min, q_sat, csp, cst)))
        assert st["n_clusters"] == len(want)
        got = [(int(c["pad"]), int(c["time"]), int(c["qmax"]), int(c["qtot"]), int(c["flags"])) for c in cl]
        assert got == [(w[0], w[1], w[2], w[3], w[8]) for w in want]


def _frame():
    from datagen import gen
    c = dict(gen.CONFIGS[4]); c["n_sectors"] = 1; c["n_rows"] = 3; c["n_time"] = 2048
    return gen.generate(c), gen.geometry(c)


def test_flags_off_is_the_base_definition_and_cut_is_a_filter():
    digits, geom = _frame()
    base, bst = orc.run(digits, *geom[:4])
    assert np.all(base["flags"] == 0)
    full, fst = orc.run(digits, *geom[:4], flags=orc.CLUSTER_FLAGS, q_saturation=200)
    assert fst["n_clusters"] == bst["n_clusters"]
    stripped = full.copy(); stripped["flags"] = 0
    assert np.array_equal(stripped.view(np.uint8), base.view(np.uint8)), "flags must not change anything else"
    fl = full["flags"]
    assert (fl & orc.F_SATURATED).astype(bool).tolist() == (full["qmax"] >= 200).tolist()
    assert np.all(((fl & orc.F_SINGLE_PAD) != 0) == (full["sigma_pad"] == 0))       # S2p == 0  <=>  sigma_pad == 0
    assert np.all(((fl & orc.F_SINGLE_TIME) != 0) == (full["sigma_time"] == 0))
    P, T = geom[2], geom[3]
    assert np.all(((fl & orc.F_EDGE_PAD) != 0) == ((full["pad"] < 2) | (full["pad"].astype(int) + 2 >= P)))
    assert np.all(((fl & orc.F_EDGE_TIME) != 0) == ((full["time"] < 2) | (full["time"].astype(int) + 2 >= T)))
    assert 0 < np.count_nonzero(fl & orc.F_SINGLE_PAD) < len(fl) and np.count_nonzero(fl & orc.F_EDGE_TIME) > 0
    for q_tot_min, cuts in ((60, 0), (0, orc.CUT_SINGLE_PAD), (25, orc.CUT_SINGLE_PAD | orc.CUT_SINGLE_TIME)):
        cut, cst = orc.run(digits, *geom[:4], flags=orc.CLUSTER_FLAGS | cuts, q_tot_min=q_tot_min, q_saturation=200)
        keep = full["qtot"] >= q_tot_min
        if cuts & orc.CUT_SINGLE_PAD:
            keep &= (fl & orc.F_SINGLE_PAD) == 0
        if cuts & orc.CUT_SINGLE_TIME:
            keep &= (fl & orc.F_SINGLE_TIME) == 0
        assert cst["n_clusters"] == int(keep.sum()) < fst["n_clusters"]
        assert np.array_equal(cut.view(np.uint8), full[keep].view(np.uint8))
        # V1 and V2 are independent: without the flags request the same clusters come out with a zero flags byte
        cut0, _ = orc.run(digits, *geom[:4], flags=cuts, q_tot_min=q_tot_min)
        z = cut.copy(); z["flags"] = 0
        assert np.array_equal(cut0.view(np.uint8), z.view(np.uint8))


def test_cut_counts_against_capacity_like_the_base():
    digits, geom = _frame()
    full, fst = orc.run(digits, *geom[:4], q_tot_min=60)
    part, pst = orc.run(digits, *geom[:4], q_tot_min=60, capacity=10)
    assert pst["n_clusters"] == fst["n_clusters"] and pst["overflow"] == 1
    assert np.array_equal(part.view(np.uint8), full[:10].view(np.uint8))
