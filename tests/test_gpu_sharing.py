"""GPU parity of CHARGE SHARING between overlapping clusters (variant V4, include/tpc_cf.h; SURVEY.md §8(f) NEXT #1
second half): the K6 post-pass behind every CUDA path against the oracle with the same switch — hand examples, frame
slices with and without the other variants, random geometries in every route, full frames, the host pipeline."""
import numpy as np
import pytest

from datagen import gen
from oracle import oracle as orc
from parity import assert_clusters_equal
from test_gpu_parity import (EXPECT_PATH, PATHS, TUNING, _cf, _fused_kernel_tuning, gpu_run,  # noqa: F401 (fixture)
                             sort_digits)

pytestmark = pytest.mark.gpu

SHARE = 32


@pytest.mark.parametrize("path", list(PATHS))
def test_sharing_worked_examples(path):
    """tests/golden/sharing_examples.txt (S1..S7, hand-evaluated) through every CUDA path."""
    import test_oracle_sharing as ts
    for ex in ts.EXAMPLES:
        kw = ts.share_kwargs(ex["v"])
        digits = sort_digits(orc.make_digits(ex["digits"]))
        geom = (1, 1, 12, 12, None)
        ora, ost = orc.run(digits, *geom[:4], **kw)
        cl, st = gpu_run(digits, geom, PATHS[path] | kw["flags"], q_tot_min=kw["q_tot_min"],
                         q_saturation=kw["q_saturation"])
        assert st["n_clusters"] == ost["n_clusters"] == len(ex["clusters"]), ex["name"]
        assert_clusters_equal(cl, ora, "sharing %s/%s" % (ex["name"], path))
        assert [(int(c["qtot"]), int(c["flags"])) for c in cl] == [(c[3], c[9]) for c in ex["clusters"]], ex["name"]


def test_all_examples_on_distinct_rows_at_once():
    """The same examples side by side on the rows of one sector (neighbour search across line ends, planes apart)."""
    import test_oracle_sharing as ts
    ex = [e for e in ts.EXAMPLES if e["v"] == (0, 0, 0, 0)]
    digits = sort_digits(np.concatenate([orc.make_digits(e["digits"], sector=0, row=i) for i, e in enumerate(ex)]))
    geom = (1, len(ex), 12, 12, None)
    ora, ost = orc.run(digits, *geom[:4], flags=SHARE | 4)
    for path in ("fused", "sorted_on_device", "general"):
        cl, st = gpu_run(digits, geom, PATHS[path] | SHARE | 4, tuning={})
        assert_clusters_equal(cl, ora, "sharing examples at once/" + path)
    assert [int(c["qtot"]) for c in ora] == [c[3] for e in ex for c in e["clusters"]]


SHARE_VARIANTS = [dict(vflags=SHARE, q_tot_min=0, q_saturation=0), dict(vflags=SHARE | 4, q_tot_min=0, q_saturation=150),
                  dict(vflags=SHARE | 4 | 8, q_tot_min=25, q_saturation=90)]


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("v", SHARE_VARIANTS, ids=["share", "share+flags", "share+flags+cuts"])
def test_sharing_full_parity(v, path):
    """Config 1, a 10 % occupancy slice with 30 % close pairs (config 4, 3 rows) and a variable-pads slice of config 5:
    every cluster against the oracle, qtot and flags bit-exact; clusters removed by a cut claim nothing."""
    cases = [(gen.generate(1), gen.geometry(1))]
    c = dict(gen.CONFIGS[4]); c["n_sectors"] = 1; c["n_rows"] = 3
    cases.append((gen.generate(c), gen.geometry(c)))
    c = dict(gen.CONFIGS[5]); c["n_sectors"] = 1; c["n_rows"] = 6
    c["npads"] = gen.npads_linear(152, 66, 138)[::30][:6]
    cases.append((gen.generate(c), gen.geometry(c)))
    n_shared = 0
    for digits, geom in cases:
        ora, ost = orc.run(digits, *geom[:4], npads=geom[4], flags=v["vflags"], q_tot_min=v["q_tot_min"],
                           q_saturation=v["q_saturation"])
        base, _ = orc.run(digits, *geom[:4], npads=geom[4], flags=v["vflags"] & ~SHARE, q_tot_min=v["q_tot_min"],
                          q_saturation=v["q_saturation"])
        cl, st = gpu_run(digits, geom, PATHS[path] | v["vflags"], q_tot_min=v["q_tot_min"],
                         q_saturation=v["q_saturation"], max_clusters=ost["n_clusters"] + 16)
        assert st["n_clusters"] == ost["n_clusters"]
        assert_clusters_equal(cl, ora, "sharing %r/%s" % (v, path))
        n_shared += int(np.count_nonzero(ora["qtot"] != base["qtot"]))
    assert n_shared > 1000                                       # the switch did something on these inputs


@pytest.mark.parametrize("seed", list(range(8)))
def test_sharing_random_geometries_every_route(seed):
    """Random geometry, dense random clusters (many overlapping windows, charges up to 65535), random order for the
    routes that take any order; sharing + flags in every route against the oracle."""
    rng = np.random.default_rng(2000 + seed)
    n_sectors, n_rows = int(rng.integers(1, 3)), int(rng.integers(1, 5))
    max_pads = int(rng.integers(3, 30))
    n_time = int(rng.choice([17, 64, 100, 513, 2000]))
    npads = rng.integers(max(1, max_pads // 2), max_pads + 1, size=n_rows).astype(np.uint16)
    npads[int(rng.integers(0, n_rows))] = max_pads
    cells = {}
    for s in range(n_sectors):
        for r in range(n_rows):
            for _ in range(int(rng.integers(1, 2 + max(1, int(npads[r]) * n_time // 25)))):
                p0, t0 = int(rng.integers(0, npads[r])), int(rng.integers(0, n_time))
                for dp in range(-1, 2):
                    for dt in range(-2, 3):
                        p, t = p0 + dp, t0 + dt
                        if 0 <= p < npads[r] and 0 <= t < n_time and rng.random() < 0.7:
                            cells[(s, r, p, t)] = int(rng.choice([1, 2, 3, 4, 5, 7, 20, 300, 65535]))
    digits = np.array([(s, r, p, 0, t, q) for (s, r, p, t), q in cells.items()], dtype=orc.DIGIT)
    geom = (n_sectors, n_rows, max_pads, n_time, npads)
    ora, ost = orc.run(digits, *geom[:4], npads=npads, flags=SHARE | 4)
    assert np.count_nonzero(ora["flags"] & 32) > 0
    srt = sort_digits(digits)
    shuffled = digits[rng.permutation(digits.shape[0])]
    for route, data in (("sorted_on_device", shuffled), ("general", shuffled), ("fused", srt), ("fused_pairs", srt),
                        ("fused_blocks", srt), ("fused_lines", srt), ("general_hint", srt)):
        cl, st = gpu_run(data, geom, PATHS[route] | SHARE | 4, tuning=TUNING.get(route, {}))
        assert st["path"] == EXPECT_PATH.get(route, 3), (route, st)
        assert st["n_clusters"] == ost["n_clusters"], (route, st, ost)
        assert_clusters_equal(cl, ora, "sharing random geometry %d/%s" % (seed, route))


def _full_frame_sharing(cfg_id, sectors=None, shuffle=False, flags=SHARE | 4):
    import torch
    cf = _cf()
    c = dict(gen.CONFIGS[cfg_id])
    if sectors is not None:
        c["n_sectors"] = sectors
    geom = gen.geometry(c)
    digits = gen.generate(c)
    n = digits.shape[0]
    ora, ost, _ = orc.run_parallel(digits, *geom[:4], npads=geom[4], flags=flags)
    f = cf.ClusterFinder(*geom[:4], npads=geom[4], max_digits=n, max_clusters=ost["n_clusters"] + 1024)
    d = cf.to_device(digits)
    if shuffle:
        g = torch.Generator(device="cuda:0")
        g.manual_seed(cfg_id)
        d = d.view(torch.int64)[torch.randperm(n, device="cuda:0", generator=g)].contiguous().view(torch.uint8)
    f.run(d, n, flags=flags | (0 if shuffle else cf.DIGITS_SORTED))
    cl, st = f.result()
    assert st["path"] == (2 if shuffle else 3) and st["overflow"] == 0 and st["n_clusters"] == ost["n_clusters"]
    assert_clusters_equal(cl, ora, "config %d with charge sharing" % cfg_id)
    shared = int(np.count_nonzero(ora["flags"] & 32))
    f.close()
    return ora.shape[0], shared


def test_config3_full_frame_with_sharing():
    """BASELINE.json configs[2] at full size with V4: all 5472 planes, every cluster against the oracle."""
    total, shared = _full_frame_sharing(3)
    assert total > 10_000_000 and shared > 100_000


def test_config4_eight_sectors_with_sharing():
    """configs[3] (10 % occupancy, 30 % close pairs — the workload that exposes double counting) at 8 sectors."""
    total, shared = _full_frame_sharing(4, sectors=8)
    assert total > 10_000_000 and shared > 0.2 * total


def test_config3_shuffled_full_frame_with_sharing():
    """Any-order input: digit sort + fused path + K6 on the sorted copy in the workspace."""
    total, shared = _full_frame_sharing(3, shuffle=True)
    assert total > 10_000_000


def test_run_host_pipelined_with_sharing():
    """tpc_cf_run_host cuts a sorted frame at sector boundaries and runs the groups back to back on one workspace: K6
    runs inside every group (planes never span groups)."""
    cf = _cf()
    c = dict(gen.CONFIGS[4]); c["n_sectors"] = 4; c["n_rows"] = 40
    geom = gen.geometry(c)
    digits = gen.generate(c)
    assert digits.shape[0] >= 1 << 22
    ora, ost, _ = orc.run_parallel(digits, *geom[:4], flags=SHARE | 4)
    f = cf.ClusterFinder(*geom[:4], max_digits=digits.shape[0], max_clusters=ost["n_clusters"] + 4096)
    cl, st = f.run_host(digits, flags=cf.DIGITS_SORTED | SHARE | 4)
    assert st["n_clusters"] == ost["n_clusters"]
    assert_clusters_equal(cl, ora, "run_host pipelined with sharing")
    f.close()


def test_capacity_overflow_with_sharing_reports_and_does_not_crash():
    digits, geom = gen.generate(1), gen.geometry(1)
    ora, ost = orc.run(digits, *geom[:4], flags=SHARE)
    for path in ("fused", "sorted_on_device", "general"):
        cl, st = gpu_run(digits, geom, PATHS[path] | SHARE, capacity=100, tuning={})
        assert st["overflow"] == 1 and st["n_clusters"] == ost["n_clusters"]
        # records far from the cut have all their neighbours: identical to the full run
        assert_clusters_equal(cl[:50], ora[:50], "overflow with sharing/" + path)


@pytest.mark.parametrize("path", ["fused", "sorted_on_device", "general"])
def test_sharing_at_the_limits_of_the_geometry(path):
    """The largest plane the record fields allow (255 pads x 65535 time bins: the digit searches of K6 run on 16-bit
    times up to 65534 and the fused path there is k_fused_blocks), tiny planes (fewer pads / time bins than a 5x5 window
    and than the +-4 neighbour search), and overlapping clusters pressed into the corners."""
    rng = np.random.default_rng(77)
    for (P, T, ncl) in ((255, 65535, 3000), (3, 4, 3), (2, 300, 20), (200, 3, 30), (1, 1, 1), (9, 257, 60)):
        cells = {}
        for _ in range(ncl):
            p0, t0 = int(rng.integers(0, P)), int(rng.integers(0, T))
            for (a, b) in ((0, 0), (0, 3), (2, 1)):                 # three peaks whose windows overlap
                for dp in range(-1, 2):
                    for dt in range(-1, 2):
                        p, t = p0 + a + dp, t0 + b + dt
                        if 0 <= p < P and 0 <= t < T and rng.random() < 0.8:
                            cells[(p, t)] = int(rng.integers(1, 400))
        for p, t in ((P - 1, T - 1), (0, 0), (0, T - 1), (P - 1, 0)):
            cells[(p, t)] = int(rng.integers(4, 65535))
        digits = sort_digits(orc.make_digits([(p, t, q) for (p, t), q in cells.items()]))
        geom = (1, 1, P, T, None)
        ora, ost = orc.run(digits, *geom[:4], flags=SHARE | 4)
        data = digits if PATHS[path] & 1 else digits[rng.permutation(digits.shape[0])]
        cl, st = gpu_run(data, geom, PATHS[path] | SHARE | 4, max_clusters=ost["n_clusters"] + 8, tuning={})
        assert st["n_clusters"] == ost["n_clusters"]
        assert_clusters_equal(cl, ora, "sharing at the limits %dx%d/%s" % (P, T, path))
