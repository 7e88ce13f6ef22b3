"""-m gpu parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the same
seeded inputs.  Bar: tests/parity.py.  Paths: "general" (T1, map in HBM, any order) and "fused" (T3, sorted).
Citations: SURVEY.md §8(a) K0..K5, §8(b) boundary, §8(c) readings; definition BASELINE.json:north_star.
"""
import os

import numpy as np
import pytest

from datagen import gen
from oracle import oracle as orc
from parity import assert_clusters_equal, key

pytestmark = pytest.mark.gpu

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "worked_examples.txt")


def _cf():
    import paper_2402_01205_b200 as cf
    return cf


def parse_golden(path=GOLDEN):
    ex, cur = [], None
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        tag, rest = line[0], line[1:].split()
        if tag == "E":
            cur = {"name": rest[0], "digits": []}
            ex.append(cur)
        elif tag == "D":
            cur["digits"].append(tuple(int(x) for x in rest))
    return ex


# flags: DIGITS_SORTED=1, FORCE_GENERAL=2.  "fused" lets the library choose the fused kernel from the mean line length;
# "fused_pairs" / "fused_blocks" / "fused_lines" force one of the three fused kernels (tpc_cf_debug_set), so that each
# runs every case — including the ones far outside its range, which exercise its exact slow paths.
# "*_p3" additionally covers the time axis in 3 passes, the shape long lines get.
# "sorted_on_device": no promise, no FORCE_GENERAL: the library sorts the digits on the device and runs the fused path
# (status.path 2); "general": FORCE_GENERAL without the hint (map in HBM + key sort of the clusters).
PATHS = {"general": 2, "general_hint": 3, "sorted_on_device": 0, "fused": 1, "fused_pairs": 1, "fused_pairs_p3": 1,
         "fused_blocks": 1, "fused_blocks_p3": 1, "fused_lines": 1}
EXPECT_PATH = {"general": 1, "general_hint": 1, "sorted_on_device": 2}
TUNING = {"fused_pairs": dict(fused_kernel="pairs"), "fused_pairs_p3": dict(fused_kernel="pairs", passes=3),
          "fused_blocks": dict(fused_kernel="blocks"), "fused_blocks_p3": dict(fused_kernel="blocks", passes=3),
          "fused_lines": dict(fused_kernel="lines")}
_tuning = {}


@pytest.fixture(autouse=True)
def _fused_kernel_tuning(request):
    """The handle overrides (tpc_cf_debug_set) the test's `path` parameter asks for; gpu_run applies them."""
    params = getattr(getattr(request.node, "callspec", None), "params", {})
    _tuning.clear()
    _tuning.update(TUNING.get(params.get("path"), {}))
    yield
    _tuning.clear()


def gpu_run(digits, geom, flags, max_clusters=None, capacity=None, q_peak_min=4, q_inner_gate=2, finder=None,
            q_tot_min=0, q_saturation=0, tuning=None, expect_kernel=None):
    cf = _cf()
    n_sectors, n_rows, max_pads, n_time, npads = geom
    n = int(digits.shape[0])
    own = finder is None
    if own:
        finder = cf.ClusterFinder(n_sectors, n_rows, max_pads, n_time, npads=npads, max_digits=max(n, 1),
                                  max_clusters=max_clusters if max_clusters is not None else max(n, 1),
                                  q_peak_min=q_peak_min, q_inner_gate=q_inner_gate, q_tot_min=q_tot_min,
                                  q_saturation=q_saturation)
    tun = dict(_tuning) if tuning is None else dict(tuning)
    finder.debug_set(**tun)
    d = cf.to_device(digits)
    finder.run(d, n, flags=flags, capacity=capacity)
    cl, st = finder.result()
    st["kernel"] = finder.last_kernel()
    forced = tun.get("fused_kernel") if expect_kernel is None else expect_kernel
    if forced and n and st["path"] == 3:
        assert st["kernel"] == "k_fused_" + forced, (st["kernel"], forced)
    if capacity is not None:
        cl = cl[:capacity]
    if own:
        finder.close()
    return cl, st


def sort_digits(d):
    k = ((d["sector"].astype(np.uint64) << 32) | (d["row"].astype(np.uint64) << 24) |
         (d["pad"].astype(np.uint64) << 16) | d["time"].astype(np.uint64))
    return d[np.argsort(k, kind="stable")]


@pytest.mark.parametrize("path", list(PATHS))
def test_worked_examples(path):
    """E1..E15 (tests/golden/worked_examples.txt) placed on distinct rows of one 12x12 sector, all at once."""
    ex = parse_golden()
    digits = np.concatenate([orc.make_digits(e["digits"], sector=0, row=i) for i, e in enumerate(ex)])
    geom = (1, len(ex), 12, 12, None)
    if PATHS[path] & 1:
        digits = sort_digits(digits)       # the golden file lists each example's digits in no particular order
    ora, ost = orc.run(digits, *geom[:4])
    cl, st = gpu_run(digits, geom, PATHS[path])
    assert st["n_clusters"] == ost["n_clusters"] and st["n_bad_digits"] == 0 and st["overflow"] == 0
    assert st["path"] == EXPECT_PATH.get(path, 3)
    assert_clusters_equal(cl, ora, "worked examples/" + path)


def test_map_parity_config1():
    """K1 scatter: dense planes equal the oracle's (SURVEY.md §7.2 minimum slice), and the map is clean after."""
    cf = _cf()
    digits = gen.generate(1)
    geom = gen.geometry(1)
    f = cf.ClusterFinder(*geom[:4], max_digits=digits.shape[0])
    d = cf.to_device(digits)
    for row in (0, 1, 77, 151):
        got = f.dense_plane(d, digits.shape[0], 0, row, geom[2])
        want = orc.dense_plane(digits, *geom[:4], 0, row)
        assert np.array_equal(got, want), "plane row %d differs" % row
    empty = f.dense_plane(d, 0, 0, 5, geom[2])
    assert not empty.any(), "map not restored to zero by the un-scatter"
    f.close()


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("cfg", [1, 2])
def test_config_full_parity(cfg, path):
    digits = gen.generate(cfg)
    geom = gen.geometry(cfg)
    ora, ost = orc.run(digits, *geom[:4], npads=geom[4])
    cl, st = gpu_run(digits, geom, PATHS[path], max_clusters=ost["n_clusters"] + 16)
    assert st["n_clusters"] == ost["n_clusters"] and st["n_digits_used"] == ost["n_digits_used"]
    assert_clusters_equal(cl, ora, "config %d/%s" % (cfg, path))


@pytest.mark.parametrize("route", ["sorted_on_device", "general"])
@pytest.mark.parametrize("cfg", [1, 2])
def test_shuffled_input_general(cfg, route):
    """Any-order contract (R12, I1): a random permutation of the digits gives the identical output array — by the
    digit sort + fused path (the default for input without the promise) and by the general path (FORCE_GENERAL)."""
    digits = gen.generate(cfg)
    geom = gen.geometry(cfg)
    ora, ost = orc.run(digits, *geom[:4])
    rng = np.random.default_rng(100 + cfg)
    sh = digits[rng.permutation(digits.shape[0])]
    cl, st = gpu_run(sh, geom, PATHS[route], max_clusters=ost["n_clusters"] + 16)
    assert st["path"] == EXPECT_PATH[route] and st["n_clusters"] == ost["n_clusters"]
    assert_clusters_equal(cl, ora, "config %d shuffled/%s" % (cfg, route))


@pytest.mark.parametrize("flags", [1, 3])
def test_false_sorted_promise_is_detected(flags):
    """include/tpc_cf.h: a false DIGITS_SORTED promise is detected on the device and reported as path 0."""
    digits = gen.generate(1)
    geom = gen.geometry(1)
    sh = digits[np.random.default_rng(7).permutation(digits.shape[0])]
    cl, st = gpu_run(sh, geom, flags)
    assert st["path"] == 0 and st["n_clusters"] == 0


def test_run_host_retries_on_false_promise():
    cf = _cf()
    digits = gen.generate(1)
    geom = gen.geometry(1)
    ora, _ = orc.run(digits, *geom[:4])
    sh = digits[np.random.default_rng(8).permutation(digits.shape[0])]
    f = cf.ClusterFinder(*geom[:4], max_digits=digits.shape[0], max_clusters=ora.shape[0] + 8)
    cl, st = f.run_host(sh, flags=cf.DIGITS_SORTED)
    assert st["path"] == 2                                   # rerun without the promise: digit sort + fused path
    assert_clusters_equal(cl.copy(), ora, "run_host retry")
    cl, st = f.run_host(digits, flags=cf.DIGITS_SORTED)
    assert st["path"] == 3
    assert_clusters_equal(cl.copy(), ora, "run_host sorted")
    f.close()


@pytest.mark.parametrize("path", list(PATHS))
def test_empty_and_single(path):
    geom = (2, 3, 20, 40, None)
    cl, st = gpu_run(np.zeros(0, dtype=orc.DIGIT), geom, PATHS[path])
    assert st["n_clusters"] == 0 and cl.shape[0] == 0 and st["n_bad_digits"] == 0
    one = orc.make_digits([(19, 39, 9)], sector=1, row=2)      # last cell of the last plane
    ora, _ = orc.run(one, *geom[:4])
    cl, st = gpu_run(one, geom, PATHS[path])
    assert_clusters_equal(cl, ora, "single digit/" + path)


@pytest.mark.parametrize("path", list(PATHS))
def test_bad_digits_are_skipped_and_counted(path):
    """R11: out-of-range (sector,row,pad for that row,time) and zero-charge digits are skipped and counted."""
    npads = np.array([10, 12, 16], dtype=np.uint16)
    geom = (2, 3, 16, 64, npads)
    good = [(0, 0, 5, 10, 9), (0, 0, 5, 11, 4), (0, 1, 11, 63, 7), (1, 2, 15, 0, 30), (1, 2, 14, 0, 6)]
    bad = [(0, 0, 10, 5, 50),    # pad 10 does not exist in row 0
           (0, 1, 12, 5, 50),    # pad 12 does not exist in row 1
           (0, 1, 3, 64, 50),    # time out of range
           (1, 1, 3, 3, 0),      # zero charge
           (2, 0, 1, 1, 50),     # sector out of range
           (1, 3, 1, 1, 50)]     # row out of range
    d = np.zeros(len(good) + len(bad), dtype=orc.DIGIT)
    for i, (s, r, p, t, q) in enumerate(good + bad):
        d[i] = (s, r, p, 0, t, q)
    d = sort_digits(d)
    ora, ost = orc.run(d, *geom[:4], npads=npads)
    assert ost["n_bad_digits"] == len(bad)
    cl, st = gpu_run(d, geom, PATHS[path])
    assert st["n_bad_digits"] == len(bad) and st["n_digits_used"] == len(good)
    assert_clusters_equal(cl, ora, "bad digits/" + path)


@pytest.mark.parametrize("path", list(PATHS))
def test_capacity_overflow(path):
    """§8(b): more peaks than capacity => first `capacity` clusters in output order, true count, overflow = 1."""
    digits = gen.generate(1)
    geom = gen.geometry(1)
    ora, ost = orc.run(digits, *geom[:4])
    cap = 1000
    cl, st = gpu_run(digits, geom, PATHS[path], capacity=cap)
    assert st["overflow"] == 1 and st["n_clusters"] == ost["n_clusters"]
    assert_clusters_equal(cl[:cap], ora[:cap], "overflow/" + path)


@pytest.mark.parametrize("path", list(PATHS))
def test_variable_pads_and_back_to_back_frames(path):
    """config 5 at 2 sectors: npads 66->138 (R19), 4 frames enqueued back to back on one stream with one
    workspace (R16): a stale map or stale staging would show up as ghost clusters."""
    cf = _cf()
    import torch
    c = dict(gen.CONFIGS[5]); c["n_sectors"] = 2
    geom = gen.geometry(c)
    frames = [gen.generate(c, frame=f) for f in range(4)]
    nmax = max(f.shape[0] for f in frames)
    finder = cf.ClusterFinder(*geom[:4], npads=geom[4], max_digits=nmax, max_clusters=nmax // 8)
    devs = [cf.to_device(f) for f in frames]
    outs = [torch.empty(finder.max_clusters * 32, dtype=torch.uint8, device="cuda:0") for _ in frames]
    sts = [torch.zeros(32, dtype=torch.uint8, device="cuda:0") for _ in frames]
    for f, d, o, s in zip(frames, devs, outs, sts):
        finder.run(d, f.shape[0], flags=PATHS[path], clusters=o, status=s)
    for i, (f, o, s) in enumerate(zip(frames, outs, sts)):
        cl, st = finder.result(clusters=o, status=s)
        ora, ost = orc.run(f, *geom[:4], npads=geom[4])
        assert st["n_clusters"] == ost["n_clusters"]
        assert_clusters_equal(cl, ora, "config5 frame %d/%s" % (i, path))
    finder.close()


@pytest.mark.parametrize("path", list(PATHS))
def test_dense_pairs_plateaus(path):
    """config 4 at 1 sector: ~10% occupancy, 30% close pairs, flat-top plateaus (R1b, R5)."""
    c = dict(gen.CONFIGS[4]); c["n_sectors"] = 1
    geom = gen.geometry(c)
    digits = gen.generate(c)
    ora, ost = orc.run(digits, *geom[:4])
    cl, st = gpu_run(digits, geom, PATHS[path], max_clusters=ost["n_clusters"] + 16)
    assert st["n_clusters"] == ost["n_clusters"]
    assert_clusters_equal(cl, ora, "config4x1/" + path)


@pytest.mark.parametrize("path", list(PATHS))
def test_thresholds_and_saturated_charges(path):
    """Non-default thresholds and full-range uint16 charges (R13, P5): random 40x60 planes, values up to 65535."""
    rng = np.random.default_rng(11)
    geom = (1, 6, 40, 60, None)
    cells = []
    d = []
    for row in range(6):
        m = rng.random((40, 60)) < (0.05 + 0.15 * row)
        p, t = np.nonzero(m)
        q = rng.choice([1, 2, 3, 4, 5, 9, 200, 65535], size=p.size)
        for a, b, c_ in zip(p, t, q):
            d.append((0, row, a, 0, b, c_))
    digits = sort_digits(np.array(d, dtype=orc.DIGIT))
    for qmin, gate in ((4, 2), (1, 0), (5, 65535), (200, 3)):
        ora, ost = orc.run(digits, *geom[:4], q_peak_min=qmin, q_inner_gate=gate)
        cl, st = gpu_run(digits, geom, PATHS[path], q_peak_min=qmin, q_inner_gate=gate)
        assert_clusters_equal(cl, ora, "thresholds %d/%d %s" % (qmin, gate, path))


def test_full_frame_sampled_planes():
    """BASELINE.json configs[2] at full size (36 sectors, ~2%), in the launch configuration bench.py times (fused
    path, DIGITS_SORTED): cluster count and order checked globally, and the clusters of sampled planes compared
    one by one with the oracle run on exactly those planes."""
    cf = _cf()
    geom = gen.geometry(3)
    digits = gen.generate(3)
    n = digits.shape[0]
    f = cf.ClusterFinder(*geom[:4], max_digits=n, max_clusters=n // 12)
    d = cf.to_device(digits)
    f.run(d, n, flags=cf.DIGITS_SORTED)
    cl, st = f.result()
    assert st["path"] == 3 and st["overflow"] == 0 and st["n_digits_used"] == n
    k = key(cl)
    assert np.all(k[1:] > k[:-1])
    plane_of = cl["sector"].astype(np.int64) * geom[1] + cl["row"]
    dplane = digits["sector"].astype(np.int64) * geom[1] + digits["row"]
    rng = np.random.default_rng(3)
    total = 0
    for pl in [0, geom[0] * geom[1] - 1] + list(rng.integers(0, geom[0] * geom[1], size=22)):
        lo, hi = np.searchsorted(dplane, [pl, pl + 1])
        ora, ost = orc.run(digits[lo:hi], *geom[:4], planes=(int(pl), int(pl) + 1))
        a, b = np.searchsorted(plane_of, [pl, pl + 1])
        assert_clusters_equal(cl[a:b], ora, "config 3 plane %d" % pl)
        total += ora.shape[0]
    assert total > 10000
    # general path on the same frame: identical array
    f.run(d, n, flags=cf.DIGITS_SORTED | cf.FORCE_GENERAL)
    cl2, st2 = f.result()
    assert st2["path"] == 1 and st2["n_clusters"] == st["n_clusters"]
    assert np.array_equal(cl2.view(np.uint8), cl.view(np.uint8)), "general and fused path differ on config 3"
    # variants at full size (flags + q_tot_min cut + single-pad cut): count by filtering the uncut output, sampled
    # planes one by one against the oracle with the same knobs
    f.params.q_tot_min, f.params.q_saturation = 40, 200
    vflags = cf.CLUSTER_FLAGS | cf.CUT_SINGLE_PAD
    f.run(d, n, flags=cf.DIGITS_SORTED | vflags)
    cv, sv = f.result()
    keep = (cl["qtot"] >= 40) & (cl["sigma_pad"] != 0)
    assert sv["n_clusters"] == int(keep.sum()) and np.array_equal(key(cv), key(cl[keep]))
    vplane = cv["sector"].astype(np.int64) * geom[1] + cv["row"]
    for pl in (0, 1234, geom[0] * geom[1] - 1):
        lo, hi = np.searchsorted(dplane, [pl, pl + 1])
        ora, ost = orc.run(digits[lo:hi], *geom[:4], planes=(int(pl), int(pl) + 1), flags=vflags, q_tot_min=40,
                           q_saturation=200)
        a, b = np.searchsorted(vplane, [pl, pl + 1])
        assert_clusters_equal(cv[a:b], ora, "config 3 variants plane %d" % pl)
    f.close()


@pytest.mark.parametrize("path", list(PATHS))
def test_dense_isolated_peaks_overflow_the_peak_queue(path):
    """Degenerate density: a checkerboard-like pattern where every digit is a peak (2048 peaks per pad line) — far
    more than the fused kernel's per-step shared-memory peak queue holds, so its exact slow path is exercised;
    lines longer than the tq capacity of a slot are exercised too (a fully occupied row)."""
    rng = np.random.default_rng(5)
    geom = (1, 3, 12, 4096, None)
    d = []
    for pad in range(0, 12, 2):
        for t in range(pad % 4, 4096, 2):
            d.append((0, 1, pad, 0, t, int(rng.integers(4, 500))))
    for pad in range(12):                      # a fully occupied row: every cell holds charge
        for t in range(0, 4096):
            d.append((0, 2, pad, 0, t, int(rng.integers(1, 60))))
    d.append((0, 0, 3, 0, 7, 9))
    digits = sort_digits(np.array(d, dtype=orc.DIGIT))
    ora, ost = orc.run(digits, *geom[:4])
    assert ost["n_clusters"] > 12000
    cl, st = gpu_run(digits, geom, PATHS[path])
    assert st["n_clusters"] == ost["n_clusters"]
    assert_clusters_equal(cl, ora, "dense isolated peaks/" + path)


@pytest.mark.parametrize("kernel", ["pairs", "blocks"])
@pytest.mark.parametrize("passes", [1, 2, 5])
@pytest.mark.parametrize("pool,scap", [(2, 4), (9, 8), (40, 4), (255, 12)])
def test_block_kernel_slow_paths(pool, scap, passes, kernel):
    """The block-sparse kernels with a block pool / survivor list far too small for the data (tpc_cf_debug_set
    block_pool, surv_cap): window cells whose block is not in the pool are looked up in the digit array, survivors
    beyond the list are re-derived from the digit array.  Results must not change (config 1, and a ~5 % single row)."""
    tun = dict(fused_kernel=kernel, block_pool=pool, surv_cap=scap, passes=passes)
    digits = gen.generate(1)
    geom = gen.geometry(1)
    ora, ost = orc.run(digits, *geom[:4], npads=geom[4])
    cl, st = gpu_run(digits, geom, 1, tuning=tun)
    assert st["kernel"] == "k_fused_" + kernel and st["n_clusters"] == ost["n_clusters"]
    assert_clusters_equal(cl, ora, "config 1, pool %d scap %d" % (pool, scap))
    c = dict(gen.CONFIGS[2]); c["n_rows"] = 2
    geom = gen.geometry(c)
    digits = gen.generate(c)
    ora, ost = orc.run(digits, *geom[:4])
    cl, st = gpu_run(digits, geom, 1, tuning=tun)
    assert st["kernel"] == "k_fused_" + kernel and st["n_clusters"] == ost["n_clusters"]
    assert_clusters_equal(cl, ora, "config 2 (2 rows), pool %d scap %d" % (pool, scap))


def test_run_host_pipelined_over_sector_groups():
    """tpc_cf_run_host on a frame large enough for its sector-group pipeline (config 3 cut to 4 sectors, ~24 M digits):
    same array as one device-resident run and as the oracle on sampled planes; a false promise (two digits swapped
    across sectors) and a capacity too small for a group's share fall back to the single-shot route."""
    import torch
    cf = _cf()
    c = dict(gen.CONFIGS[3]); c["n_sectors"] = 4
    geom = gen.geometry(c)
    digits = gen.generate(c)
    n = digits.shape[0]
    assert n >= (1 << 22)
    f = cf.ClusterFinder(*geom[:4], max_digits=n, max_clusters=n // 12)
    d = cf.to_device(digits)
    f.run(d, n, flags=cf.DIGITS_SORTED)
    ref, rst = f.result()
    ref = ref.copy()
    pinned = torch.from_numpy(digits.view(np.uint8)).pin_memory()
    cl, st = f.run_host(pinned, flags=cf.DIGITS_SORTED)
    assert st["path"] == 3 and st["n_clusters"] == rst["n_clusters"] and st["n_digits_used"] == n
    assert np.array_equal(cl.view(np.uint8), ref.view(np.uint8)), "pipelined run_host differs from the device-resident run"
    dplane = digits["sector"].astype(np.int64) * geom[1] + digits["row"]
    lo, hi = np.searchsorted(dplane, [2 * geom[1], 2 * geom[1] + 3])
    ora, _ = orc.run(digits[lo:hi], *geom[:4], planes=(2 * geom[1], 2 * geom[1] + 3))
    a, b = np.searchsorted(key(cl), [np.uint64(2) << np.uint64(32), (np.uint64(2) << np.uint64(32)) + (np.uint64(3) << np.uint64(24))])
    assert_clusters_equal(cl[a:b].copy(), ora, "pipelined run_host, sector 2 rows 0..2")
    # false promise: swap one digit of sector 0 with one of sector 3
    sw = digits.copy()
    i, j = 12345, n - 54321
    sw[[i, j]] = sw[[j, i]]
    cl2, st2 = f.run_host(sw, flags=cf.DIGITS_SORTED)
    assert st2["path"] == 2 and st2["n_clusters"] == rst["n_clusters"]
    assert np.array_equal(cl2.view(np.uint8), ref.view(np.uint8))
    f.close()
    # capacity that holds the frame but not a proportional share per group is still honoured
    f = cf.ClusterFinder(*geom[:4], max_digits=n, max_clusters=int(rst["n_clusters"]) + 8)
    cl3, st3 = f.run_host(pinned, flags=cf.DIGITS_SORTED)
    assert st3["n_clusters"] == rst["n_clusters"] and st3["overflow"] == 0
    assert np.array_equal(cl3.view(np.uint8), ref.view(np.uint8))
    f.close()


# ---- variants (flags V1, cuts V2/V3) ------------------------------------------------------
VARIANTS = [dict(vflags=4, q_tot_min=0, q_saturation=150), dict(vflags=0, q_tot_min=60, q_saturation=0),
            dict(vflags=4 | 8, q_tot_min=0, q_saturation=0), dict(vflags=4 | 8 | 16, q_tot_min=25, q_saturation=90)]


@pytest.mark.parametrize("path", list(PATHS))
def test_variant_worked_examples(path):
    """tests/golden/variant_examples.txt through every CUDA path, against the oracle with the same knobs."""
    import test_oracle_variants as tv
    for ex in tv.EXAMPLES:
        kw = tv.variant_kwargs(ex["v"])
        digits = sort_digits(orc.make_digits(ex["digits"]))
        geom = (1, 1, 12, 12, None)
        ora, ost = orc.run(digits, *geom[:4], **kw)
        cl, st = gpu_run(digits, geom, PATHS[path] | kw["flags"], q_tot_min=kw["q_tot_min"],
                         q_saturation=kw["q_saturation"])
        assert st["n_clusters"] == ost["n_clusters"] == len(ex["clusters"]), ex["name"]
        assert_clusters_equal(cl, ora, "variant %s/%s" % (ex["name"], path))
        assert [int(f) for f in cl["flags"]] == [c[8] for c in ex["clusters"]], ex["name"]


@pytest.mark.parametrize("path", list(PATHS))
@pytest.mark.parametrize("v", VARIANTS, ids=["flags", "qtot60", "flags+cut_pad", "all"])
def test_variants_full_parity(v, path):
    """Flags and cuts on config 1, on a 10 % frame slice (config 4, 3 rows) and on a variable-pads slice of config 5:
    bit-exact flags, counts and order against the oracle; the cut changes counts and ordinals in every kernel."""
    cases = [(gen.generate(1), gen.geometry(1))]
    c = dict(gen.CONFIGS[4]); c["n_sectors"] = 1; c["n_rows"] = 3
    cases.append((gen.generate(c), gen.geometry(c)))
    c = dict(gen.CONFIGS[5]); c["n_sectors"] = 1; c["n_rows"] = 6
    c["npads"] = gen.npads_linear(152, 66, 138)[::30][:6]
    cases.append((gen.generate(c), gen.geometry(c)))
    for digits, geom in cases:
        ora, ost = orc.run(digits, *geom[:4], npads=geom[4], flags=v["vflags"], q_tot_min=v["q_tot_min"],
                           q_saturation=v["q_saturation"])
        cl, st = gpu_run(digits, geom, PATHS[path] | v["vflags"], q_tot_min=v["q_tot_min"],
                         q_saturation=v["q_saturation"], max_clusters=ost["n_clusters"] + 16)
        assert st["n_clusters"] == ost["n_clusters"]
        assert_clusters_equal(cl, ora, "variants %r/%s" % (v, path))
        assert np.array_equal(cl["flags"], ora["flags"])
        if v["vflags"] & 4:
            assert np.count_nonzero(cl["flags"]) > 0


@pytest.mark.parametrize("path", list(PATHS))
def test_maximum_geometry(path):
    """The largest plane the 8/16-bit record fields allow (255 pads x 65535 time bins), sparse clusters plus digits in
    the last pads and time bins, and odd sizes that are no multiple of the kernels' tile sizes (7 pads x 61 bins).
    The bitmap slots of k_fused_lines do not fit shared memory above ~50 k time bins and k_fused_pairs needs
    n_time < 65470 (its sentinel times): the library then runs k_fused_blocks, which takes any geometry."""
    rng = np.random.default_rng(21)
    for (P, T, ncl) in ((255, 65535, 4000), (255, 65469, 2000), (7, 61, 12), (9, 257, 40)):
        cells = {}
        for _ in range(ncl):
            p0, t0 = int(rng.integers(0, P)), int(rng.integers(0, T))
            for dp in range(-1, 2):
                for dt in range(-2, 3):
                    p, t = p0 + dp, t0 + dt
                    if 0 <= p < P and 0 <= t < T and rng.random() < 0.8:
                        cells[(p, t)] = int(rng.integers(1, 400))
        for p, t in ((P - 1, T - 1), (P - 1, T - 2), (P - 2, T - 1), (0, 0), (0, T - 1), (P - 1, 0)):
            cells[(p, t)] = int(rng.integers(4, 999))
        digits = sort_digits(orc.make_digits([(p, t, q) for (p, t), q in cells.items()]))
        geom = (1, 1, P, T, None)
        ora, ost = orc.run(digits, *geom[:4])
        expect = None
        if T > 65469 and path in ("fused_lines", "fused_pairs", "fused_pairs_p3"):
            expect = "blocks"
        elif T > 40000 and path == "fused_lines":
            expect = "pairs"
        cl, st = gpu_run(digits, geom, PATHS[path], max_clusters=ost["n_clusters"] + 8, expect_kernel=expect)
        assert st["n_clusters"] == ost["n_clusters"] and st["n_bad_digits"] == 0
        assert_clusters_equal(cl, ora, "max geometry %dx%d/%s" % (P, T, path))


# ---- full-size parity in the launch shape bench.py times (every config, every plane) -------------------------
def _full_frame_check(cfg_id, frames=1, sectors=None):
    """All clusters of the full-size config (all planes) against the oracle run on all host cores (the same
    single-threaded routine over plane blocks), element by element; fused path as bench.py launches it.  Frames of a
    multi-frame config are enqueued back to back on one stream with one workspace."""
    import torch
    cf = _cf()
    c = dict(gen.CONFIGS[cfg_id])
    if sectors is not None:
        c["n_sectors"] = sectors
    geom = gen.geometry(c)
    fr = [gen.generate(c, frame=f) for f in range(frames)]
    nmax = max(f.shape[0] for f in fr)
    finder = cf.ClusterFinder(*geom[:4], npads=geom[4], max_digits=nmax, max_clusters=nmax // 10 + 1024)
    devs = [cf.to_device(f) for f in fr]
    outs = [torch.empty(finder.max_clusters * 32, dtype=torch.uint8, device="cuda:0") for _ in fr]
    sts = [torch.zeros(32, dtype=torch.uint8, device="cuda:0") for _ in fr]
    for f, d, o, s in zip(fr, devs, outs, sts):
        finder.run(d, f.shape[0], flags=cf.DIGITS_SORTED, clusters=o, status=s)
    kernel = finder.last_kernel()
    total = 0
    for i, (f, o, s) in enumerate(zip(fr, outs, sts)):
        cl, st = finder.result(clusters=o, status=s)
        assert st["path"] == 3 and st["overflow"] == 0
        ora, ost, nthr = orc.run_parallel(f, *geom[:4], npads=geom[4])
        assert st["n_clusters"] == ost["n_clusters"] and st["n_bad_digits"] == ost["n_bad_digits"] == 0
        assert_clusters_equal(cl, ora, "config %d frame %d, all %d planes (%s)" % (cfg_id, i, geom[0] * geom[1], kernel))
        total += ora.shape[0]
        del cl, ora
    finder.close()
    return total, kernel


def test_config3_full_frame_every_plane():
    """BASELINE.json configs[2]: the whole 36-sector frame, all 5472 planes, 10.9 M clusters compared one by one."""
    total, kernel = _full_frame_check(3)
    assert total > 10_000_000


def test_config4_eight_sectors_every_plane():
    """configs[3] at 8 sectors (1216 planes >= 1184: whole-plane units, several time passes): fully compared."""
    total, kernel = _full_frame_check(4, sectors=8)
    assert total > 10_000_000


def test_config5_eight_sectors_four_frames():
    """configs[4] at 8 sectors, 4 frames back to back (whole-plane units, short lines): fully compared."""
    total, kernel = _full_frame_check(5, frames=4, sectors=8)
    assert total > 1_000_000


def test_config4_full_frame_every_plane():
    """configs[3] at full size: 1.09e9 digits (indices past 2^30, staging offsets past 2^32), 51 M clusters, every
    plane compared with the oracle."""
    total, kernel = _full_frame_check(4)
    assert total > 50_000_000


def test_config5_full_four_frames_every_plane():
    """configs[4] at full size: 36 sectors, pads 66 -> 138, 4 frames back to back on one stream: every cluster."""
    total, kernel = _full_frame_check(5, frames=4)
    assert total > 7_000_000


@pytest.mark.parametrize("path", ["fused_pairs", "fused_blocks", "fused_lines", "general", "sorted_on_device"])
@pytest.mark.parametrize("odd_n", [0, 1])
def test_digit_buffer_eight_bytes_off_a_16_byte_boundary(path, odd_n):
    """The ABI asks for 8-byte aligned digits only: a buffer that starts 8 bytes off a 16-byte boundary (and one whose
    last digit ends 8 bytes off) must give the same clusters — the bulk copies of k_fused_pairs move 16-byte aligned
    pieces and copy the ragged first / last digit of the array by hand."""
    import torch
    cf = _cf()
    digits = gen.generate(1)
    if (digits.shape[0] & 1) != odd_n:
        digits = digits[:-1]
    geom = gen.geometry(1)
    ora, ost = orc.run(digits, *geom[:4])
    n = digits.shape[0]
    finder = cf.ClusterFinder(*geom[:4], max_digits=n, max_clusters=ost["n_clusters"] + 16)
    finder.debug_set(**TUNING.get(path, {}))
    buf = torch.zeros((n + 2) * 8, dtype=torch.uint8, device="cuda:0")
    assert buf.data_ptr() % 16 == 0
    buf[8:8 + n * 8] = torch.from_numpy(digits.view(np.uint8)).cuda()
    finder.run(buf[8:], n, flags=PATHS[path])
    cl, st = finder.result()
    assert st["n_clusters"] == ost["n_clusters"] and st["n_bad_digits"] == 0
    assert_clusters_equal(cl, ora, "misaligned buffer/" + path)
    finder.close()


def test_sharded_cluster_finder_world_size_1_nccl():
    """NEXT #4 on the one GPU there is: ShardedClusterFinder under a world-size-1 NCCL group drives plane_partition ->
    tpc_cf_run (with the frame-wide launch-shape hint) -> gather_records on device tensors; result against the oracle."""
    import socket
    import torch
    import torch.distributed as dist
    cf = _cf()
    c = dict(gen.CONFIGS[3]); c["n_sectors"] = 2
    geom = gen.geometry(c)
    digits = gen.generate(c)
    ora, ost = orc.run_parallel(digits, *geom[:4])[:2]
    created = not dist.is_initialized()
    if created:
        s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
        dist.init_process_group("nccl", init_method="tcp://127.0.0.1:%d" % port, rank=0, world_size=1,
                                device_id=torch.device("cuda:0"))
    try:
        sf = cf.ShardedClusterFinder(*geom[:4], max_digits=digits.shape[0], max_clusters=ost["n_clusters"] + 16)
        out, counts, part = sf.run(digits)
        assert counts == [ost["n_clusters"]] and part[:2] == (0, geom[0] * geom[1])
        cl = out.cpu().numpy().view(cf.CLUSTER)
        assert_clusters_equal(cl, ora, "sharded, world size 1")
        sf.close()
    finally:
        if created:
            dist.destroy_process_group()


def test_unsorted_input_more_peaks_than_the_workspace_holds():
    """unsorted input, workspace max_clusters < n_clusters <= capacity: the key sort keeps max_clusters
    records only, so the run must say overflow = 1 (and the true count) instead of handing back uninitialised tail
    records.  What is written: the first max_clusters peaks in digit order, sorted by key (A2)."""
    import torch
    cf = _cf()
    digits = gen.generate(1)
    geom = gen.geometry(1)
    ora, ost = orc.run(digits, *geom[:4])
    n = digits.shape[0]
    sh = digits[np.random.default_rng(5).permutation(n)]
    mc = 1000
    f = cf.ClusterFinder(*geom[:4], max_digits=n, max_clusters=mc)
    big = torch.zeros(ost["n_clusters"] * 32 + 64, dtype=torch.uint8, device="cuda:0")
    f.run(cf.to_device(sh), n, flags=cf.FORCE_GENERAL, clusters=big, capacity=ost["n_clusters"] + 2)
    cl, st = f.result(clusters=big)
    assert st["path"] == 1 and st["n_clusters"] == ost["n_clusters"] and st["overflow"] == 1
    # the kept subset: peaks of the first digits (in the shuffled order) that are peaks, mc of them, sorted
    k_all = key(ora)
    dk = ((sh["sector"].astype(np.uint64) << 32) | (sh["row"].astype(np.uint64) << 24) |
          (sh["pad"].astype(np.uint64) << 16) | sh["time"].astype(np.uint64))
    is_peak = np.isin(dk, k_all)
    first = np.sort(dk[is_peak][:mc])
    assert np.array_equal(key(cl[:mc]), first)
    f.close()


def test_sorted_only_workspace():
    """TPC_CF_WS_SORTED_ONLY: no charge map, no sort scratch in the workspace (22 GB less at the full geometry); sorted
    runs give the same clusters; a run that needs the general path is refused synchronously."""
    cf = _cf()
    digits = gen.generate(2)
    geom = gen.geometry(2)
    ora, ost = orc.run_parallel(digits, *geom[:4])[:2]
    n = digits.shape[0]
    full = cf.ClusterFinder(*geom[:4], max_digits=n, max_clusters=ost["n_clusters"] + 16)
    lean = cf.ClusterFinder(*geom[:4], max_digits=n, max_clusters=ost["n_clusters"] + 16, sorted_only=True)
    assert lean.workspace_bytes < full.workspace_bytes - 2 * 152 * 138 * 14336
    full.close()
    d = cf.to_device(digits)
    lean.run(d, n, flags=cf.DIGITS_SORTED)
    cl, st = lean.result()
    assert st["path"] == 3 and st["n_clusters"] == ost["n_clusters"]
    assert_clusters_equal(cl, ora, "sorted-only workspace")
    for flags in (0, cf.DIGITS_SORTED | cf.FORCE_GENERAL):
        with pytest.raises(cf.TpcCfError) as e:
            lean.run(d, n, flags=flags)
        assert e.value.code == -5
    lean.close()


@pytest.mark.parametrize("route", ["sorted_on_device", "general"])
def test_shuffled_full_frame_config3(route):
    """Any-order contract at full size: the whole 36-sector config-3 frame in a random order, no
    DIGITS_SORTED promise: the identical array (R12), every cluster against the oracle — digit sort + fused path, and
    the general path + key sort of the clusters."""
    import torch
    cf = _cf()
    geom = gen.geometry(3)
    digits = gen.generate(3)
    n = digits.shape[0]
    ora, ost, _ = orc.run_parallel(digits, *geom[:4])
    f = cf.ClusterFinder(*geom[:4], max_digits=n, max_clusters=ost["n_clusters"] + 1024)
    d = cf.to_device(digits)
    g = torch.Generator(device="cuda:0")
    g.manual_seed(3)
    sh = d.view(torch.int64)[torch.randperm(n, device="cuda:0", generator=g)].contiguous().view(torch.uint8)
    del d
    f.run(sh, n, flags=PATHS[route])
    cl, st = f.result()
    assert st["path"] == EXPECT_PATH[route] and st["overflow"] == 0 and st["n_clusters"] == ost["n_clusters"]
    assert st["n_bad_digits"] == 0 and st["n_digits_used"] == n
    assert_clusters_equal(cl, ora, "config 3 shuffled/" + route)
    f.close()


def test_duplicate_cell_in_unsorted_input_is_reported():
    """Two digits on the same cell are a contract violation (R11).  On input without the DIGITS_SORTED promise the digit
    sort sees the cell's bit already set in the line's time bitmap: the run reports path 0 and no output, exactly like a
    false promise (on the general path the result for that cell stays unspecified, but nothing crashes)."""
    digits = gen.generate(1)
    geom = gen.geometry(1)
    dup = np.concatenate([digits, digits[1234:1235]])
    dup = dup[np.random.default_rng(9).permutation(dup.shape[0])]
    cl, st = gpu_run(dup, geom, PATHS["sorted_on_device"])
    assert st["path"] == 0 and st["n_clusters"] == 0
    cl, st = gpu_run(dup, geom, PATHS["general"])
    assert st["path"] == 1 and st["n_clusters"] > 3000


@pytest.mark.parametrize("seed", list(range(12)))
def test_random_geometries_every_route(seed):
    """Randomised cross-check: random geometry (sectors, rows, pads per row, time bins — including sizes that are no
    multiple of any tile), random clustered digits with invalid ones mixed in (R11), in random order for the routes that
    take any order; every route against the oracle, counts of invalid digits included."""
    rng = np.random.default_rng(1000 + seed)
    n_sectors, n_rows = int(rng.integers(1, 4)), int(rng.integers(1, 7))
    max_pads = int(rng.integers(3, 40))
    n_time = int(rng.choice([17, 64, 100, 513, 2000, 14336]))
    npads = rng.integers(max(1, max_pads // 2), max_pads + 1, size=n_rows).astype(np.uint16)
    npads[int(rng.integers(0, n_rows))] = max_pads
    cells = {}
    for s in range(n_sectors):
        for r in range(n_rows):
            for _ in range(int(rng.integers(0, 1 + max(1, int(npads[r]) * n_time // 40)))):
                p0, t0 = int(rng.integers(0, npads[r])), int(rng.integers(0, n_time))
                for dp in range(-1, 2):
                    for dt in range(-2, 3):
                        p, t = p0 + dp, t0 + dt
                        if 0 <= p < npads[r] and 0 <= t < n_time and rng.random() < 0.75:
                            cells[(s, r, p, t)] = int(rng.choice([1, 2, 3, 4, 5, 7, 20, 300, 65535]))
    rows = [(s, r, p, 0, t, q) for (s, r, p, t), q in cells.items()]
    n_bad = int(rng.integers(0, 6))
    for _ in range(n_bad):                                  # invalid digits, each unique so that nothing is a duplicate cell
        kind = int(rng.integers(0, 5))
        s, r = int(rng.integers(0, n_sectors)), int(rng.integers(0, n_rows))
        if kind == 0:
            rows.append((n_sectors + int(rng.integers(0, 3)), r, 0, 0, len(rows) % n_time, 9))
        elif kind == 1:
            rows.append((s, n_rows + int(rng.integers(0, 3)), 0, 0, len(rows) % n_time, 9))
        elif kind == 2:
            rows.append((s, r, int(npads[r]) + int(rng.integers(0, 3)), 0, len(rows) % n_time, 9))
        elif kind == 3:
            rows.append((s, r, 0, 0, n_time + len(rows) % 50, 9))
        else:
            free = [(p, t) for p in range(int(npads[r])) for t in range(min(n_time, 40)) if (s, r, p, t) not in cells]
            p, t = free[int(rng.integers(0, len(free)))]
            cells[(s, r, p, t)] = 0
            rows.append((s, r, p, 0, t, 0))               # zero charge
    digits = np.array(rows, dtype=orc.DIGIT) if rows else np.zeros(0, dtype=orc.DIGIT)
    geom = (n_sectors, n_rows, max_pads, n_time, npads)
    ora, ost = orc.run(digits, *geom[:4], npads=npads)
    assert ost["n_bad_digits"] == n_bad
    srt = sort_digits(digits)
    shuffled = digits[rng.permutation(digits.shape[0])]
    for route, data in (("sorted_on_device", shuffled), ("general", shuffled), ("fused", srt), ("fused_pairs", srt),
                        ("fused_blocks", srt), ("fused_lines", srt), ("general_hint", srt)):
        cl, st = gpu_run(data, geom, PATHS[route], tuning=TUNING.get(route, {}))
        assert st["path"] == EXPECT_PATH.get(route, 3), (route, st)
        assert st["n_clusters"] == ost["n_clusters"] and st["n_bad_digits"] == n_bad, (route, st, ost)
        assert_clusters_equal(cl, ora, "random geometry %d/%s" % (seed, route))


@pytest.mark.parametrize("route", ["fused", "sorted_on_device", "general", "fused+share"])
def test_run_is_capturable_in_a_cuda_graph(route):
    """tpc_cf_run only enqueues work on the caller's stream (no allocation, no synchronisation, no host read): the whole
    call can be captured in a CUDA graph and replayed — the launch-bound small frames (config 1: 3 launches, 64 us) are
    the case that wants it.  The replay must recompute from the buffers' present contents."""
    import torch
    cf = _cf()
    digits, geom = gen.generate(1), gen.geometry(1)
    n = digits.shape[0]
    share = route.endswith("+share")
    flags = PATHS[route.split("+")[0]] | (cf.SHARE_CHARGE if share else 0)
    ora, ost = orc.run(digits, *geom[:4], flags=orc.SHARE_CHARGE if share else 0)
    f = cf.ClusterFinder(*geom[:4], max_digits=n, max_clusters=ost["n_clusters"] + 64)
    buf = cf.to_device(digits).clone()
    f.run(buf, n, flags=flags)                    # warm-up outside the capture (module load, attributes)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g):
        f.run(buf, n, flags=flags)
    for rep in range(3):
        if rep and not (flags & cf.DIGITS_SORTED):
            # another order of the same digits in the same buffer: the result must be the same array (R12)
            perm = torch.from_numpy(np.random.default_rng(rep).permutation(n)).cuda()
            buf.view(torch.int64).copy_(cf.to_device(digits).view(torch.int64)[perm])
        f.clusters.zero_(); f.status.zero_()
        g.replay()
        cl, st = f.result()
        assert st["n_clusters"] == ost["n_clusters"] and st["path"] == EXPECT_PATH.get(route.split("+")[0], 3)
        assert_clusters_equal(cl, ora, "graph replay %d/%s" % (rep, route))
    del g
    f.close()
