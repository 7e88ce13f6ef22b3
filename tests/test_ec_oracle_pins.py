"""CPU pins of the TPC-EC v1 oracle (oracle/tpc_ec_oracle.c; SURVEY.md §8(f) NEXT #2, step named in PAPER.md:55, 57).

The paper prints no format and no example for this step, so the pins are: hand-evaluated coder steps, normalisations
and symbol bytes (tests/golden/ec_examples.txt); an independent decoder / container parser / symboliser in another
language (tests/ec_brute.py); the information-content identity of rANS (bytes emitted = sum of log2(M/f) to within
log2(1 + 2^-11) bits per symbol — the bound that follows from the renormalisation interval); closed forms
(single-symbol stream: zero bytes; uniform counts: 16 each; counts that divide 4096: exact); round trips; quantisation
bounds; malformed containers."""
import math
import os

import numpy as np
import pytest

import ec_brute
from datagen.ec_gen import synthetic_clusters
from oracle import ec_oracle as eco

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "ec_examples.txt")


def parse_golden():
    rans, norms, clusters, streams = [], [], [], {}
    cur = None
    for line in open(GOLDEN):
        line = line.rstrip("\n")
        if not line.strip() or line.startswith("#"):
            continue
        tag, rest = line[0], line[1:].split()
        if tag == "R":
            cur = {"name": rest[0]}
            rans.append(cur)
        elif tag == "F":
            cur["freq"] = {int(rest[i]): int(rest[i + 1]) for i in range(0, len(rest), 2)}
        elif tag == "M":
            cur["msg"] = [int(x) for x in rest]
        elif tag == "X":
            cur["state"] = int(rest[0])
        elif tag == "B":
            cur["bytes"] = [int(x) for x in rest]
        elif tag == "H":
            norms.append({"hist": {int(rest[i]): int(rest[i + 1]) for i in range(0, len(rest), 2)}})
        elif tag == "N":
            norms[-1]["freq"] = {int(rest[i]): int(rest[i + 1]) for i in range(0, len(rest), 2)}
        elif tag == "C":
            clusters.append(tuple(float(x) for x in rest))
        elif tag == "S":
            streams[int(rest[0])] = [int(x) for x in rest[1:]]
    return rans, norms, clusters, streams


RANS, NORMS, GCLUSTERS, GSTREAMS = parse_golden()


def table(d):
    f = np.zeros(256, dtype=np.uint16)
    for s, v in d.items():
        f[s] = v
    return f


def golden_clusters():
    cl = np.zeros(len(GCLUSTERS), dtype=eco.CLUSTER)
    for i, c in enumerate(GCLUSTERS):
        cl[i] = (int(c[0]), int(c[1]), int(c[2]), int(c[3]), int(c[4]), int(c[5]), int(c[6]), c[7], c[8], c[9], c[10], 0)
    return cl


# ---- (C) lane coder ---------------------------------------------------------------------------------------------

@pytest.mark.parametrize("ex", RANS, ids=[e["name"] for e in RANS])
def test_lane_encoder_hand_evaluated(ex):
    x, b = eco.lane_encode(np.array(ex["msg"], dtype=np.uint8), table(ex["freq"]))
    assert x == ex["state"] and list(b) == ex["bytes"]
    sym, err = eco.lane_decode(x, b, table(ex["freq"]), len(ex["msg"]))
    assert err == 0 and list(sym) == ex["msg"]
    assert ec_brute.lane_decode(x, list(b), table(ex["freq"]), len(ex["msg"])) == ex["msg"]


def random_table(rng, k):
    syms = rng.choice(256, size=k, replace=False)
    w = rng.gamma(0.5, size=k) + 1e-3
    hist = np.zeros(256, dtype=np.uint64)
    hist[syms] = np.maximum(1, (w / w.sum() * 100000).astype(np.uint64))
    return eco.normalize(hist), hist


@pytest.mark.parametrize("seed", range(12))
def test_lane_round_trip_with_independent_decoder_and_information_identity(seed):
    rng = np.random.default_rng(100 + seed)
    k = [1, 2, 3, 7, 16, 40, 100, 256, 256, 5, 2, 64][seed]
    freq, hist = random_table(rng, k)
    assert int(freq.astype(np.int64).sum()) == 4096
    p = hist.astype(np.float64) / hist.sum()
    m = int(rng.integers(1, 700))
    msg = rng.choice(256, size=m, p=p).astype(np.uint8)
    x, b = eco.lane_encode(msg, freq)
    assert (1 << 23) <= x < (1 << 31)
    # independent decoder (another language, searchsorted symbol lookup) reproduces the message and ends at x == L
    assert ec_brute.lane_decode(x, list(b), freq, m) == list(msg)
    sym, err = eco.lane_decode(x, b, freq, m)
    assert err == 0 and np.array_equal(sym, msg)
    # information identity: every coding step multiplies x by M/f to within a factor 1 +- 2^-11
    bits = 8 * len(b) + math.log2(x) - 23
    want = ec_brute.information_bits(msg, freq)
    assert abs(bits - want) <= m * math.log2(1 + 2.0 ** -11) + 1e-6, (bits, want)
    assert len(b) <= 3 * m // 2 + 2


def test_lane_decoder_flags_a_corrupted_lane():
    freq = table({0: 4000, 1: 96})
    msg = np.array([0, 1, 0, 0, 1, 1, 0, 1] * 20, dtype=np.uint8)
    x, b = eco.lane_encode(msg, freq)
    assert len(b) > 4
    _, err = eco.lane_decode(x, b[:-1], freq, len(msg))           # a missing byte
    assert err == eco.ERR_CONTAINER
    _, err = eco.lane_decode(x, np.concatenate([b, [7]]).astype(np.uint8), freq, len(msg))   # a spare byte
    assert err == eco.ERR_CONTAINER


# ---- (N) normalisation -----------------------------------------------------------------------------------------

@pytest.mark.parametrize("i", range(len(NORMS)))
def test_normalisation_hand_evaluated(i):
    hist = np.zeros(256, dtype=np.uint64)
    for s, v in NORMS[i]["hist"].items():
        hist[s] = v
    assert np.array_equal(eco.normalize(hist), table(NORMS[i]["freq"]))


def test_normalisation_closed_forms_and_invariants():
    assert np.array_equal(eco.normalize(np.full(256, 5, np.uint64)), np.full(256, 16, np.uint16))
    assert np.array_equal(eco.normalize(np.zeros(256, np.uint64)), np.zeros(256, np.uint16))
    rng = np.random.default_rng(7)
    for _ in range(200):
        k = int(rng.integers(1, 257))
        hist = np.zeros(256, dtype=np.uint64)
        hist[rng.choice(256, size=k, replace=False)] = rng.integers(1, 10 ** int(rng.integers(1, 8)), size=k)
        f = eco.normalize(hist).astype(np.int64)
        assert f.sum() == 4096 and np.array_equal(f > 0, hist > 0)
        # counts that already sum to a divisor-friendly total are reproduced exactly
    hist = np.zeros(256, dtype=np.uint64)
    hist[[1, 2, 3, 4]] = [1024, 512, 512, 2048]
    assert np.array_equal(eco.normalize(hist * 3)[[1, 2, 3, 4]], [1024, 512, 512, 2048])
    # away from the corrected symbol the frequency is floor(c * 4096 / n), at least 1
    hist = np.zeros(256, dtype=np.uint64)
    hist[:50] = rng.integers(1, 100000, size=50)
    f = eco.normalize(hist).astype(np.int64)
    n = int(hist.sum())
    a = int(np.argmax(hist))
    for s in range(50):
        if s != a:
            assert f[s] == max(1, int(hist[s]) * 4096 // n)


# ---- (Q) symbol streams ----------------------------------------------------------------------------------------

def test_symbol_streams_hand_evaluated():
    cl = golden_clusters()
    st, err = eco.symbolize(cl, 2, 4)
    assert err == 0
    for s in range(13):
        assert list(st[s]) == GSTREAMS[s], s
    assert np.array_equal(ec_brute.symbol_bytes(cl, 4), st)


def test_symbol_streams_against_independent_symboliser():
    rng = np.random.default_rng(3)
    cl = synthetic_clusters(rng, 2, 3, 3000, max_pads=20, n_time=300)   # dense: many same-pad successors
    st, err = eco.symbolize(cl, 2, 3)
    assert err == 0
    assert np.array_equal(ec_brute.symbol_bytes(cl, 3), st)
    assert (st[0] == 0).sum() > 500          # the time-delta branch is exercised


def test_symboliser_error_bits():
    cl = golden_clusters()
    bad = cl.copy()
    bad[[1, 2]] = bad[[2, 1]]
    assert eco.symbolize(bad, 2, 4)[1] & eco.ERR_UNSORTED
    dup = cl.copy()
    dup[1] = dup[0]
    assert eco.symbolize(dup, 2, 4)[1] & eco.ERR_UNSORTED
    assert eco.symbolize(cl, 1, 4)[1] & eco.ERR_UNSORTED          # sector 1 outside the geometry
    q = cl.copy()
    q["qtot"][0] = 3
    assert eco.symbolize(q, 2, 4)[1] == eco.ERR_QTOT


# ---- (F) container ---------------------------------------------------------------------------------------------

def dequantised(cl, n_rows):
    """what the decoder must return: integers untouched, floats replaced by their quantised values (from ec_brute)"""
    st = ec_brute.symbol_bytes(cl, n_rows).astype(np.float64)
    out = cl.copy()
    out["pad_mean"] = cl["pad"] + (st[9] - 128) / 64
    out["time_mean"] = cl["time"] + (st[10] - 128) / 64
    out["sigma_pad"] = st[11] / 128
    out["sigma_time"] = st[12] / 128
    out["rsv"] = 0
    return out


@pytest.mark.parametrize("n", [0, 1, 31, 33, 700, 16384, 16385, 40000])
def test_container_round_trip_and_independent_parser(n):
    rng = np.random.default_rng(n + 1)
    cl = synthetic_clusters(rng, 3, 5, n) if n else np.zeros(0, dtype=eco.CLUSTER)
    n = cl.shape[0]
    buf, err, total = eco.encode(cl, 3, 5)
    assert err == 0 and total == buf.shape[0] and total <= eco.max_bytes(3, 5, n)
    want = dequantised(cl, 5) if n else cl
    dec, derr = eco.decode(buf)
    assert derr == 0 and dec.shape[0] == n
    assert dec.tobytes() == want.tobytes()
    if n <= 16385:      # the pure-Python walk is slow
        c = ec_brute.parse(buf)
        assert c["n"] == n and int(c["counts"].sum()) == n
        assert np.array_equal(c["counts"], np.bincount(cl["sector"].astype(np.int64) * 5 + cl["row"], minlength=15))
        if n <= 700:
            streams = ec_brute.decode_streams(c)
            assert np.array_equal(streams, eco.symbolize(cl, 3, 5)[0])
            assert ec_brute.rebuild(c, streams, eco.CLUSTER).tobytes() == want.tobytes()


def test_round_trip_keeps_integers_and_bounds_the_float_error():
    rng = np.random.default_rng(11)
    cl = synthetic_clusters(rng, 2, 4, 20000)
    buf, err, _ = eco.encode(cl, 2, 4)
    dec, derr = eco.decode(buf)
    assert err == 0 and derr == 0
    for f in ("sector", "row", "pad", "time", "qmax", "qtot", "flags"):
        assert np.array_equal(dec[f], cl[f]), f
    assert np.abs(dec["pad_mean"].astype(np.float64) - cl["pad_mean"]).max() <= 1 / 128 + 1e-6
    assert np.abs(dec["time_mean"].astype(np.float64) - cl["time_mean"]).max() <= 1 / 128 + 2e-4   # fp32 ulp at t ~ 2000
    assert np.abs(dec["sigma_pad"].astype(np.float64) - cl["sigma_pad"]).max() <= 1 / 256 + 1e-6
    assert np.abs(dec["sigma_time"].astype(np.float64) - cl["sigma_time"]).max() <= 1 / 256 + 1e-6


def test_container_size_is_the_cross_entropy_plus_the_stated_overheads():
    rng = np.random.default_rng(5)
    cl = synthetic_clusters(rng, 2, 4, 60000)
    n = cl.shape[0]
    buf, err, total = eco.encode(cl, 2, 4)
    st, _ = eco.symbolize(cl, 2, 4)
    bits = 0.0
    for s in range(13):
        hist = np.bincount(st[s], minlength=256).astype(np.uint64)
        f = eco.normalize(hist).astype(np.float64)
        nz = hist > 0
        bits += float((hist[nz] * np.log2(4096 / f[nz])).sum())
    nb = (n + 16383) // 16384
    fixed = (64 + 4 * 8 + 2 * 256 * 13 + 7) // 8 * 8 + 8 * (13 * nb + 1) + 13 * nb * 192
    payload = total - fixed
    # every lane keeps at most one byte of slack in its final state, and padding is < 4 bytes per record
    assert bits / 8 - 13 * nb * 32 - n * 13 * 1e-4 <= payload <= bits / 8 + 13 * nb * (32 + 3) + n * 13 * 1e-4
    assert total < 0.6 * 32 * n          # and it does compress (13 raw symbol bytes per cluster would be 0.41)


def test_degenerate_streams_cost_no_bytes():
    cl = np.zeros(100, dtype=eco.CLUSTER)
    cl["time"] = np.arange(1, 101)           # one pad line, time step 1: every stream is constant except c0's T_LO
    cl["qmax"] = 9
    cl["qtot"] = 9
    buf, err, total = eco.encode(cl, 1, 1)
    c = ec_brute.parse(buf)
    assert err == 0
    for s in range(13):
        r0, r1 = int(c["rec_off"][s]), int(c["rec_off"][s + 1])
        assert r1 - r0 == 192, s             # 32 states + 32 zero byte counts, no payload
    dec, derr = eco.decode(buf)
    assert derr == 0 and np.array_equal(dec["time"], cl["time"])


def test_decoder_rejects_malformed_containers_and_small_buffers():
    rng = np.random.default_rng(2)
    cl = synthetic_clusters(rng, 2, 4, 500)
    buf, err, total = eco.encode(cl, 2, 4)
    assert eco.decode(buf[:40])[1] == eco.ERR_CONTAINER
    bad = buf.copy(); bad[0] ^= 1
    assert eco.decode(bad)[1] == eco.ERR_CONTAINER
    assert eco.decode(buf[:-4])[1] == eco.ERR_CONTAINER
    bad = buf.copy(); bad[64 + 4 * 8 + 3] ^= 0x10      # a frequency table that no longer sums to 4096
    assert eco.decode(bad)[1] == eco.ERR_CONTAINER
    _, e2, t2 = eco.encode(cl, 2, 4, capacity=total - 1)
    assert e2 == eco.ERR_CAPACITY and t2 == total
    assert eco.decode(buf, capacity=10)[1] == eco.ERR_CAPACITY


def test_cluster_finder_output_round_trips():
    """the coder sits behind the cluster finder: oracle clusters of BASELINE.json configs[0] go through unchanged in
    their integers"""
    from datagen import gen
    from oracle import oracle as orc
    digits = gen.generate(1)
    g = gen.geometry(1)
    cl, _ = orc.run(digits, *g[:4], npads=g[4])
    buf, err, total = eco.encode(cl, g[0], g[1])
    dec, derr = eco.decode(buf)
    assert err == 0 and derr == 0 and dec.shape[0] == cl.shape[0]
    for f in ("sector", "row", "pad", "time", "qmax", "qtot", "flags"):
        assert np.array_equal(dec[f], cl[f]), f
    assert dec.tobytes() == dequantised(cl, g[1]).tobytes()
    assert total < 0.5 * 32 * cl.shape[0]
