"""-m gpu parity tests of the entropy coder (include/tpc_ec.h, csrc/tpc_ec.cu) against the CPU oracle
(oracle/tpc_ec_oracle.c): byte work, so the bar is bit-exact — the encoder's container equals the oracle's byte for
byte on the same clusters, the decoder's records equal the oracle decoder's byte for byte, error bits agree.
Step named in PAPER.md:55, 57; format: the TPC-EC v1 text in include/tpc_ec.h.
"""
import numpy as np
import pytest

from datagen import gen
from datagen.ec_gen import synthetic_clusters
from oracle import ec_oracle as eco
from oracle import oracle as orc

pytestmark = pytest.mark.gpu


def _cf():
    import paper_2402_01205_b200 as cf
    return cf


def gpu_encode(cl, n_sectors, n_rows, capacity=None, coder=None):
    """Returns (container bytes or None, status dict)."""
    import torch
    cf = _cf()
    n = int(cl.shape[0])
    own = coder is None
    if own:
        coder = cf.ClusterCoder(n_sectors, n_rows, max(n, 1))
    cap = coder.max_encoded_bytes(n) if capacity is None else capacity
    out = torch.full((max(cap, 16) + 64,), 0xA5, dtype=torch.uint8, device="cuda:0")   # poisoned: every byte must be written
    d = cf.clusters_to_device(cl)
    coder.encode(d, n, out, out_capacity=cap)
    st = coder.read_status()
    buf = out[:min(st["bytes"], cap)].cpu().numpy() if st["error"] & cf.EC_ERR_CAPACITY == 0 else None
    tail = out[cap:].cpu().numpy()
    assert np.all(tail == 0xA5), "the encoder wrote beyond out_capacity"
    if own:
        coder.close()
    return buf, st


def gpu_decode(buf, n, n_sectors, n_rows, capacity=None, coder=None, in_bytes=None):
    import torch
    cf = _cf()
    own = coder is None
    if own:
        coder = cf.ClusterCoder(n_sectors, n_rows, max(n, 1))
    cap = n if capacity is None else capacity
    b = torch.from_numpy(np.ascontiguousarray(buf)).to("cuda:0")
    out = torch.full(((max(cap, 1) + 2) * 32,), 0xA5, dtype=torch.uint8, device="cuda:0")
    coder.decode(b, buf.shape[0] if in_bytes is None else in_bytes, n, out, capacity=cap)
    st = coder.read_status()
    rec = out[:min(n, cap) * 32].cpu().numpy().view(cf.CLUSTER).copy()
    assert np.all(out[cap * 32:].cpu().numpy() == 0xA5), "the decoder wrote beyond capacity"
    if own:
        coder.close()
    return rec, st


def check_both_ways(cl, n_sectors, n_rows, what):
    want, werr, total = eco.encode(cl, n_sectors, n_rows)
    got, st = gpu_encode(cl, n_sectors, n_rows)
    assert st["error"] == werr == 0, (what, st, werr)
    assert st["bytes"] == total and st["n_clusters"] == cl.shape[0], (what, st, total)
    bad = np.nonzero(got != want)[0]
    assert bad.size == 0, "%s: container differs from the oracle's at %d bytes, first offset %d" % (what, bad.size, bad[0])
    odec, oerr = eco.decode(want)
    dec, dst = gpu_decode(want, cl.shape[0], n_sectors, n_rows)
    assert dst["error"] == oerr == 0 and dst["bytes"] == total and dst["n_clusters"] == cl.shape[0], (what, dst)
    assert dec.tobytes() == odec.tobytes(), "%s: decoded records differ from the oracle decoder's" % what
    for f in ("sector", "row", "pad", "time", "qmax", "qtot", "flags"):
        assert np.array_equal(dec[f], cl[f]), (what, f)
    return total


# sizes around the lane count (32), the block size (16384) and several blocks with a ragged tail
@pytest.mark.parametrize("n", [0, 1, 2, 31, 32, 33, 700, 16383, 16384, 16385, 3 * 16384 + 77, 200000])
def test_container_and_decoder_bit_exact(n):
    rng = np.random.default_rng(1000 + n)
    cl = synthetic_clusters(rng, 3, 5, n) if n else np.zeros(0, dtype=eco.CLUSTER)
    check_both_ways(cl, 3, 5, "n=%d" % n)


def test_dense_lines_many_planes_and_empty_planes():
    rng = np.random.default_rng(5)
    cl = synthetic_clusters(rng, 36, 152, 60000, max_pads=138, n_time=14336)     # ~11 clusters per plane, some empty
    check_both_ways(cl, 36, 152, "sparse planes")
    cl = synthetic_clusters(rng, 2, 3, 90000, max_pads=20, n_time=3000)          # long same-pad runs: time deltas
    assert (np.diff(cl["pad"].astype(int)) == 0).mean() > 0.9
    check_both_ways(cl, 2, 3, "dense lines")
    cl = synthetic_clusters(rng, 4, 4, 5000)
    cl = cl[(cl["sector"] == 1) | (cl["sector"] == 3)]                          # whole sectors empty, first plane empty
    check_both_ways(cl, 4, 4, "empty sectors")
    check_both_ways(cl, 256, 256, "largest geometry")


def test_extreme_field_values():
    """field maxima (pad 255, time 65535, qmax 65535, qtot - qmax = 2^24 - 1, flags 255) and floats that clamp:
    NaN, +-inf, negative sigma, centroid far from the peak, ties of round-half-even"""
    rng = np.random.default_rng(9)
    cl = synthetic_clusters(rng, 2, 256, 4000, max_pads=256, n_time=65536)
    m = cl.shape[0]
    cl["flags"] = rng.integers(0, 256, size=m)
    cl["qmax"][::7] = 65535
    cl["qtot"][::7] = 65535 + (1 << 24) - 1
    cl["qmax"][1::7] = 0
    cl["qtot"][1::7] = 0
    special = np.array([np.nan, np.inf, -np.inf, -1.0, 1e30, -0.0, 1.99609375, 2.0, 0.00390625, 0.01171875], np.float32)
    for f in ("pad_mean", "time_mean", "sigma_pad", "sigma_time"):
        idx = rng.choice(m, size=400, replace=False)
        cl[f][idx] = rng.choice(special, size=400)
    # exact ties: (x + 2) * 64 = k + 0.5
    cl["pad_mean"][:64] = cl["pad"][:64] + (np.arange(64) + 0.5) / 64 - 2
    cl["sigma_time"][:64] = (np.arange(64) + 0.5) / 128
    last = cl[-1:].copy()
    last["sector"], last["row"], last["pad"], last["time"] = 1, 255, 255, 65535
    cl = np.concatenate([cl[:-1], last]) if (cl["sector"][-1], cl["row"][-1]) != (1, 255) else cl
    check_both_ways(cl, 2, 256, "extreme values")


def test_encoder_error_bits_match_the_oracle():
    cf = _cf()
    rng = np.random.default_rng(12)
    cl = synthetic_clusters(rng, 2, 4, 40000)
    # qtot < qmax: coded modulo 2^24, flagged, container still identical
    q = cl.copy()
    q["qtot"][123] = 1
    q["qmax"][123] = 9
    want, werr, total = eco.encode(q, 2, 4)
    got, st = gpu_encode(q, 2, 4)
    assert werr == eco.ERR_QTOT and st["error"] == cf.EC_ERR_QTOT and st["bytes"] == total
    assert np.array_equal(got, want)
    # unsorted / duplicate keys / sector outside the geometry
    bad = cl.copy()
    bad[[20000, 20001]] = bad[[20001, 20000]]
    assert eco.encode(bad, 2, 4)[1] & eco.ERR_UNSORTED
    assert gpu_encode(bad, 2, 4)[1]["error"] & cf.EC_ERR_UNSORTED
    dup = cl.copy()
    dup[777] = dup[776]
    assert eco.encode(dup, 2, 4)[1] & eco.ERR_UNSORTED
    assert gpu_encode(dup, 2, 4)[1]["error"] & cf.EC_ERR_UNSORTED
    assert eco.encode(cl, 1, 4)[1] & eco.ERR_UNSORTED
    assert gpu_encode(cl, 1, 4)[1]["error"] & cf.EC_ERR_UNSORTED
    # capacity: one byte short -> flagged, size reported, nothing beyond the capacity written (checked in gpu_encode)
    _, e2, t2 = eco.encode(cl, 2, 4, capacity=total_of(cl) - 1)
    buf, st = gpu_encode(cl, 2, 4, capacity=total_of(cl) - 1)
    assert e2 == eco.ERR_CAPACITY and st["error"] == cf.EC_ERR_CAPACITY and st["bytes"] == t2 and buf is None
    # capacity below the fixed part: synchronous error
    with pytest.raises(cf.TpcCfError):
        gpu_encode(cl, 2, 4, capacity=100)


def total_of(cl):
    return eco.encode(cl, 2, 4)[2]


def test_decoder_rejects_malformed_containers():
    cf = _cf()
    rng = np.random.default_rng(2)
    cl = synthetic_clusters(rng, 2, 4, 50000)
    n = cl.shape[0]
    buf, err, total = eco.encode(cl, 2, 4)
    c = parse_dir(buf, n)

    def both(b, in_bytes=None):
        o = eco.decode(b[:in_bytes] if in_bytes else b)[1]
        g = gpu_decode(b, n, 2, 4, in_bytes=in_bytes)[1]["error"]
        return o, g

    bad = buf.copy(); bad[0] ^= 1                                   # magic
    assert both(bad) == (eco.ERR_CONTAINER, cf.EC_ERR_CONTAINER)
    assert both(buf, in_bytes=total - 4) == (eco.ERR_CONTAINER, cf.EC_ERR_CONTAINER)          # truncated
    bad = buf.copy(); bad[64 + 4 * 8 + 3] ^= 0x10                   # a frequency table that no longer sums to 4096
    assert both(bad) == (eco.ERR_CONTAINER, cf.EC_ERR_CONTAINER)
    bad = buf.copy(); bad[64] ^= 1                                  # plane counts that no longer sum to n
    assert both(bad)[1] == cf.EC_ERR_CONTAINER
    bad = buf.copy(); bad[c["dir"] + 8 * 3 + 4] = 0x7f              # a record offset far outside the buffer
    assert both(bad) == (eco.ERR_CONTAINER, cf.EC_ERR_CONTAINER)
    bad = buf.copy(); bad[c["rec0"] + 128] ^= 1                     # lane 0's byte count: the lanes no longer end at L
    assert both(bad) == (eco.ERR_CONTAINER, cf.EC_ERR_CONTAINER)
    bad = buf.copy(); bad[c["rec0"] + 2] ^= 0x40                    # lane 0's final state
    assert both(bad) == (eco.ERR_CONTAINER, cf.EC_ERR_CONTAINER)
    # wrong n announced by the caller; output capacity too small; buffer shorter than the fixed part
    assert gpu_decode(buf, n - 1, 2, 4)[1]["error"] & cf.EC_ERR_CONTAINER
    rec, st = gpu_decode(buf, n, 2, 4, capacity=10)
    assert st["error"] == cf.EC_ERR_CAPACITY and eco.decode(buf, capacity=10)[1] == eco.ERR_CAPACITY
    with pytest.raises(cf.TpcCfError):
        gpu_decode(buf[:40], n, 2, 4)
    # random corruption anywhere in the payload: never a crash, never an out-of-bounds write (poison checked)
    for k in range(20):
        bad = buf.copy()
        pos = rng.integers(c["rec0"], total, size=8)
        bad[pos] ^= rng.integers(1, 256, size=8).astype(np.uint8)
        gpu_decode(bad, n, 2, 4)


def parse_dir(buf, n):
    n_sectors, n_rows = int(buf[16:20].view("<u4")[0]), int(buf[20:24].view("<u4")[0])
    off = 64 + 4 * n_sectors * n_rows + 2 * 256 * 13
    d = (off + 7) & ~7
    return {"dir": d, "rec0": int(buf[d:d + 8].view("<u8")[0])}


def test_handle_reuse_and_chain_behind_the_cluster_finder():
    """one handle, several streams of different sizes back to back (stale workspace must not leak), then the chain
    the paper describes: cluster finder output coded on the device without leaving it"""
    import torch
    cf = _cf()
    rng = np.random.default_rng(21)
    coder = cf.ClusterCoder(3, 5, 70000)
    for n in (70000, 10, 33000, 0, 70000):
        cl = synthetic_clusters(rng, 3, 5, n) if n else np.zeros(0, dtype=eco.CLUSTER)
        want, werr, total = eco.encode(cl, 3, 5)
        got, st = gpu_encode(cl, 3, 5, coder=coder)
        assert st["error"] == 0 and np.array_equal(got, want), n
        dec, dst = gpu_decode(want, cl.shape[0], 3, 5, coder=coder)
        assert dst["error"] == 0 and dec.tobytes() == eco.decode(want)[0].tobytes(), n
    coder.close()
    digits = gen.generate(1)
    g = gen.geometry(1)
    f = cf.ClusterFinder(*g[:4], npads=g[4], max_digits=digits.shape[0], max_clusters=digits.shape[0] // 4)
    f.run(cf.to_device(digits), digits.shape[0], flags=cf.DIGITS_SORTED)
    cl, st = f.result()
    n = st["n_clusters"]
    coder = cf.ClusterCoder(g[0], g[1], n)
    out = torch.empty(coder.max_encoded_bytes(n), dtype=torch.uint8, device="cuda:0")
    coder.encode(f.clusters, n, out)                       # device to device
    est = coder.read_status()
    want, werr, total = eco.encode(cl, g[0], g[1])         # the oracle coder on the same records
    assert est["error"] == werr == 0 and est["bytes"] == total
    assert np.array_equal(out[:total].cpu().numpy(), want)
    assert total < 0.5 * 32 * n
    back = torch.empty(n * 32, dtype=torch.uint8, device="cuda:0")
    coder.decode(out, total, n, back)
    assert coder.read_status()["error"] == 0
    dec = back.cpu().numpy().view(cf.CLUSTER)
    assert dec.tobytes() == eco.decode(want)[0].tobytes()
    # and the oracle chain (oracle finder -> oracle coder) agrees in every integer field
    ocl, _ = orc.run(digits, *g[:4], npads=g[4])
    for fld in ("sector", "row", "pad", "time", "qmax", "qtot", "flags"):
        assert np.array_equal(dec[fld], ocl[fld]), fld
    coder.close()
    f.close()


def test_full_frame_cluster_stream():
    """BASELINE.json configs[2] at full size: the cluster finder's ~10^7 clusters coded on the device, container equal
    to the oracle coder's on the same records, decoded back bit-exactly — in the launch configuration bench.py
    --stage ec times."""
    import torch
    cf = _cf()
    geom = gen.geometry(3)
    digits = gen.generate(3)
    n_d = digits.shape[0]
    f = cf.ClusterFinder(*geom[:4], max_digits=n_d, max_clusters=n_d // 12)
    d = cf.to_device(digits)
    f.run(d, n_d, flags=cf.DIGITS_SORTED)
    cl, st = f.result()
    del d
    n = st["n_clusters"]
    assert n > 5_000_000
    coder = cf.ClusterCoder(geom[0], geom[1], n)
    out = torch.empty(coder.max_encoded_bytes(n), dtype=torch.uint8, device="cuda:0")
    coder.encode(f.clusters, n, out)
    est = coder.read_status()
    want, werr, total = eco.encode(cl, geom[0], geom[1])
    assert est["error"] == werr == 0 and est["bytes"] == total
    got = out[:total].cpu().numpy()
    bad = np.nonzero(got != want)[0]
    assert bad.size == 0, "container differs at %d bytes, first %d" % (bad.size, bad[0] if bad.size else -1)
    back = torch.empty(n * 32, dtype=torch.uint8, device="cuda:0")
    coder.decode(out, total, n, back)
    assert coder.read_status()["error"] == 0
    odec, oerr = eco.decode(want)
    assert oerr == 0 and back.cpu().numpy().tobytes() == odec.tobytes()
    assert total < 0.45 * 32 * n
    coder.close()
    f.close()
