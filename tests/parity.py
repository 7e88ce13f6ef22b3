"""Element-by-element comparison of the CUDA path's clusters with the oracle's (test helper).

Bar (BASELINE.json:north_star): bit-exact for the peak set, count, order, qMax, qTot,
flags/rsv; floats pass iff |g-o| <= 1e-4 (pads / time bins) or |g-o| <= 1e-5 * |o|.
"""
import numpy as np

ABS_TOL = 1e-4
REL_TOL = 1e-5
INT_FIELDS = ("sector", "row", "pad", "flags", "time", "qmax", "qtot", "rsv")
FLOAT_FIELDS = ("pad_mean", "time_mean", "sigma_pad", "sigma_time")


def key(c):
    return ((c["sector"].astype(np.uint64) << 32) | (c["row"].astype(np.uint64) << 24) |
            (c["pad"].astype(np.uint64) << 16) | c["time"].astype(np.uint64))


def assert_clusters_equal(gpu, ora, what=""):
    assert gpu.shape[0] == ora.shape[0], "%s: cluster count %d != oracle %d" % (what, gpu.shape[0], ora.shape[0])
    for f in INT_FIELDS:
        bad = np.nonzero(gpu[f] != ora[f])[0]
        assert bad.size == 0, "%s: field %s differs at %d entries, first index %d: gpu %s oracle %s" % (
            what, f, bad.size, bad[0], gpu[bad[0]], ora[bad[0]])
    for f in FLOAT_FIELDS:
        g = gpu[f].astype(np.float64)
        o = ora[f].astype(np.float64)
        err = np.abs(g - o)
        ok = (err <= ABS_TOL) | (err <= REL_TOL * np.abs(o))
        bad = np.nonzero(~ok)[0]
        assert bad.size == 0, "%s: field %s out of tolerance at %d entries, first index %d: gpu %s oracle %s" % (
            what, f, bad.size, bad[0], gpu[bad[0]], ora[bad[0]])
    if gpu.shape[0] > 1:
        k = key(gpu)
        assert np.all(k[1:] > k[:-1]), "%s: output not strictly ascending in (sector,row,pad,time)" % what


def max_float_err(gpu, ora):
    return {f: float(np.max(np.abs(gpu[f].astype(np.float64) - ora[f].astype(np.float64)))) if gpu.shape[0] else 0.0
            for f in FLOAT_FIELDS}
