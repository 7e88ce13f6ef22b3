"""ctypes wrapper around the CPU ORACLE (oracle/tpc_cf_oracle.c).  TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
module.  It imports nothing from paper_2402_01205_b200 and the package imports nothing from here.
Definition implemented: SURVEY.md §8(c) (BASELINE.json:north_star; step named in PAPER.md:57).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libtpc_cf_oracle.so")

# Record layouts restated (see tpc_cf_oracle.h); independent of the product's binding on purpose.
DIGIT = np.dtype([("sector", "u1"), ("row", "u1"), ("pad", "u1"), ("rsv", "u1"),
                  ("time", "<u2"), ("charge", "<u2")])
CLUSTER = np.dtype([("sector", "u1"), ("row", "u1"), ("pad", "u1"), ("flags", "u1"),
                    ("time", "<u2"), ("qmax", "<u2"), ("qtot", "<u4"),
                    ("pad_mean", "<f4"), ("time_mean", "<f4"),
                    ("sigma_pad", "<f4"), ("sigma_time", "<f4"), ("rsv", "<u4")])
assert DIGIT.itemsize == 8 and CLUSTER.itemsize == 32


class _Geometry(ctypes.Structure):
    _fields_ = [("n_sectors", ctypes.c_uint32), ("n_rows", ctypes.c_uint32),
                ("max_pads", ctypes.c_uint32), ("n_time", ctypes.c_uint32),
                ("npads", ctypes.c_void_p)]


class _Params(ctypes.Structure):
    _fields_ = [("q_peak_min", ctypes.c_uint16), ("q_inner_gate", ctypes.c_uint16),
                ("flags", ctypes.c_uint32), ("q_tot_min", ctypes.c_uint32),
                ("q_saturation", ctypes.c_uint16), ("rsv", ctypes.c_uint16)]


# variant bits of params.flags (restated from tpc_cf_oracle.h) and cluster flag bits (V1)
CLUSTER_FLAGS, CUT_SINGLE_PAD, CUT_SINGLE_TIME, SHARE_CHARGE = 4, 8, 16, 32
F_EDGE_PAD, F_EDGE_TIME, F_SINGLE_PAD, F_SINGLE_TIME, F_SATURATED, F_SHARED = 1, 2, 4, 8, 16, 32


class _Status(ctypes.Structure):
    _fields_ = [("n_clusters", ctypes.c_uint64), ("n_digits_used", ctypes.c_uint64),
                ("n_bad_digits", ctypes.c_uint64), ("overflow", ctypes.c_uint32),
                ("rsv", ctypes.c_uint32)]


def build(force=False):
    """Compile the oracle with gcc (-O2, no CUDA).  Building the checker is not using it."""
    src = os.path.join(_HERE, "tpc_cf_oracle.c")
    hdr = os.path.join(_HERE, "tpc_cf_oracle.h")
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(src), os.path.getmtime(hdr))):
        return _SO
    tmp = _SO + ".tmp.%d" % os.getpid()
    subprocess.check_call(["gcc", "-std=c99", "-O2", "-fPIC", "-shared", "-Wall", "-Wextra",
                           "-o", tmp, src, "-lm"])
    os.replace(tmp, _SO)
    return _SO


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_SO)
        _lib.tpc_cf_oracle_run_planes.restype = ctypes.c_int
        _lib.tpc_cf_oracle_dense_plane.restype = ctypes.c_int
    return _lib


def _geom(n_sectors, n_rows, max_pads, n_time, npads):
    keep = None
    ptr = None
    if npads is not None:
        keep = np.ascontiguousarray(npads, dtype=np.uint16)
        assert keep.shape == (n_rows,)
        ptr = keep.ctypes.data
    return _Geometry(n_sectors, n_rows, max_pads, n_time, ptr), keep


def run(digits, n_sectors, n_rows, max_pads, n_time, npads=None, q_peak_min=4, q_inner_gate=2,
        capacity=None, planes=None, flags=0, q_tot_min=0, q_saturation=0):
    """Run the oracle.  digits: numpy array of DIGIT (any order).  Returns (clusters, status dict).

    planes=(begin, end) restricts the run to planes sector*n_rows+row in [begin, end).
    capacity=None sizes the output so that nothing overflows (one peak needs one digit)."""
    lib = _load()
    digits = np.ascontiguousarray(digits, dtype=DIGIT)
    n = int(digits.shape[0])
    if capacity is None:
        capacity = max(n, 1)
    out = np.zeros(int(capacity), dtype=CLUSTER)
    g, keep = _geom(n_sectors, n_rows, max_pads, n_time, npads)
    prm = _Params(q_peak_min, q_inner_gate, flags, q_tot_min, q_saturation, 0)
    st = _Status()
    b, e = planes if planes is not None else (0, n_sectors * n_rows)
    rc = lib.tpc_cf_oracle_run_planes(ctypes.c_void_p(digits.ctypes.data), ctypes.c_uint64(n),
                                      ctypes.byref(g), ctypes.byref(prm),
                                      ctypes.c_uint32(b), ctypes.c_uint32(e),
                                      ctypes.c_void_p(out.ctypes.data), ctypes.c_uint64(capacity),
                                      ctypes.byref(st))
    del keep
    if rc != 0:
        raise RuntimeError("tpc_cf_oracle_run failed: %d" % rc)
    status = {"n_clusters": int(st.n_clusters), "n_digits_used": int(st.n_digits_used),
              "n_bad_digits": int(st.n_bad_digits), "overflow": int(st.overflow)}
    return out[:min(int(st.n_clusters), int(capacity))].copy(), status


def dense_plane(digits, n_sectors, n_rows, max_pads, n_time, sector, row, npads=None):
    """Dense uint16 [npads(row), n_time] charge map of one plane, as the definition builds it."""
    lib = _load()
    digits = np.ascontiguousarray(digits, dtype=DIGIT)
    P = int(npads[row]) if npads is not None else max_pads
    dense = np.zeros((P, n_time), dtype=np.uint16)
    g, keep = _geom(n_sectors, n_rows, max_pads, n_time, npads)
    rc = lib.tpc_cf_oracle_dense_plane(ctypes.c_void_p(digits.ctypes.data),
                                       ctypes.c_uint64(digits.shape[0]), ctypes.byref(g),
                                       ctypes.c_uint32(sector), ctypes.c_uint32(row),
                                       ctypes.c_void_p(dense.ctypes.data))
    del keep
    if rc != 0:
        raise RuntimeError("tpc_cf_oracle_dense_plane failed: %d" % rc)
    return dense


def make_digits(cells, sector=0, row=0):
    """Helper for hand-built grids: cells = iterable of (pad, time, charge)."""
    cells = list(cells)
    d = np.zeros(len(cells), dtype=DIGIT)
    for i, (p, t, q) in enumerate(cells):
        d[i] = (sector, row, p, 0, t, q)
    return d


def run_parallel(digits, n_sectors, n_rows, max_pads, n_time, npads=None, n_threads=None, **kw):
    """The same single-threaded routine called on contiguous blocks of (sector,row) planes from n_threads host
    threads; outputs concatenated in plane order.  Planes are independent (R2), so the result
    is the single-threaded result; the caller may check that.  Needs digits whose planes are non-decreasing (sorted
    input), so that a plane block is one contiguous slice; otherwise falls back to one thread.
    Returns (clusters, status dict, threads used)."""
    import concurrent.futures
    import os
    digits = np.ascontiguousarray(digits, dtype=DIGIT)
    n = int(digits.shape[0])
    n_planes = n_sectors * n_rows
    if n_threads is None:
        n_threads = os.cpu_count() or 1
    plane = digits["sector"].astype(np.int32) * np.int32(n_rows) + digits["row"]
    ok = n > 0 and bool(np.all(plane[1:] >= plane[:-1])) and int(plane[-1]) < n_planes and n_threads > 1
    if not ok:
        cl, st = run(digits, n_sectors, n_rows, max_pads, n_time, npads=npads, **kw)
        return cl, st, 1
    # blocks: ~8 per thread, cut at plane boundaries by digit count
    n_blocks = min(n_planes, 8 * n_threads)
    starts = np.searchsorted(plane, np.arange(n_planes + 1))
    cuts = [0]
    for b in range(1, n_blocks):
        p = int(np.searchsorted(starts, n * b // n_blocks))
        p = min(max(p, cuts[-1]), n_planes)
        if p > cuts[-1]:
            cuts.append(p)
    if cuts[-1] != n_planes:
        cuts.append(n_planes)
    del plane

    def work(i):
        b, e = cuts[i], cuts[i + 1]
        lo, hi = int(starts[b]), int(starts[e])
        cap = kw.get("capacity")
        return run(digits[lo:hi], n_sectors, n_rows, max_pads, n_time, npads=npads, planes=(b, e),
                   **{k: v for k, v in kw.items() if k != "capacity"},
                   capacity=max(1, (hi - lo) // 4 + 64) if cap is None else cap)

    with concurrent.futures.ThreadPoolExecutor(max_workers=n_threads) as ex:
        parts = list(ex.map(work, range(len(cuts) - 1)))
    for cl, st in parts:
        if st["overflow"]:
            raise RuntimeError("oracle block overflowed its output estimate")
    status = {k: sum(st[k] for _, st in parts) for k in ("n_clusters", "n_digits_used", "n_bad_digits")}
    status["overflow"] = 0
    return np.concatenate([cl for cl, _ in parts]), status, n_threads
