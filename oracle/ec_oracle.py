"""ctypes wrapper around the CPU ORACLE of the TPC-EC v1 entropy coder (oracle/tpc_ec_oracle.c).
TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.  It
imports nothing from paper_2402_01205_b200 and the package imports nothing from here.  Definition: tpc_ec_oracle.h
(step named in PAPER.md:55, 57).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libtpc_ec_oracle.so")

CLUSTER = np.dtype([("sector", "u1"), ("row", "u1"), ("pad", "u1"), ("flags", "u1"),
                    ("time", "<u2"), ("qmax", "<u2"), ("qtot", "<u4"),
                    ("pad_mean", "<f4"), ("time_mean", "<f4"),
                    ("sigma_pad", "<f4"), ("sigma_time", "<f4"), ("rsv", "<u4")])
assert CLUSTER.itemsize == 32
N_STREAMS, BLOCK_SYMS, LANES = 13, 16384, 32
ERR_UNSORTED, ERR_CAPACITY, ERR_CONTAINER, ERR_QTOT = 1, 2, 4, 8


def build(force=False):
    """Compile the oracle with gcc (-O2, no CUDA, no floating-point contraction)."""
    src = os.path.join(_HERE, "tpc_ec_oracle.c")
    hdr = os.path.join(_HERE, "tpc_ec_oracle.h")
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(src), os.path.getmtime(hdr))):
        return _SO
    tmp = _SO + ".tmp.%d" % os.getpid()
    subprocess.check_call(["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-Wextra",
                           "-o", tmp, src, "-lm"])
    os.replace(tmp, _SO)
    return _SO


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_SO)
        _lib.tpc_ec_oracle_symbolize.restype = ctypes.c_uint32
        _lib.tpc_ec_oracle_lane_encode.restype = ctypes.c_uint32
        _lib.tpc_ec_oracle_lane_decode.restype = ctypes.c_uint32
        _lib.tpc_ec_oracle_max_bytes.restype = ctypes.c_uint64
        _lib.tpc_ec_oracle_encode.restype = ctypes.c_uint64
        _lib.tpc_ec_oracle_decode.restype = ctypes.c_uint32
        _lib.tpc_ec_oracle_normalize.restype = None
    return _lib


def _p(a):
    return ctypes.c_void_p(a.ctypes.data)


def symbolize(clusters, n_sectors, n_rows):
    """(Q): returns (streams uint8 [13, n], error bits)."""
    cl = np.ascontiguousarray(clusters, dtype=CLUSTER)
    n = cl.shape[0]
    streams = np.zeros((N_STREAMS, max(n, 1)), dtype=np.uint8)
    err = _load().tpc_ec_oracle_symbolize(_p(cl), ctypes.c_uint64(n), ctypes.c_uint32(n_sectors),
                                          ctypes.c_uint32(n_rows), _p(streams))
    return streams[:, :n].copy() if n else np.zeros((N_STREAMS, 0), np.uint8), int(err)


def normalize(hist):
    """(N): hist = 256 counts -> freq uint16 [256] summing to 4096 (or all zero)."""
    h = np.ascontiguousarray(hist, dtype=np.uint64)
    assert h.shape == (256,)
    f = np.zeros(256, dtype=np.uint16)
    _load().tpc_ec_oracle_normalize(_p(h), _p(f))
    return f


def lane_encode(symbols, freq):
    """(C): one lane over `symbols` (uint8).  Returns (final state, emitted bytes in emission order)."""
    s = np.ascontiguousarray(symbols, dtype=np.uint8)
    f = np.ascontiguousarray(freq, dtype=np.uint16)
    out = np.zeros(3 * s.shape[0] // 2 + 8, dtype=np.uint8)
    nb = ctypes.c_uint32(0)
    x = _load().tpc_ec_oracle_lane_encode(_p(s), ctypes.c_uint64(s.shape[0]), ctypes.c_uint64(1), _p(f), _p(out),
                                          ctypes.byref(nb))
    return int(x), out[:nb.value].copy()


def lane_decode(state, data, freq, m):
    """(C) inverse.  Returns (symbols, error bits)."""
    d = np.ascontiguousarray(data, dtype=np.uint8)
    f = np.ascontiguousarray(freq, dtype=np.uint16)
    out = np.zeros(max(m, 1), dtype=np.uint8)
    err = _load().tpc_ec_oracle_lane_decode(ctypes.c_uint32(state), _p(d) if d.size else None,
                                            ctypes.c_uint32(d.shape[0]), _p(f), _p(out), ctypes.c_uint64(m),
                                            ctypes.c_uint64(1))
    return out[:m].copy(), int(err)


def max_bytes(n_sectors, n_rows, n):
    return int(_load().tpc_ec_oracle_max_bytes(ctypes.c_uint32(n_sectors), ctypes.c_uint32(n_rows), ctypes.c_uint64(n)))


def encode(clusters, n_sectors, n_rows, capacity=None):
    """(F): returns (container uint8 array, error bits)."""
    cl = np.ascontiguousarray(clusters, dtype=CLUSTER)
    n = cl.shape[0]
    cap = max_bytes(n_sectors, n_rows, n) if capacity is None else int(capacity)
    out = np.zeros(max(cap, 1), dtype=np.uint8)
    err = ctypes.c_uint32(0)
    total = _load().tpc_ec_oracle_encode(_p(cl), ctypes.c_uint64(n), ctypes.c_uint32(n_sectors),
                                         ctypes.c_uint32(n_rows), _p(out), ctypes.c_uint64(cap), ctypes.byref(err))
    total = int(total)
    return (out[:total].copy() if total <= cap else out[:0].copy()), int(err.value), total


def decode(container, capacity=None):
    """(F) inverse: returns (clusters, error bits)."""
    c = np.ascontiguousarray(container, dtype=np.uint8)
    n_hdr = int(np.frombuffer(c[8:16].tobytes(), dtype="<u8")[0]) if c.shape[0] >= 16 else 0
    cap = n_hdr if capacity is None else int(capacity)
    out = np.zeros(max(cap, 1), dtype=CLUSTER)
    n = ctypes.c_uint64(0)
    err = _load().tpc_ec_oracle_decode(_p(c), ctypes.c_uint64(c.shape[0]), _p(out), ctypes.c_uint64(cap), ctypes.byref(n))
    return out[:min(int(n.value), cap)].copy(), int(err)
