"""ctypes wrapper around the CPU ORACLE of the TPC-FE v1 front-end filter (oracle/tpc_fe_oracle.c).
TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.  It
imports nothing from paper_2402_01205_b200 and the package imports nothing from here.  Definition: tpc_fe_oracle.h
(step named in PAPER.md:57).
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libtpc_fe_oracle.so")

DIGIT = np.dtype([("sector", "u1"), ("row", "u1"), ("pad", "u1"), ("rsv", "u1"), ("time", "<u2"), ("charge", "<u2")])
assert DIGIT.itemsize == 8
DEFAULTS = dict(zs_threshold=2, cm_quiet4=12, cm_min_pads=8, it_decay_shift=6, it_kappa_shift=8)


class _Geometry(ctypes.Structure):
    _fields_ = [("n_sectors", ctypes.c_uint32), ("n_rows", ctypes.c_uint32), ("max_pads", ctypes.c_uint32),
                ("n_time", ctypes.c_uint32), ("npads", ctypes.c_void_p)]


class _Params(ctypes.Structure):
    _fields_ = [("zs_threshold", ctypes.c_uint16), ("cm_quiet4", ctypes.c_uint16), ("cm_min_pads", ctypes.c_uint16),
                ("it_decay_shift", ctypes.c_uint8), ("it_kappa_shift", ctypes.c_uint8)]


class _Status(ctypes.Structure):
    _fields_ = [("n_digits", ctypes.c_uint64), ("overflow", ctypes.c_uint32), ("rsv", ctypes.c_uint32)]


def build(force=False):
    """Compile the oracle with gcc (-O2, no CUDA).  Building the checker is not using it."""
    src = os.path.join(_HERE, "tpc_fe_oracle.c")
    hdr = os.path.join(_HERE, "tpc_fe_oracle.h")
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(src), os.path.getmtime(hdr))):
        return _SO
    tmp = _SO + ".tmp.%d" % os.getpid()
    subprocess.check_call(["gcc", "-std=c99", "-O2", "-fPIC", "-shared", "-Wall", "-Wextra", "-o", tmp, src])
    os.replace(tmp, _SO)
    return _SO


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_SO)
        _lib.tpc_fe_oracle_run.restype = ctypes.c_int
    return _lib


def pad_stride(max_pads):
    return (int(max_pads) + 7) // 8 * 8


def run(raw, ped4, n_sectors, n_rows, max_pads, n_time, npads=None, planes=None, capacity=None, **params):
    """raw: uint16 [n_planes, n_time, W]; ped4: uint16 [n_planes, W]  ->  (digits, status dict).  Raises on a
    synchronous error code."""
    lib = _load()
    W = pad_stride(max_pads)
    n_planes = n_sectors * n_rows
    raw = np.ascontiguousarray(raw, dtype=np.uint16)
    ped4 = np.ascontiguousarray(ped4, dtype=np.uint16)
    assert raw.shape == (n_planes, n_time, W) and ped4.shape == (n_planes, W), (raw.shape, ped4.shape)
    np_arr = None if npads is None else np.ascontiguousarray(npads, dtype=np.uint16)
    g = _Geometry(n_sectors, n_rows, max_pads, n_time, None if np_arr is None else np_arr.ctypes.data)
    pr = dict(DEFAULTS)
    pr.update(params)
    prm = _Params(**pr)
    b, e = (0, n_planes) if planes is None else planes
    if capacity is None:
        capacity = int((e - b) * n_time * max_pads)
        capacity = min(capacity, max(1 << 20, capacity // 4))
    out = np.zeros(capacity, dtype=DIGIT)
    st = _Status()
    rc = lib.tpc_fe_oracle_run(ctypes.c_void_p(raw.ctypes.data), ctypes.c_void_p(ped4.ctypes.data), ctypes.byref(g),
                               ctypes.byref(prm), ctypes.c_uint32(b), ctypes.c_uint32(e),
                               ctypes.c_void_p(out.ctypes.data), ctypes.c_uint64(capacity), ctypes.byref(st))
    if rc != 0:
        raise ValueError("tpc_fe_oracle_run: error %d" % rc)
    n = min(int(st.n_digits), capacity)
    return out[:n], {"n_digits": int(st.n_digits), "overflow": int(st.overflow)}
