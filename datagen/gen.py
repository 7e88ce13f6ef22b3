"""Seeded synthetic TPC time frames (inputs only).  ctypes wrapper around datagen/tpc_gen.c.

This module serves both sides (oracle tests and the CUDA path) and holds none of the cluster finder's
arithmetic.  Recipe and calibration: SURVEY.md §8(d), DESIGN.md §6.  Stand-in for the paper's Pb-Pb / pp time
frames, which are not available.
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libtpc_gen.so")

DIGIT = np.dtype([("sector", "u1"), ("row", "u1"), ("pad", "u1"), ("rsv", "u1"),
                  ("time", "<u2"), ("charge", "<u2")])
assert DIGIT.itemsize == 8


def npads_linear(n_rows=152, lo=66, hi=138):
    """config 5 geometry: pads per row linear lo -> hi (66 + floor(72*r/151))."""
    r = np.arange(n_rows, dtype=np.int64)
    return (lo + (hi - lo) * r // (n_rows - 1)).astype(np.uint16)


# BASELINE.json:configs[i-1]; rho calibrated in SURVEY.md §8(d) to the stated occupancies.
CONFIGS = {
    1: dict(seed=1, n_sectors=1, n_rows=152, max_pads=138, n_time=512, rho=20.0 / (138 * 512), npads=None,
            pair_prob=0.0, plateau_rate=0.0, frames=1, label="1 sector, 152x138x512, Poisson(20)/row"),
    2: dict(seed=2, n_sectors=1, n_rows=152, max_pads=138, n_time=14336, rho=2.5e-3, npads=None,
            pair_prob=0.0, plateau_rate=0.0, frames=1, label="1 sector, 152x138x14336, ~5% occupancy"),
    3: dict(seed=3, n_sectors=36, n_rows=152, max_pads=138, n_time=14336, rho=1.0e-3, npads=None,
            pair_prob=0.0, plateau_rate=0.0, frames=1, label="36 sectors, 152x138x14336, ~2% occupancy"),
    4: dict(seed=4, n_sectors=36, n_rows=152, max_pads=138, n_time=14336, rho=4.8e-3, npads=None,
            pair_prob=3.0 / 17.0, plateau_rate=0.01, frames=1,
            label="36 sectors, ~10% occupancy, 30% close pairs, plateaus"),
    5: dict(seed=5, n_sectors=36, n_rows=152, max_pads=138, n_time=14336, rho=2.5e-4, npads="linear",
            pair_prob=0.0, plateau_rate=0.0, frames=4, label="36 sectors, pads 66->138, ~0.5% occupancy, 4 frames"),
}


class _Cfg(ctypes.Structure):
    _fields_ = [("seed", ctypes.c_uint64),
                ("n_sectors", ctypes.c_uint32), ("n_rows", ctypes.c_uint32),
                ("max_pads", ctypes.c_uint32), ("n_time", ctypes.c_uint32),
                ("npads", ctypes.c_void_p),
                ("rho", ctypes.c_double), ("pair_prob", ctypes.c_double), ("plateau_rate", ctypes.c_double),
                ("n_threads", ctypes.c_uint32),
                ("sector_begin", ctypes.c_uint32), ("sector_end", ctypes.c_uint32)]


def build(force=False):
    src = os.path.join(_HERE, "tpc_gen.c")
    if not force and os.path.exists(_SO) and os.path.getmtime(_SO) >= os.path.getmtime(src):
        return _SO
    tmp = _SO + ".tmp.%d" % os.getpid()
    subprocess.check_call(["gcc", "-std=c99", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall",
                           "-Wno-misleading-indentation", "-o", tmp, src, "-lm"])
    os.replace(tmp, _SO)
    return _SO


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_SO)
        _lib.tpc_gen_frame.restype = ctypes.c_int
        _lib.tpc_gen_checksum.restype = ctypes.c_uint64
        _lib.tpc_gen_free.restype = None
    return _lib


def geometry(cfg):
    """(n_sectors, n_rows, max_pads, n_time, npads array or None) of a CONFIGS entry or dict."""
    c = CONFIGS[cfg] if isinstance(cfg, int) else cfg
    npads = c.get("npads")
    if isinstance(npads, str) and npads == "linear":
        npads = npads_linear(c["n_rows"], 66, c["max_pads"])
    return c["n_sectors"], c["n_rows"], c["max_pads"], c["n_time"], npads


def generate(cfg, frame=0, n_threads=0, sectors=None, out=None):
    """Digits of one frame, sorted ascending (sector,row,pad,time).  cfg: key of CONFIGS or a dict with the same
    fields.  sectors=(begin,end) generates only those sectors (same bytes as the full frame's slice).
    out: optional numpy DIGIT array (e.g. pinned) to receive the digits; returns a view of its first n."""
    lib = _load()
    c = CONFIGS[cfg] if isinstance(cfg, int) else cfg
    n_sectors, n_rows, max_pads, n_time, npads = geometry(c)
    keep = None
    ptr = None
    if npads is not None:
        keep = np.ascontiguousarray(npads, dtype=np.uint16)
        ptr = keep.ctypes.data
    b, e = sectors if sectors is not None else (0, 0)
    cc = _Cfg(c["seed"], n_sectors, n_rows, max_pads, n_time, ptr, c["rho"], c.get("pair_prob", 0.0),
              c.get("plateau_rate", 0.0), n_threads, b, e)
    p = ctypes.c_void_p()
    n = ctypes.c_uint64()
    rc = lib.tpc_gen_frame(ctypes.byref(cc), ctypes.c_uint32(frame), ctypes.byref(p), ctypes.byref(n))
    del keep
    if rc != 0:
        raise MemoryError("tpc_gen_frame failed")
    n = int(n.value)
    try:
        src = np.ctypeslib.as_array(ctypes.cast(p, ctypes.POINTER(ctypes.c_uint8)), shape=(max(n, 1) * 8,))
        src = src[:n * 8].view(DIGIT)
        if out is None:
            res = src.copy()
        else:
            if out.shape[0] < n:
                raise ValueError("out too small: need %d digits" % n)
            out[:n] = src
            res = out[:n]
    finally:
        lib.tpc_gen_free(p)
    return res


def checksum(digits):
    lib = _load()
    d = np.ascontiguousarray(digits, dtype=DIGIT)
    return int(lib.tpc_gen_checksum(ctypes.c_void_p(d.ctypes.data), ctypes.c_uint64(d.shape[0])))


def occupancy(digits, cfg):
    n_sectors, n_rows, max_pads, n_time, npads = geometry(cfg)
    pads = int(np.sum(npads)) if npads is not None else n_rows * max_pads
    return digits.shape[0] / float(n_sectors * pads * n_time)
