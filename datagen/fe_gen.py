"""Seeded synthetic raw TPC samples (inputs only) for the front-end filter.  ctypes wrapper around
datagen/tpc_fe_gen.c: a floating-point forward model (pedestal, common-mode dip, ion-tail undershoot, noise) laid over
the digits of datagen/gen.py.  Holds none of the filter's arithmetic; serves the oracle tests and the CUDA path alike.
Stand-in for the detector's raw stream, which is not available.  Recipe: DESIGN.md §11.
"""
import ctypes
import os
import subprocess

import numpy as np

from . import gen

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libtpc_fe_gen.so")

MODEL = dict(noise_sigma=0.5, cm_frac=1.0, tail_lambda=1.0 - 2.0 ** -6, tail_kappa=2.0 ** -8)


class _Cfg(ctypes.Structure):
    _fields_ = [("seed", ctypes.c_uint64),
                ("n_sectors", ctypes.c_uint32), ("n_rows", ctypes.c_uint32),
                ("max_pads", ctypes.c_uint32), ("n_time", ctypes.c_uint32),
                ("npads", ctypes.c_void_p),
                ("noise_sigma", ctypes.c_double), ("cm_frac", ctypes.c_double),
                ("tail_lambda", ctypes.c_double), ("tail_kappa", ctypes.c_double),
                ("plane_begin", ctypes.c_uint32), ("plane_end", ctypes.c_uint32)]


def build(force=False):
    src = os.path.join(_HERE, "tpc_fe_gen.c")
    if not force and os.path.exists(_SO) and os.path.getmtime(_SO) >= os.path.getmtime(src):
        return _SO
    tmp = _SO + ".tmp.%d" % os.getpid()
    subprocess.check_call(["gcc", "-std=c99", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-o", tmp, src, "-lm"])
    os.replace(tmp, _SO)
    return _SO


def pad_stride(max_pads):
    return (int(max_pads) + 7) // 8 * 8


def raw_from_digits(digits, n_sectors, n_rows, max_pads, n_time, npads=None, seed=1, planes=None, out=None, **model):
    """digits (sorted, datagen.gen.DIGIT) -> (raw uint16 [n, n_time, W], ped4 uint16 [n, W]) for planes [b, e).
    `out` may be a preallocated (raw, ped4) pair (e.g. views of pinned memory)."""
    build()
    lib = ctypes.CDLL(_SO)
    lib.tpc_fe_gen_raw.restype = ctypes.c_int
    b, e = (0, n_sectors * n_rows) if planes is None else planes
    W = pad_stride(max_pads)
    if out is None:
        raw = np.empty((e - b, n_time, W), dtype=np.uint16)
        ped4 = np.empty((e - b, W), dtype=np.uint16)
    else:
        raw, ped4 = out
        assert raw.shape == (e - b, n_time, W) and ped4.shape == (e - b, W)
        assert raw.dtype == np.uint16 and ped4.dtype == np.uint16 and raw.flags.c_contiguous and ped4.flags.c_contiguous
    m = dict(MODEL)
    m.update(model)
    np_arr = None if npads is None else np.ascontiguousarray(npads, dtype=np.uint16)
    d = np.ascontiguousarray(digits, dtype=gen.DIGIT)
    cfg = _Cfg(seed, n_sectors, n_rows, max_pads, n_time, None if np_arr is None else np_arr.ctypes.data,
               m["noise_sigma"], m["cm_frac"], m["tail_lambda"], m["tail_kappa"], b, e)
    rc = lib.tpc_fe_gen_raw(ctypes.byref(cfg), ctypes.c_void_p(d.ctypes.data), ctypes.c_uint64(d.shape[0]),
                            ctypes.c_void_p(raw.ctypes.data), ctypes.c_void_p(ped4.ctypes.data))
    if rc != 0:
        raise MemoryError("tpc_fe_gen_raw")
    return raw, ped4
