"""Thin ctypes binding of the C ABI in include/tpc_cf.h — argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libtpc_cf.so; PyTorch is used for device memory and
streams (BASELINE.json:north_star).  There is no CPU fallback: if the library cannot be loaded, or CUDA is not
available, the calls raise.  Function names mirror the C entry points.
"""
import ctypes
import os

import numpy as np

from . import build as _build

DIGIT = np.dtype([("sector", "u1"), ("row", "u1"), ("pad", "u1"), ("rsv", "u1"),
                  ("time", "<u2"), ("charge", "<u2")])
CLUSTER = np.dtype([("sector", "u1"), ("row", "u1"), ("pad", "u1"), ("flags", "u1"),
                    ("time", "<u2"), ("qmax", "<u2"), ("qtot", "<u4"),
                    ("pad_mean", "<f4"), ("time_mean", "<f4"),
                    ("sigma_pad", "<f4"), ("sigma_time", "<f4"), ("rsv", "<u4")])
STATUS = np.dtype([("n_clusters", "<u8"), ("n_digits_used", "<u8"), ("n_bad_digits", "<u8"),
                   ("overflow", "<u4"), ("path", "<u4")])
assert DIGIT.itemsize == 8 and CLUSTER.itemsize == 32 and STATUS.itemsize == 32

DIGITS_SORTED = 1
FORCE_GENERAL = 2
WS_SORTED_ONLY = 1      # tpc_cf_create_ex / tpc_cf_workspace_bytes_ex
# cluster-finder variants (include/tpc_cf.h V1..V3): params.flags bits and tpc_cluster.flags bits
CLUSTER_FLAGS, CUT_SINGLE_PAD, CUT_SINGLE_TIME, SHARE_CHARGE = 4, 8, 16, 32
F_EDGE_PAD, F_EDGE_TIME, F_SINGLE_PAD, F_SINGLE_TIME, F_SATURATED, F_SHARED = 1, 2, 4, 8, 16, 32

# tpc_cf_debug_set keys and the values of "fused_kernel" (include/tpc_cf.h)
DEBUG_KEYS = {"fused_kernel": 1, "passes": 2, "block_pool": 3, "surv_cap": 4, "pads_per_unit": 5, "ctas_per_sm": 6}
FUSED_KERNELS = {"auto": 0, "pairs": 1, "blocks": 2, "lines": 3}

EXPORTS = ["tpc_cf_workspace_bytes", "tpc_cf_workspace_bytes_ex", "tpc_cf_create", "tpc_cf_create_ex", "tpc_cf_run", "tpc_cf_run_host",
           "tpc_cf_debug_dense_plane", "tpc_cf_debug_set", "tpc_cf_set_frame_digits", "tpc_cf_scan_static_max_n",
           "tpc_cf_scan_static_setup", "tpc_cf_scan_u32_static", "tpc_cf_debug_scan_u32", "tpc_cf_last_launch_count", "tpc_cf_last_kernel", "tpc_cf_set_profiling",
           "tpc_cf_profile_ms", "tpc_cf_destroy", "tpc_cf_strerror"]


class Geometry(ctypes.Structure):
    _fields_ = [("n_sectors", ctypes.c_uint32), ("n_rows", ctypes.c_uint32),
                ("max_pads", ctypes.c_uint32), ("n_time", ctypes.c_uint32),
                ("npads", ctypes.c_void_p)]


class Params(ctypes.Structure):
    _fields_ = [("q_peak_min", ctypes.c_uint16), ("q_inner_gate", ctypes.c_uint16),
                ("flags", ctypes.c_uint32), ("q_tot_min", ctypes.c_uint32),
                ("q_saturation", ctypes.c_uint16), ("rsv", ctypes.c_uint16)]


class Out(ctypes.Structure):
    _fields_ = [("clusters", ctypes.c_void_p), ("capacity", ctypes.c_uint64),
                ("status", ctypes.c_void_p), ("stream", ctypes.c_void_p)]


class TpcCfError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("tpc_cf error %d: %s" % (code, text))
        self.code = code


_lib = None


def load(build_if_missing=True):
    """Loads libtpc_cf.so (building it with nvcc if it is missing or stale).  Raises if that fails."""
    global _lib
    if _lib is not None:
        return _lib
    if build_if_missing and _build.stale():
        _build.build()
    if not os.path.exists(_build.SO):
        raise ImportError("libtpc_cf.so is missing; run paper_2402_01205_b200/build.py (needs nvcc)")
    lib = ctypes.CDLL(_build.SO)
    lib.tpc_cf_workspace_bytes.restype = ctypes.c_size_t
    lib.tpc_cf_workspace_bytes.argtypes = [ctypes.POINTER(Geometry), ctypes.c_uint64, ctypes.c_uint64]
    lib.tpc_cf_create.restype = ctypes.c_int
    lib.tpc_cf_create.argtypes = [ctypes.POINTER(ctypes.c_void_p), ctypes.POINTER(Geometry), ctypes.c_uint64,
                                  ctypes.c_uint64, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p]
    lib.tpc_cf_workspace_bytes_ex.restype = ctypes.c_size_t
    lib.tpc_cf_workspace_bytes_ex.argtypes = [ctypes.POINTER(Geometry), ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint32]
    lib.tpc_cf_create_ex.restype = ctypes.c_int
    lib.tpc_cf_create_ex.argtypes = [ctypes.POINTER(ctypes.c_void_p), ctypes.POINTER(Geometry), ctypes.c_uint64,
                                     ctypes.c_uint64, ctypes.c_uint32, ctypes.c_void_p, ctypes.c_size_t, ctypes.c_void_p]
    lib.tpc_cf_run.restype = ctypes.c_int
    lib.tpc_cf_run.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64, ctypes.POINTER(Geometry),
                               ctypes.POINTER(Params), ctypes.POINTER(Out)]
    lib.tpc_cf_run_host.restype = ctypes.c_int
    lib.tpc_cf_run_host.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64, ctypes.POINTER(Geometry),
                                    ctypes.POINTER(Params), ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                    ctypes.c_void_p, ctypes.c_uint64, ctypes.c_void_p, ctypes.c_void_p]
    lib.tpc_cf_debug_dense_plane.restype = ctypes.c_int
    lib.tpc_cf_debug_dense_plane.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint32,
                                             ctypes.c_uint32, ctypes.c_void_p, ctypes.c_void_p]
    lib.tpc_cf_set_frame_digits.restype = ctypes.c_int
    lib.tpc_cf_set_frame_digits.argtypes = [ctypes.c_void_p, ctypes.c_uint64]
    lib.tpc_cf_scan_static_max_n.restype = ctypes.c_uint64
    lib.tpc_cf_scan_static_max_n.argtypes = []
    lib.tpc_cf_scan_static_setup.restype = ctypes.c_int
    lib.tpc_cf_scan_static_setup.argtypes = []
    lib.tpc_cf_scan_u32_static.restype = ctypes.c_int
    lib.tpc_cf_scan_u32_static.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64, ctypes.c_void_p, ctypes.c_void_p]
    lib.tpc_cf_debug_scan_u32.restype = ctypes.c_int
    lib.tpc_cf_debug_scan_u32.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64,
                                          ctypes.c_void_p, ctypes.c_void_p]
    lib.tpc_cf_debug_set.restype = ctypes.c_int
    lib.tpc_cf_debug_set.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int]
    lib.tpc_cf_last_launch_count.restype = ctypes.c_int
    lib.tpc_cf_last_launch_count.argtypes = [ctypes.c_void_p]
    lib.tpc_cf_last_kernel.restype = ctypes.c_char_p
    lib.tpc_cf_last_kernel.argtypes = [ctypes.c_void_p]
    lib.tpc_cf_set_profiling.restype = ctypes.c_int
    lib.tpc_cf_set_profiling.argtypes = [ctypes.c_void_p, ctypes.c_int]
    lib.tpc_cf_profile_ms.restype = ctypes.c_float
    lib.tpc_cf_profile_ms.argtypes = [ctypes.c_void_p, ctypes.c_uint32, ctypes.c_int]
    lib.tpc_cf_destroy.restype = ctypes.c_int
    lib.tpc_cf_destroy.argtypes = [ctypes.c_void_p]
    lib.tpc_cf_strerror.restype = ctypes.c_char_p
    lib.tpc_cf_strerror.argtypes = [ctypes.c_int]
    _lib = lib
    return lib


def _check(rc):
    if rc != 0:
        raise TpcCfError(rc, load().tpc_cf_strerror(rc).decode())


def make_geometry(n_sectors, n_rows, max_pads, n_time, npads=None):
    """Returns (Geometry, keepalive).  npads: optional sequence of n_rows pad counts (host)."""
    keep = None
    ptr = None
    if npads is not None:
        keep = np.ascontiguousarray(npads, dtype=np.uint16)
        if keep.shape != (n_rows,):
            raise ValueError("npads must have n_rows entries")
        ptr = keep.ctypes.data
    return Geometry(n_sectors, n_rows, max_pads, n_time, ptr), keep


def tpc_cf_workspace_bytes(geom, max_digits, max_clusters):
    return int(load().tpc_cf_workspace_bytes(ctypes.byref(geom), max_digits, max_clusters))


def tpc_cf_create(geom, max_digits, max_clusters, workspace_ptr, workspace_bytes, stream_ptr):
    h = ctypes.c_void_p()
    _check(load().tpc_cf_create(ctypes.byref(h), ctypes.byref(geom), max_digits, max_clusters,
                                workspace_ptr, workspace_bytes, stream_ptr))
    return h


def tpc_cf_run(h, digits_ptr, n, geom, params, out):
    _check(load().tpc_cf_run(h, digits_ptr, n, ctypes.byref(geom), ctypes.byref(params), ctypes.byref(out)))


def scan_u32_static(inp, out, n, total=None):
    """tpc_cf_scan_u32_static on torch device tensors (uint32 viewed as int32 or uint8 storage): no allocation, scratch
    in the library's static device array; enqueues on the current torch stream.  Raises TpcCfError beyond the limit."""
    import torch
    stream = torch.cuda.current_stream(inp.device).cuda_stream
    with torch.cuda.device(inp.device):
        _check(load().tpc_cf_scan_u32_static(inp.data_ptr() if n else None, out.data_ptr() if n else None, int(n),
                                             total.data_ptr() if total is not None else None, stream))


def tpc_cf_destroy(h):
    _check(load().tpc_cf_destroy(h))


class ClusterFinder:
    """Owns the torch allocations (workspace, cluster and status buffers) one handle needs.

    run(digits_dev, n) only enqueues on the current torch stream; result() synchronises and reads back."""

    def __init__(self, n_sectors, n_rows, max_pads, n_time, npads=None, max_digits=1 << 20, max_clusters=None,
                 q_peak_min=4, q_inner_gate=2, q_tot_min=0, q_saturation=0, device="cuda:0", sorted_only=False):
        """sorted_only: a workspace without the dense charge map and the sort scratch (TPC_CF_WS_SORTED_ONLY): every
        run must then carry DIGITS_SORTED (22 GB less for the full 36-sector geometry)."""
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("tpc_cf needs a CUDA device; there is no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        self.lib = load()
        self.geom, self._keep = make_geometry(n_sectors, n_rows, max_pads, n_time, npads)
        self.max_digits = int(max_digits)
        self.max_clusters = int(max_clusters if max_clusters is not None else max(1, self.max_digits // 4))
        self.params = Params(q_peak_min, q_inner_gate, 0, q_tot_min, q_saturation, 0)
        ws_flags = WS_SORTED_ONLY if sorted_only else 0
        nbytes = int(self.lib.tpc_cf_workspace_bytes_ex(ctypes.byref(self.geom), self.max_digits, self.max_clusters,
                                                        ws_flags))
        if nbytes == 0:
            raise TpcCfError(-2, "invalid geometry or capacities")
        self.workspace_bytes = nbytes
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            self._ws_ptr = (self.workspace.data_ptr() + 255) & ~255
            self.clusters = torch.empty(self.max_clusters * 32, dtype=torch.uint8, device=self.device)
            self.status = torch.zeros(32, dtype=torch.uint8, device=self.device)
            stream = torch.cuda.current_stream(self.device).cuda_stream
            self.h = ctypes.c_void_p()
            _check(self.lib.tpc_cf_create_ex(ctypes.byref(self.h), ctypes.byref(self.geom), self.max_digits,
                                             self.max_clusters, ws_flags, self._ws_ptr, nbytes, stream))

    def run(self, digits_dev, n=None, flags=0, clusters=None, capacity=None, status=None):
        """digits_dev: torch uint8 tensor on the device holding n 8-byte records."""
        torch = self.torch
        n = int(n if n is not None else digits_dev.numel() // 8)
        clusters = self.clusters if clusters is None else clusters
        capacity = int(capacity if capacity is not None else clusters.numel() // 32)
        status = self.status if status is None else status
        self.params.flags = flags
        out = Out(clusters.data_ptr(), capacity, status.data_ptr(),
                  torch.cuda.current_stream(self.device).cuda_stream)
        tpc_cf_run(self.h, digits_dev.data_ptr() if n else None, n, self.geom, self.params, out)

    def result(self, clusters=None, status=None):
        """Synchronises and returns (numpy CLUSTER array, status dict)."""
        clusters = self.clusters if clusters is None else clusters
        status = self.status if status is None else status
        st = status.cpu().numpy().view(STATUS)[0]
        sd = {k: int(st[k]) for k in STATUS.names}
        m = min(sd["n_clusters"], clusters.numel() // 32)
        cl = clusters[:m * 32].cpu().numpy().view(CLUSTER).copy()
        return cl, sd

    def run_host(self, digits_host, flags=0, dev_digits=None, host_clusters=None):
        """End-to-end call (tpc_cf_run_host): host digits in, host clusters out, copies included."""
        torch = self.torch
        d = digits_host if isinstance(digits_host, torch.Tensor) else torch.from_numpy(
            np.ascontiguousarray(digits_host, dtype=DIGIT).view(np.uint8))
        n = d.numel() // 8
        if dev_digits is None:
            dev_digits = torch.empty(max(n, 1) * 8, dtype=torch.uint8, device=self.device)
        if host_clusters is None:
            host_clusters = torch.empty(self.max_clusters * 32, dtype=torch.uint8, pin_memory=True)
        host_status = torch.zeros(32, dtype=torch.uint8)
        self.params.flags = flags
        stream = torch.cuda.current_stream(self.device).cuda_stream
        _check(self.lib.tpc_cf_run_host(self.h, d.data_ptr() if n else None, n, ctypes.byref(self.geom),
                                        ctypes.byref(self.params), dev_digits.data_ptr(),
                                        self.clusters.data_ptr(), self.status.data_ptr(),
                                        host_clusters.data_ptr(), self.max_clusters, host_status.data_ptr(), stream))
        st = host_status.numpy().view(STATUS)[0]
        sd = {k: int(st[k]) for k in STATUS.names}
        m = min(sd["n_clusters"], self.max_clusters)
        return host_clusters[:m * 32].numpy().view(CLUSTER), sd

    def dense_plane(self, digits_dev, n, sector, row, npads_row):
        torch = self.torch
        dense = torch.empty(npads_row * self.geom.n_time, dtype=torch.int16, device=self.device)
        stream = torch.cuda.current_stream(self.device).cuda_stream
        _check(self.lib.tpc_cf_debug_dense_plane(self.h, digits_dev.data_ptr() if n else None, n, sector, row,
                                                 dense.data_ptr(), stream))
        return dense.cpu().numpy().view(np.uint16).reshape(npads_row, self.geom.n_time)

    def set_frame_digits(self, frame_digits):
        """Launch-shape hint: the following runs are slices of a frame of `frame_digits` digits (0 = whole frames)."""
        _check(self.lib.tpc_cf_set_frame_digits(self.h, int(frame_digits)))

    def debug_set(self, **kw):
        """Test / tuning overrides of this handle (include/tpc_cf.h TPC_CF_DEBUG_*): fused_kernel ("pairs", "blocks",
        "lines" or 0), passes, block_pool, surv_cap, pads_per_unit, ctas_per_sm.  0 restores the library's choice."""
        for name, value in kw.items():
            if name == "fused_kernel" and isinstance(value, str):
                value = FUSED_KERNELS[value]
            _check(self.lib.tpc_cf_debug_set(self.h, DEBUG_KEYS[name], int(value)))

    def debug_scan_u32(self, inp, out, n, total=None):
        """The existing scan path: scratch in this handle's workspace (tpc_cf_debug_scan_u32)."""
        stream = self.torch.cuda.current_stream(self.device).cuda_stream
        _check(self.lib.tpc_cf_debug_scan_u32(self.h, inp.data_ptr() if n else None, out.data_ptr() if n else None, int(n),
                                              total.data_ptr() if total is not None else None, stream))

    def set_profiling(self, on):
        _check(self.lib.tpc_cf_set_profiling(self.h, 1 if on else 0))

    def profile_ms(self, run, which):
        return float(self.lib.tpc_cf_profile_ms(self.h, run, which))

    def last_launch_count(self):
        return int(self.lib.tpc_cf_last_launch_count(self.h))

    def last_kernel(self):
        return self.lib.tpc_cf_last_kernel(self.h).decode()

    def close(self):
        if getattr(self, "h", None) is not None:
            self.torch.cuda.synchronize(self.device)
            tpc_cf_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def to_device(digits, device="cuda:0"):
    """numpy DIGIT array -> torch uint8 device tensor (8 bytes per record)."""
    import torch
    a = np.ascontiguousarray(digits, dtype=DIGIT).view(np.uint8)
    if a.size == 0:
        return torch.empty(8, dtype=torch.uint8, device=device)
    return torch.from_numpy(a).to(device)
