"""Thin ctypes binding of the C ABI in include/tpc_fe.h (front-end filter "TPC-FE v1": common-mode correction, ion-tail
cancellation, zero suppression; step named in PAPER.md:57) — argument marshalling only.

Every step runs in the CUDA kernels of libtpc_cf.so (csrc/tpc_fe.cu).  PyTorch is used for device memory and streams.
No CPU fallback.
"""
import ctypes

import numpy as np

from .binding import Geometry, TpcCfError, load, make_geometry

FE_STATUS = np.dtype([("n_digits", "<u8"), ("overflow", "<u4"), ("rsv", "<u4")])
assert FE_STATUS.itemsize == 16
FE_OVF_PLANE, FE_OVF_OUTPUT = 1, 2
FE_DEFAULTS = dict(zs_threshold=2, cm_quiet4=12, cm_min_pads=8, it_decay_shift=6, it_kappa_shift=8)

FE_EXPORTS = ["tpc_fe_pad_stride", "tpc_fe_workspace_bytes", "tpc_fe_create", "tpc_fe_run", "tpc_fe_last_launch_count",
              "tpc_fe_set_profiling", "tpc_fe_profile_ms", "tpc_fe_destroy"]


class FeParams(ctypes.Structure):
    _fields_ = [("zs_threshold", ctypes.c_uint16), ("cm_quiet4", ctypes.c_uint16), ("cm_min_pads", ctypes.c_uint16),
                ("it_decay_shift", ctypes.c_uint8), ("it_kappa_shift", ctypes.c_uint8)]


_typed = False


def _lib():
    global _typed
    lib = load()
    if not _typed:
        u32, u64, vp = ctypes.c_uint32, ctypes.c_uint64, ctypes.c_void_p
        lib.tpc_fe_pad_stride.restype = u32
        lib.tpc_fe_pad_stride.argtypes = [u32]
        lib.tpc_fe_workspace_bytes.restype = ctypes.c_size_t
        lib.tpc_fe_workspace_bytes.argtypes = [ctypes.POINTER(Geometry), u64]
        lib.tpc_fe_create.restype = ctypes.c_int
        lib.tpc_fe_create.argtypes = [ctypes.POINTER(vp), ctypes.POINTER(Geometry), u64, vp, ctypes.c_size_t]
        lib.tpc_fe_run.restype = ctypes.c_int
        lib.tpc_fe_run.argtypes = [vp, vp, vp, ctypes.POINTER(FeParams), vp, u64, vp, vp]
        lib.tpc_fe_last_launch_count.restype = ctypes.c_int
        lib.tpc_fe_last_launch_count.argtypes = [vp]
        lib.tpc_fe_set_profiling.restype = ctypes.c_int
        lib.tpc_fe_set_profiling.argtypes = [vp, ctypes.c_int]
        lib.tpc_fe_profile_ms.restype = ctypes.c_float
        lib.tpc_fe_profile_ms.argtypes = [vp]
        lib.tpc_fe_destroy.restype = ctypes.c_int
        lib.tpc_fe_destroy.argtypes = [vp]
        _typed = True
    return lib


def _check(rc):
    if rc != 0:
        raise TpcCfError(rc, load().tpc_cf_strerror(rc).decode())


def tpc_fe_pad_stride(max_pads):
    return int(_lib().tpc_fe_pad_stride(max_pads))


def tpc_fe_workspace_bytes(geom, max_digits_per_plane):
    return int(_lib().tpc_fe_workspace_bytes(ctypes.byref(geom), max_digits_per_plane))


def tpc_fe_create(geom, max_digits_per_plane, workspace_ptr, workspace_bytes):
    h = ctypes.c_void_p()
    _check(_lib().tpc_fe_create(ctypes.byref(h), ctypes.byref(geom), max_digits_per_plane, workspace_ptr,
                                workspace_bytes))
    return h


def tpc_fe_run(h, raw_ptr, ped4_ptr, params, out_ptr, capacity, status_ptr, stream_ptr):
    _check(_lib().tpc_fe_run(h, raw_ptr, ped4_ptr, ctypes.byref(params), out_ptr, capacity, status_ptr, stream_ptr))


def tpc_fe_destroy(h):
    _check(_lib().tpc_fe_destroy(h))


class FrontEndFilter:
    """Owns the torch allocations one tpc_fe handle needs (workspace, status).  run() only enqueues on the current
    torch stream; read_status() synchronises and reads back."""

    def __init__(self, n_sectors, n_rows, max_pads, n_time, npads=None, max_digits_per_plane=1 << 16, device="cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("tpc_fe needs a CUDA device; there is no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        self.geom, self._keep = make_geometry(n_sectors, n_rows, max_pads, n_time, npads)
        self.n_planes, self.n_time = int(n_sectors) * int(n_rows), int(n_time)
        self.W = tpc_fe_pad_stride(max_pads)
        nbytes = tpc_fe_workspace_bytes(self.geom, int(max_digits_per_plane))
        if nbytes == 0:
            raise TpcCfError(-2, "invalid geometry or capacity")
        self.workspace_bytes = nbytes
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        ws_ptr = (self.workspace.data_ptr() + 255) & ~255
        self.status = torch.zeros(FE_STATUS.itemsize, dtype=torch.uint8, device=self.device)
        with torch.cuda.device(self.device):
            self.h = tpc_fe_create(self.geom, int(max_digits_per_plane), ws_ptr, nbytes)

    def run(self, raw_dev, ped4_dev, out_dev, capacity=None, **params):
        """raw_dev: torch device tensor of uint16 samples [n_planes, n_time, W] (any 2-byte dtype); ped4_dev:
        [n_planes, W]; out_dev: torch uint8 device tensor receiving 8-byte digits."""
        pr = dict(FE_DEFAULTS)
        pr.update(params)
        need = self.n_planes * self.n_time * self.W * 2
        if raw_dev.numel() * raw_dev.element_size() < need or \
                ped4_dev.numel() * ped4_dev.element_size() < self.n_planes * self.W * 2:
            raise ValueError("raw / ped4 smaller than the geometry")
        cap = int(out_dev.numel() * out_dev.element_size() // 8 if capacity is None else capacity)
        tpc_fe_run(self.h, raw_dev.data_ptr(), ped4_dev.data_ptr(), FeParams(**pr), out_dev.data_ptr(), cap,
                   self.status.data_ptr(), self.torch.cuda.current_stream(self.device).cuda_stream)

    def read_status(self):
        st = self.status.cpu().numpy().view(FE_STATUS)[0]
        return {"n_digits": int(st["n_digits"]), "overflow": int(st["overflow"])}

    def last_launch_count(self):
        return int(_lib().tpc_fe_last_launch_count(self.h))

    def set_profiling(self, on):
        _check(_lib().tpc_fe_set_profiling(self.h, 1 if on else 0))

    def profile_ms(self):
        """milliseconds of the dominant kernel (k_fe_filter) in the last run; waits for it"""
        return float(_lib().tpc_fe_profile_ms(self.h))

    def close(self):
        if getattr(self, "h", None) is not None:
            self.torch.cuda.synchronize(self.device)
            tpc_fe_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
