"""Thin ctypes binding of the C ABI in include/tpc_ec.h (entropy coder of the cluster stream, "TPC-EC v1"; step named
in PAPER.md:55, 57) — argument marshalling only.

Symbolisation, statistics, rANS coding, container layout, decoding and record rebuild all run in the CUDA kernels of
libtpc_cf.so (csrc/tpc_ec.cu).  PyTorch is used for device memory and streams.  No CPU fallback.
"""
import ctypes

import numpy as np

from .binding import CLUSTER, TpcCfError, load

EC_STATUS = np.dtype([("n_clusters", "<u8"), ("bytes", "<u8"), ("error", "<u4"), ("rsv", "<u4")])
assert EC_STATUS.itemsize == 24
EC_ERR_UNSORTED, EC_ERR_CAPACITY, EC_ERR_CONTAINER, EC_ERR_QTOT = 1, 2, 4, 8

EC_EXPORTS = ["tpc_ec_workspace_bytes", "tpc_ec_max_encoded_bytes", "tpc_ec_create", "tpc_ec_encode", "tpc_ec_decode",
              "tpc_ec_last_launch_count", "tpc_ec_destroy"]

_typed = False


def _lib():
    global _typed
    lib = load()
    if not _typed:
        u32, u64, vp = ctypes.c_uint32, ctypes.c_uint64, ctypes.c_void_p
        lib.tpc_ec_workspace_bytes.restype = ctypes.c_size_t
        lib.tpc_ec_workspace_bytes.argtypes = [u32, u32, u64]
        lib.tpc_ec_max_encoded_bytes.restype = u64
        lib.tpc_ec_max_encoded_bytes.argtypes = [u32, u32, u64]
        lib.tpc_ec_create.restype = ctypes.c_int
        lib.tpc_ec_create.argtypes = [ctypes.POINTER(vp), u32, u32, u64, vp, ctypes.c_size_t]
        lib.tpc_ec_encode.restype = ctypes.c_int
        lib.tpc_ec_encode.argtypes = [vp, vp, u64, vp, u64, vp, vp]
        lib.tpc_ec_decode.restype = ctypes.c_int
        lib.tpc_ec_decode.argtypes = [vp, vp, u64, u64, vp, u64, vp, vp]
        lib.tpc_ec_last_launch_count.restype = ctypes.c_int
        lib.tpc_ec_last_launch_count.argtypes = [vp]
        lib.tpc_ec_destroy.restype = ctypes.c_int
        lib.tpc_ec_destroy.argtypes = [vp]
        _typed = True
    return lib


def _check(rc):
    if rc != 0:
        raise TpcCfError(rc, load().tpc_cf_strerror(rc).decode())


def tpc_ec_workspace_bytes(n_sectors, n_rows, max_clusters):
    return int(_lib().tpc_ec_workspace_bytes(n_sectors, n_rows, max_clusters))


def tpc_ec_max_encoded_bytes(n_sectors, n_rows, n):
    return int(_lib().tpc_ec_max_encoded_bytes(n_sectors, n_rows, n))


def tpc_ec_create(n_sectors, n_rows, max_clusters, workspace_ptr, workspace_bytes):
    h = ctypes.c_void_p()
    _check(_lib().tpc_ec_create(ctypes.byref(h), n_sectors, n_rows, max_clusters, workspace_ptr, workspace_bytes))
    return h


def tpc_ec_encode(h, clusters_ptr, n, out_ptr, out_capacity, status_ptr, stream_ptr):
    _check(_lib().tpc_ec_encode(h, clusters_ptr, n, out_ptr, out_capacity, status_ptr, stream_ptr))


def tpc_ec_decode(h, in_ptr, in_bytes, n, clusters_ptr, capacity, status_ptr, stream_ptr):
    _check(_lib().tpc_ec_decode(h, in_ptr, in_bytes, n, clusters_ptr, capacity, status_ptr, stream_ptr))


def tpc_ec_destroy(h):
    _check(_lib().tpc_ec_destroy(h))


class ClusterCoder:
    """Owns the torch allocations one tpc_ec handle needs (workspace, status).  encode() / decode() only enqueue on
    the current torch stream; the *_result() calls synchronise and read back."""

    def __init__(self, n_sectors, n_rows, max_clusters, device="cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("tpc_ec needs a CUDA device; there is no CPU fallback")
        self.torch = torch
        self.device = torch.device(device)
        self.n_sectors, self.n_rows, self.max_clusters = int(n_sectors), int(n_rows), int(max_clusters)
        nbytes = tpc_ec_workspace_bytes(self.n_sectors, self.n_rows, self.max_clusters)
        if nbytes == 0:
            raise TpcCfError(-2, "invalid geometry or capacity")
        self.workspace_bytes = nbytes
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        self._ws_ptr = (self.workspace.data_ptr() + 255) & ~255
        self.status = torch.zeros(EC_STATUS.itemsize, dtype=torch.uint8, device=self.device)
        self.h = tpc_ec_create(self.n_sectors, self.n_rows, self.max_clusters, self._ws_ptr, nbytes)

    def _stream(self):
        return self.torch.cuda.current_stream(self.device).cuda_stream

    def max_encoded_bytes(self, n):
        return tpc_ec_max_encoded_bytes(self.n_sectors, self.n_rows, n)

    def encode(self, clusters_dev, n, out_dev, out_capacity=None):
        """clusters_dev: torch uint8 device tensor of n 32-byte records; out_dev: torch uint8 device tensor."""
        cap = int(out_dev.numel() if out_capacity is None else out_capacity)
        tpc_ec_encode(self.h, clusters_dev.data_ptr() if n else None, int(n), out_dev.data_ptr(), cap,
                      self.status.data_ptr(), self._stream())

    def decode(self, in_dev, in_bytes, n, clusters_dev, capacity=None):
        cap = int(clusters_dev.numel() // 32 if capacity is None else capacity)
        tpc_ec_decode(self.h, in_dev.data_ptr(), int(in_bytes), int(n), clusters_dev.data_ptr() if n else None, cap,
                      self.status.data_ptr(), self._stream())

    def read_status(self):
        st = self.status.cpu().numpy().view(EC_STATUS)[0]
        return {k: int(st[k]) for k in ("n_clusters", "bytes", "error")}

    def last_launch_count(self):
        return int(_lib().tpc_ec_last_launch_count(self.h))

    def close(self):
        if getattr(self, "h", None) is not None:
            self.torch.cuda.synchronize(self.device)
            tpc_ec_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def clusters_to_device(clusters, device="cuda:0"):
    """numpy CLUSTER array -> torch uint8 device tensor (32 bytes per record)."""
    import torch
    a = np.ascontiguousarray(clusters, dtype=CLUSTER).view(np.uint8)
    if a.size == 0:
        return torch.empty(32, dtype=torch.uint8, device=device)
    return torch.from_numpy(a.copy()).to(device)
