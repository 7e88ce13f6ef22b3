"""Seeded synthetic cluster streams for the entropy-coder tests and bench (input generator only: none of the coder's
arithmetic lives here).  Shared by the oracle's pins and the CUDA parity tests.

Recipe: keys drawn uniformly from the (sector,row,pad,time) lattice and made unique and ascending; fields drawn like
cluster-finder output at BASELINE.json's cluster model (qtot >= qmax, centroids inside the 5x5 window, sigmas of the
order of a pad / time bin)."""
import numpy as np

CLUSTER = np.dtype([("sector", "u1"), ("row", "u1"), ("pad", "u1"), ("flags", "u1"),
                    ("time", "<u2"), ("qmax", "<u2"), ("qtot", "<u4"),
                    ("pad_mean", "<f4"), ("time_mean", "<f4"),
                    ("sigma_pad", "<f4"), ("sigma_time", "<f4"), ("rsv", "<u4")])


def synthetic_clusters(rng, n_sectors, n_rows, n, max_pads=138, n_time=2000):
    """sorted, unique keys; fields drawn like cluster-finder output (qtot >= qmax, offsets inside the 5x5 window)"""
    key = np.unique(rng.integers(0, n_sectors * n_rows * max_pads * n_time, size=n))
    cl = np.zeros(key.shape[0], dtype=CLUSTER)
    cl["time"] = key % n_time
    cl["pad"] = (key // n_time) % max_pads
    cl["row"] = (key // (n_time * max_pads)) % n_rows
    cl["sector"] = key // (n_time * max_pads * n_rows)
    m = key.shape[0]
    cl["qmax"] = np.minimum(65535, 4 + rng.geometric(0.05, size=m))
    cl["qtot"] = cl["qmax"].astype(np.uint32) + rng.geometric(0.01, size=m).astype(np.uint32) - 1
    cl["flags"] = rng.choice([0, 0, 0, 1, 4, 12], size=m)
    cl["pad_mean"] = (cl["pad"] + rng.normal(0, 0.3, size=m).clip(-1.9, 1.9)).astype(np.float32)
    cl["time_mean"] = (cl["time"] + rng.normal(0, 0.4, size=m).clip(-1.9, 1.9)).astype(np.float32)
    cl["sigma_pad"] = np.abs(rng.normal(0.6, 0.2, size=m)).clip(0, 1.9).astype(np.float32)
    cl["sigma_time"] = np.abs(rng.normal(0.9, 0.3, size=m)).clip(0, 1.9).astype(np.float32)
    return cl
