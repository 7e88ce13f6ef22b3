"""B200-native TPC cluster finder (arXiv:2402.01205, step named in PAPER.md:57): C-ABI library + thin binding.

    from paper_2402_01205_b200 import ClusterFinder
The CUDA library (libtpc_cf.so) is loaded on first use; there is no CPU fallback.
"""
from .binding import (CLUSTER, CLUSTER_FLAGS, CUT_SINGLE_PAD, CUT_SINGLE_TIME, DIGIT, DIGITS_SORTED, EXPORTS,
                      F_EDGE_PAD, F_EDGE_TIME, F_SATURATED, F_SINGLE_PAD, F_SINGLE_TIME, FORCE_GENERAL, STATUS, ClusterFinder, Geometry, Out,
                      Params, TpcCfError, load, make_geometry, to_device, tpc_cf_create, tpc_cf_destroy,
                      tpc_cf_run, tpc_cf_workspace_bytes)

__all__ = ["CLUSTER", "DIGIT", "STATUS", "DIGITS_SORTED", "FORCE_GENERAL", "CLUSTER_FLAGS", "CUT_SINGLE_PAD",
           "CUT_SINGLE_TIME", "F_EDGE_PAD", "F_EDGE_TIME", "F_SINGLE_PAD", "F_SINGLE_TIME", "F_SATURATED", "EXPORTS", "ClusterFinder", "Geometry",
           "Out", "Params", "TpcCfError", "load", "make_geometry", "to_device", "tpc_cf_create", "tpc_cf_destroy",
           "tpc_cf_run", "tpc_cf_workspace_bytes"]
