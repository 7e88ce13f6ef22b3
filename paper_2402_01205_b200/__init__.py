"""B200-native TPC cluster finder (arXiv:2402.01205, step named in PAPER.md:57): C-ABI library + thin binding.

    from paper_2402_01205_b200 import ClusterFinder, ClusterCoder, FrontEndFilter
The CUDA library (libtpc_cf.so) is loaded on first use; there is no CPU fallback.
"""
from .binding import (CLUSTER, CLUSTER_FLAGS, CUT_SINGLE_PAD, CUT_SINGLE_TIME, DIGIT, DIGITS_SORTED, EXPORTS,
                      F_EDGE_PAD, F_EDGE_TIME, F_SATURATED, F_SHARED, F_SINGLE_PAD, F_SINGLE_TIME, FORCE_GENERAL, SHARE_CHARGE, STATUS, ClusterFinder, Geometry, Out,
                      Params, TpcCfError, load, make_geometry, scan_u32_static, to_device, tpc_cf_create,
                      tpc_cf_destroy, tpc_cf_run, tpc_cf_workspace_bytes)

from .ec_binding import (EC_ERR_CAPACITY, EC_ERR_CONTAINER, EC_ERR_QTOT, EC_ERR_UNSORTED, EC_EXPORTS, EC_STATUS,
                         ClusterCoder, clusters_to_device, tpc_ec_create, tpc_ec_decode, tpc_ec_destroy,
                         tpc_ec_encode, tpc_ec_max_encoded_bytes, tpc_ec_workspace_bytes)

from .fe_binding import (FE_DEFAULTS, FE_EXPORTS, FE_OVF_OUTPUT, FE_OVF_PLANE, FE_STATUS, FeParams, FrontEndFilter,
                         tpc_fe_create, tpc_fe_destroy, tpc_fe_pad_stride, tpc_fe_run, tpc_fe_workspace_bytes)

from .shard import ShardedClusterFinder, gather_records, plane_counts, plane_partition

__all__ = ["ShardedClusterFinder", "gather_records", "plane_counts", "plane_partition", "FE_DEFAULTS", "FE_EXPORTS", "FE_OVF_OUTPUT", "FE_OVF_PLANE", "FE_STATUS", "FeParams", "FrontEndFilter",
           "tpc_fe_create", "tpc_fe_destroy", "tpc_fe_pad_stride", "tpc_fe_run", "tpc_fe_workspace_bytes",
           "EC_ERR_CAPACITY", "EC_ERR_CONTAINER", "EC_ERR_QTOT", "EC_ERR_UNSORTED", "EC_EXPORTS", "EC_STATUS",
           "ClusterCoder", "clusters_to_device", "tpc_ec_create", "tpc_ec_decode", "tpc_ec_destroy", "tpc_ec_encode",
           "tpc_ec_max_encoded_bytes", "tpc_ec_workspace_bytes",
           "CLUSTER", "DIGIT", "STATUS", "DIGITS_SORTED", "FORCE_GENERAL", "CLUSTER_FLAGS", "CUT_SINGLE_PAD",
           "CUT_SINGLE_TIME", "F_EDGE_PAD", "F_EDGE_TIME", "F_SINGLE_PAD", "F_SINGLE_TIME", "F_SATURATED", "F_SHARED", "SHARE_CHARGE", "EXPORTS", "ClusterFinder", "Geometry",
           "Out", "Params", "TpcCfError", "load", "make_geometry", "scan_u32_static", "to_device", "tpc_cf_create", "tpc_cf_destroy",
           "tpc_cf_run", "tpc_cf_workspace_bytes"]
