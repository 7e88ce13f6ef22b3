// placeholder until the fused path lands
#include "tpc_cf_internal.cuh"
namespace tpccf {
int launch_fused_sorted(const Geo&, const Workspace&, const tpc_digit*, uint64_t, uint32_t, uint32_t, cudaStream_t,
                        cudaEvent_t, cudaEvent_t) { return TPC_CF_E_PARAMS; }
}
