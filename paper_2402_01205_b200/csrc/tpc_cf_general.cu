// tpc_cf_general.cu — general path ("T1", map in HBM): works for any digit order.
//   K1  k_scatter      digits -> dense uint16 charge map [plane][pad+2][time+2] (zero border, R2); counts bad digits (R11);
//                      verifies ascending order for free (the result of which selects the key sort, R12)
//   K2+K4 k_peaks_map  digit-centric: every digit with q >= q_peak_min gathers its 3x3 neighbourhood from the map
//                      (only cells that hold a digit can be peaks), peaks gather the 5x5 window and
//                      write their cluster to stage[j]; one ballot word per 32 digits records the peak set
//   K0  k_unscatter    stores zeros at every digit's cell: the map is zero again when the run ends
// Compaction / ordering (K3, K5) is in tpc_cf_compact.cu and shared with the fused path.
#include "tpc_cf_internal.cuh"

namespace tpccf {

thread_local const char* g_last_kernel = "";

static constexpr int kThreads = 256;

__device__ __forceinline__ size_t cell_offset(const Geo& g, uint32_t w0, uint32_t w1)
{
    const uint32_t s = w0 & 0xffu, r = (w0 >> 8) & 0xffu, p = (w0 >> 16) & 0xffu, t = w1 & 0xffffu;
    const size_t plane = (size_t)s * g.n_rows + r;
    return (plane * g.PS + (p + 2u)) * (size_t)g.TS + (t + 2u);
}

__global__ void __launch_bounds__(kThreads)
k_scatter(const uint2* __restrict__ digits, uint64_t n, Geo g, uint16_t* __restrict__ map, Counters* cnt)
{
    const uint64_t i = (uint64_t)blockIdx.x * kThreads + threadIdx.x;
    bool bad = false, unsorted = false;
    if (i < n) {
        const uint2 d = __ldg(digits + i);
        if (digit_valid(g, d.x, d.y)) {
            map[cell_offset(g, d.x, d.y)] = (uint16_t)(d.y >> 16);
        } else {
            bad = true;
        }
        if (i > 0) {
            const uint2 e = __ldg(digits + i - 1);
            unsorted = key40(e.x, e.y) > key40(d.x, d.y);
        }
    }
    // bad digits and order violations are rare: one atomic per warp that saw any (n_used = n - n_bad at the end;
    // a per-warp atomic on one counter for every warp would serialise in L2)
    const unsigned mb = __ballot_sync(0xffffffffu, bad);
    const unsigned ms = __ballot_sync(0xffffffffu, unsorted);
    if ((threadIdx.x & 31) == 0) {
        if (mb) atomicAdd(&cnt->n_bad, (unsigned long long)__popc(mb));
        if (ms) atomicOr(&cnt->unsorted, 1u);
    }
}

__global__ void __launch_bounds__(kThreads)
k_unscatter(const uint2* __restrict__ digits, uint64_t n, Geo g, uint16_t* __restrict__ map)
{
    const uint64_t i = (uint64_t)blockIdx.x * kThreads + threadIdx.x;
    if (i >= n) return;
    const uint2 d = __ldg(digits + i);
    if (digit_valid(g, d.x, d.y)) map[cell_offset(g, d.x, d.y)] = 0;
}

template <bool VAR>   // VAR: flags / cuts requested (V1..V3)
__global__ void __launch_bounds__(kThreads)
k_peaks_map(const uint2* __restrict__ digits, uint64_t n, Geo g, const uint16_t* __restrict__ map,
            uint32_t q_peak_min, uint32_t q_gate, Variant var, uint32_t* __restrict__ peakmask,
            uint4* __restrict__ stage)
{
    const uint64_t i = (uint64_t)blockIdx.x * kThreads + threadIdx.x;
    bool peak = false;
    uint2 d = make_uint2(0, 0);
    const uint16_t* c0 = nullptr;
    const int TS = (int)g.TS;
    if (i < n) {
        d = __ldg(digits + i);
        const uint32_t q = d.y >> 16;
        if (q >= q_peak_min && digit_valid(g, d.x, d.y)) {
            c0 = map + cell_offset(g, d.x, d.y);
            // R1: strict against the 4 lexicographically earlier neighbours, >= against the 4 later ones
            peak = q > (uint32_t)c0[-TS - 1] && q > (uint32_t)c0[-TS] && q > (uint32_t)c0[-TS + 1] &&
                   q > (uint32_t)c0[-1] && q >= (uint32_t)c0[1] &&
                   q >= (uint32_t)c0[TS - 1] && q >= (uint32_t)c0[TS] && q >= (uint32_t)c0[TS + 1];
        }
    }
    // K4 before the peak bit is recorded: a cluster that fails a cut (V2) is not a set bit
    if (peak) {
        int c[5][5];
#pragma unroll
        for (int a = 0; a < 5; ++a)
#pragma unroll
            for (int b = 0; b < 5; ++b) c[a][b] = (int)c0[(a - 2) * TS + (b - 2)];
        const ClusterSums sums = cluster_sums(c, q_gate);
        uint32_t fl = 0u;
        if (VAR)
            peak = cluster_variant(sums, (d.x >> 16) & 0xffu, d.y & 0xffffu, d.y >> 16, g.npads[(d.x >> 8) & 0xffu],
                                   g.n_time, var, &fl);
        if (peak) {
            const ClusterWords r = cluster_finish(sums, d.x, d.y & 0xffffu, d.y >> 16, fl);
            stage[2 * i] = r.lo;
            stage[2 * i + 1] = r.hi;
        }
    }
    const unsigned m = __ballot_sync(0xffffffffu, peak);
    if ((threadIdx.x & 31) == 0 && i < n) peakmask[i >> 5] = m;
}

__global__ void k_copy_plane(Geo g, const uint16_t* __restrict__ map, uint32_t plane, uint32_t P,
                             uint16_t* __restrict__ dense)
{
    const uint32_t T = g.n_time;
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (uint64_t)P * T) return;
    const uint32_t p = (uint32_t)(i / T), t = (uint32_t)(i % T);
    dense[i] = map[((size_t)plane * g.PS + (p + 2u)) * (size_t)g.TS + (t + 2u)];
}

static inline unsigned grid_for(uint64_t n) { return (unsigned)ceil_div_u64(n ? n : 1, kThreads); }

int launch_scatter_only(const Geo& g, const Workspace& ws, const tpc_digit* digits, uint64_t n, cudaStream_t st)
{
    if (n == 0) return 0;
    k_scatter<<<grid_for(n), kThreads, 0, st>>>((const uint2*)digits, n, g, ws.map, ws.counters);
    return 1;
}

int launch_unscatter(const Geo& g, const Workspace& ws, const tpc_digit* digits, uint64_t n, cudaStream_t st)
{
    if (n == 0) return 0;
    k_unscatter<<<grid_for(n), kThreads, 0, st>>>((const uint2*)digits, n, g, ws.map);
    return 1;
}

int launch_general_peaks(const Geo& g, const Workspace& ws, const tpc_digit* digits, uint64_t n,
                         uint32_t q_peak_min, uint32_t q_gate, const Variant& var, cudaStream_t st,
                         cudaEvent_t ev_k0, cudaEvent_t ev_k1)
{
    if (n == 0) return 0;
    k_scatter<<<grid_for(n), kThreads, 0, st>>>((const uint2*)digits, n, g, ws.map, ws.counters);
    if (ev_k0) cudaEventRecord(ev_k0, st);
    g_last_kernel = "k_peaks_map";
    if (var.active)
        k_peaks_map<true><<<grid_for(n), kThreads, 0, st>>>((const uint2*)digits, n, g, ws.map, q_peak_min, q_gate, var,
                                                            ws.peakmask, (uint4*)ws.stage);
    else
        k_peaks_map<false><<<grid_for(n), kThreads, 0, st>>>((const uint2*)digits, n, g, ws.map, q_peak_min, q_gate, var,
                                                             ws.peakmask, (uint4*)ws.stage);
    if (ev_k1) cudaEventRecord(ev_k1, st);
    return 2;
}

int launch_copy_plane(const Geo& g, const Workspace& ws, uint32_t plane, uint32_t P, uint16_t* dense,
                      cudaStream_t st)
{
    const uint64_t cells = (uint64_t)P * g.n_time;
    k_copy_plane<<<(unsigned)ceil_div_u64(cells, 256), 256, 0, st>>>(g, ws.map, plane, P, dense);
    return 1;
}

}  // namespace tpccf
