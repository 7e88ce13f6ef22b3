// tpc_cf_share.cu — K6: charge sharing between overlapping clusters (variant V4, include/tpc_cf.h; SURVEY.md §8(f)
// NEXT #1, second half; the paper names no sharing rule — PAPER.md:21 only says that different cuts are used).
//
// A post-pass over the ORDERED output of any of the three paths.  V4 keeps the cluster list, the cuts and flags 1..16 of
// the unshared run, so the peak-charge map A(x) of the definition is the output array itself:
//   k_share_index          first cluster of every (plane, pad) line, by binary search on the ordered records (one thread
//                          per line) -> ws.line_cnt (idle once the records are in place); and the (time | qmax << 16)
//                          words of the records packed into a dense array (ws.stage, idle too): the peak list the next
//                          kernel searches, 4 bytes per cluster, read-only
//   k_share_find           one thread per cluster: is another peak within +-4 pads / +-4 time bins (a window reaches 2
//                          cells, a cell is claimed from 2 cells away)?  Own line: the records next to it; the other
//                          eight lines: one lower bound each in the peak list.  Most clusters have none and stay as they
//                          are, bit for bit; the others are queued (warp-aggregated append, near input order).
//   k_share_apply<MAP>     one thread per queued cluster: the qMax of every such neighbour is added into D(x) for the
//                          cells of the 5x5 window its own window covers (25 registers); the window is read again — from
//                          the sorted digits through the fused path's line index (five lower bounds on time, side by side),
//                          or from the charge map of the general path (MAP) — and every cell that enters (gates on raw
//                          charges, R3 / R4) enters with c' = floor(64 * Q * A(peak) / D), two 32-bit divisions.
// Sums over c' are below 25 * 65535 * 64 * 4 < 2^29; the variance numerator S0' S2' - S1'^2 < 2^56 is exact in int64.
// Only the sums and what follows from them are rewritten (qtot, centroids, sigmas, flag SHARED), each record by the lane
// that owns it; nothing a lane reads of another record is ever written in this pass.
#include "tpc_cf_internal.cuh"

namespace tpccf {

static constexpr int kShareThreads = 128;

__device__ __forceinline__ uint32_t cluster_line(const Geo& g, uint32_t w0)
{
    return ((w0 & 0xffu) * g.n_rows + ((w0 >> 8) & 0xffu)) * g.LS + ((w0 >> 16) & 0xffu);
}

__device__ __forceinline__ uint64_t clusters_written(const tpc_cf_status* status, uint64_t capacity)
{
    if (status->path == 0u) return 0;                         // no output (false promise / duplicate cell)
    const uint64_t n = status->n_clusters;
    return n < capacity ? n : capacity;
}

__global__ void __launch_bounds__(256)
k_share_index(const uint4* __restrict__ out, const tpc_cf_status* __restrict__ status, uint64_t capacity, Geo g,
              uint32_t n_lines, uint32_t* __restrict__ line_off, uint32_t* __restrict__ peaks_y)
{
    const uint32_t gtid = blockIdx.x * blockDim.x + threadIdx.x, stride = gridDim.x * blockDim.x;
    const uint32_t n = (uint32_t)clusters_written(status, capacity);
    for (uint32_t i = gtid; i < n; i += stride) peaks_y[i] = out[2 * (size_t)i].y;
    for (uint32_t l = gtid; l <= n_lines; l += stride) {
        uint32_t lo = 0u, hi = n;                             // first record whose line is >= l
        while (lo < hi) {
            const uint32_t mid = (lo + hi) >> 1;
            if (cluster_line(g, out[2 * (size_t)mid].x) < l) lo = mid + 1u; else hi = mid;
        }
        line_off[l] = lo;
    }
}

// first index in [lo, hi) of the ascending time fields of y[] that is >= tmin (tmin may be negative)
__device__ __forceinline__ uint32_t lower_bound_time(const uint32_t* __restrict__ y, uint32_t lo, uint32_t hi, int tmin)
{
    while (lo < hi) {
        const uint32_t mid = (lo + hi) >> 1;
        if ((int)(__ldg(y + mid) & 0xffffu) < tmin) lo = mid + 1u; else hi = mid;
    }
    return lo;
}

// the cluster ranges of lines p-4 .. p+4 of a plane: off[k] = first cluster of line p - 4 + k (k = 0 .. 9; empty ranges
// outside the plane)
__device__ __forceinline__ void neighbour_ranges(const uint32_t* __restrict__ line_off, uint32_t l, int p, int P,
                                                 uint32_t (&off)[10])
{
#pragma unroll
    for (int k = 0; k < 10; ++k) {
        const int pp = p - 4 + k;
        off[k] = __ldg(line_off + (pp < 0 ? l - (uint32_t)p : (pp > P ? l - (uint32_t)p + (uint32_t)P : l - 4u + (uint32_t)k)));
    }
}

__global__ void __launch_bounds__(256)
k_share_find(const uint4* __restrict__ out, const tpc_cf_status* __restrict__ status, uint64_t capacity, Geo g,
             const uint32_t* __restrict__ line_off, const uint32_t* __restrict__ peaks_y,
             uint32_t* __restrict__ queue, Counters* cnt)
{
    const uint32_t n = (uint32_t)clusters_written(status, capacity);
    const int lane = threadIdx.x & 31;
    const uint32_t stride = gridDim.x * blockDim.x;
    for (uint32_t i0 = (blockIdx.x * blockDim.x + threadIdx.x) & ~31u; i0 < n; i0 += stride) {
        const uint32_t i = i0 + (uint32_t)lane;
        bool any = false;
        if (i < n) {
            const uint32_t w0 = out[2 * (size_t)i].x, y = __ldg(peaks_y + i);
            const uint32_t l = cluster_line(g, w0);
            const int p = (int)((w0 >> 16) & 0xffu), t = (int)(y & 0xffffu);
            const int P = (int)g.npads[(w0 >> 8) & 0xffu];
            uint32_t off[10];
            neighbour_ranges(line_off, l, p, P, off);
            // own line: the records next to this one
            if (i > off[4] && t - (int)(__ldg(peaks_y + i - 1u) & 0xffffu) <= 4) any = true;
            if (i + 1u < off[5] && (int)(__ldg(peaks_y + i + 1u) & 0xffffu) - t <= 4) any = true;
            // the other eight lines: first peak with time >= t - 4, the eight searches side by side
            uint32_t lo[9], hi[9];
#pragma unroll
            for (int k = 0; k < 9; ++k) { lo[k] = off[k]; hi[k] = (k == 4 || any) ? off[k] : off[k + 1]; }
            for (bool more = true; more;) {
                more = false;
#pragma unroll
                for (int k = 0; k < 9; ++k) {
                    if (k == 4) continue;
                    const bool go = lo[k] < hi[k];
                    const uint32_t mid = (lo[k] + hi[k]) >> 1;
                    const int tm = go ? (int)(__ldg(peaks_y + mid) & 0xffffu) : 0;
                    if (go) { if (tm < t - 4) lo[k] = mid + 1u; else hi[k] = mid; }
                    more |= go;
                }
            }
#pragma unroll
            for (int k = 0; k < 9; ++k) {
                if (k == 4) continue;
                const bool in = !any && lo[k] < off[k + 1];
                const int tn = in ? (int)(__ldg(peaks_y + lo[k]) & 0xffffu) : 0x7fffffff;
                if (in && tn - t <= 4) any = true;
            }
        }
        const unsigned m = __ballot_sync(0xffffffffu, any);
        if (m) {
            uint32_t base = 0u;
            if (lane == 0) base = atomicAdd(&cnt->n_share, (unsigned)__popc(m));
            base = __shfl_sync(0xffffffffu, base, 0);
            if (any) queue[base + (uint32_t)__popc(m & ((1u << lane) - 1u))] = i;
        }
    }
}

template <bool MAP>
__global__ void __launch_bounds__(kShareThreads)
k_share_apply(uint4* __restrict__ out, Geo g, const uint32_t* __restrict__ line_off,
              const uint32_t* __restrict__ peaks_y, const uint32_t* __restrict__ queue, const Counters* __restrict__ cnt,
              const uint2* __restrict__ digits, const uint32_t* __restrict__ line_start,
              const uint16_t* __restrict__ map, uint32_t q_gate, uint32_t want_flags)
{
    const uint32_t n_q = cnt->n_share;
    const int T = (int)g.n_time;
    for (uint32_t qi = blockIdx.x * blockDim.x + threadIdx.x; qi < n_q; qi += gridDim.x * blockDim.x) {
        {   // (one queued cluster)
            const uint32_t i = queue[qi];
            const uint32_t w0 = out[2 * (size_t)i].x;         // (this record is written by this thread only)
            const uint32_t y = __ldg(peaks_y + i);
            const uint32_t l = cluster_line(g, w0);
            const uint32_t plane = l / g.LS;
            const int p = (int)((w0 >> 16) & 0xffu), t = (int)(y & 0xffffu);
            const int P = (int)g.npads[(w0 >> 8) & 0xffu];
            const uint32_t Az = y >> 16;
            uint32_t off[10];
            neighbour_ranges(line_off, l, p, P, off);
            uint32_t D[5][5];                                 // summed peak charges of the windows that hold cell (a, b)
#pragma unroll
            for (int a = 0; a < 5; ++a)
#pragma unroll
                for (int b = 0; b < 5; ++b) D[a][b] = Az;
            {
                // the nine lower bounds (first peak of the line with time >= t - 4) side by side: nine independent chains
                // of loads instead of one after the other
                uint32_t lo[9], hi[9];
#pragma unroll
                for (int k = 0; k < 9; ++k) { lo[k] = off[k]; hi[k] = off[k + 1]; }
                for (bool more = true; more;) {
                    more = false;
#pragma unroll
                    for (int k = 0; k < 9; ++k) {
                        const bool go = lo[k] < hi[k];
                        const uint32_t mid = (lo[k] + hi[k]) >> 1;
                        const int tm = go ? (int)(__ldg(peaks_y + mid) & 0xffffu) : 0;
                        if (go) { if (tm < t - 4) lo[k] = mid + 1u; else hi[k] = mid; }
                        more |= go;
                    }
                }
#pragma unroll
                for (int k = 0; k < 9; ++k) {
                    const int dp = k - 4;
                    for (uint32_t j = lo[k]; j < off[k + 1]; ++j) {
                        const uint32_t y2 = __ldg(peaks_y + j);
                        const int dt = (int)(y2 & 0xffffu) - t;
                        if (dt > 4) break;
                        if (dp == 0 && dt == 0) continue;
                        const uint32_t q2 = y2 >> 16;
#pragma unroll
                        for (int b = 0; b < 5; ++b) {
                            const uint32_t add = (dt - (b - 2) <= 2 && dt - (b - 2) >= -2) ? q2 : 0u;
#pragma unroll
                            for (int a = 0; a < 5; ++a)
                                if (dp - (a - 2) <= 2 && dp - (a - 2) >= -2) D[a][b] += add;   // (compile-time test)
                        }
                    }
                }
            }

            // the 5x5 window again (zero outside the plane, R2)
            uint32_t c[5][5];
#pragma unroll
            for (int a = 0; a < 5; ++a)
#pragma unroll
                for (int b = 0; b < 5; ++b) c[a][b] = 0u;
            if (MAP) {
#pragma unroll
                for (int a = 0; a < 5; ++a) {
                    const int pp = p + a - 2;
                    if (pp < 0 || pp >= P) continue;
                    const uint16_t* line = map + ((size_t)plane * g.PS + (size_t)(pp + 2)) * (size_t)g.TS + (size_t)t;
#pragma unroll
                    for (int b = 0; b < 5; ++b) c[a][b] = (uint32_t)line[b];       // cell t + b - 2 sits at index t + b
                }
            } else {
                // five lower bounds on the digit lines (first digit with time >= t - 2), side by side as above
                const int tmin = t - 2;
                uint32_t lo[5], hi[5], le[5];
#pragma unroll
                for (int a = 0; a < 5; ++a) {
                    const int pp = p + a - 2;
                    const bool ok = pp >= 0 && pp < P;
                    lo[a] = ok ? line_start[l + (uint32_t)a - 2u] : 0u;
                    le[a] = ok ? line_start[l + (uint32_t)a - 1u] : 0u;
                    hi[a] = le[a];
                }
                for (bool more = true; more;) {
                    more = false;
#pragma unroll
                    for (int a = 0; a < 5; ++a) {
                        const bool go = lo[a] < hi[a];
                        const uint32_t mid = (lo[a] + hi[a]) >> 1;
                        const int tm = go ? (int)(__ldg(&digits[mid].y) & 0xffffu) : 0;
                        if (go) { if (tm < tmin) lo[a] = mid + 1u; else hi[a] = mid; }
                        more |= go;
                    }
                }
                // times ascend strictly within a line: the cells t-2 .. t+2 are among the next five digits
#pragma unroll
                for (int a = 0; a < 5; ++a) {
#pragma unroll
                    for (int e = 0; e < 5; ++e) {
                        const uint32_t j = lo[a] + (uint32_t)e;
                        const bool in = j < le[a];
                        const uint32_t yd = in ? __ldg(&digits[j].y) : 0xffffu;
                        const int tt = (int)(yd & 0xffffu);
                        const int k = (in && tt < T) ? tt - tmin : 5;      // (times >= n_time are no cells, R11)
#pragma unroll
                        for (int b = 0; b < 5; ++b) c[a][b] = k == b ? (yd >> 16) : c[a][b];
                    }
                }
            }

            long long S0 = 0, S1p = 0, S1t = 0, S2p = 0, S2t = 0;
            bool shared = false;
#pragma unroll
            for (int a = 0; a < 5; ++a) {
#pragma unroll
                for (int b = 0; b < 5; ++b) {
                    const int dp = a - 2, dt = b - 2;
                    uint32_t v = c[a][b];
                    if (dp == 2 || dp == -2 || dt == 2 || dt == -2) {         // outer ring: gated (R3, R4)
                        const int ga = a - (dp > 0) + (dp < 0), gb = b - (dt > 0) + (dt < 0);
                        if (c[ga][gb] < q_gate) v = 0u;
                    }
                    uint32_t s = v << 6;                      // 64 Q: the cell is this cluster's alone (v < 2^16)
                    if (v != 0u && D[a][b] != Az) {
                        // floor(64 v Az / D) with v Az < 2^32, D < 2^21: 64 (v Az / D) + 64 (v Az mod D) / D
                        shared = true;
                        const uint32_t num = v * Az, d = D[a][b];
                        const uint32_t q1 = num / d, r1 = num - q1 * d;
                        s = (q1 << 6) + (r1 << 6) / d;
                    }
                    const long long sl = (long long)s;
                    S0 += sl; S1p += sl * dp; S1t += sl * dt; S2p += sl * (dp * dp); S2t += sl * (dt * dt);
                }
            }
            if (!shared) continue;                            // every cell with charge is this cluster's alone

            float pad_mean = (float)p, time_mean = (float)t, sp = 0.f, st = 0.f;
            if (S0 > 0) {
                const float r0 = __fdividef(1.f, (float)S0);
                const long long np = S0 * S2p - S1p * S1p, nt = S0 * S2t - S1t * S1t;
                const float fp = (float)np, ft = (float)nt;
                pad_mean += (float)S1p * r0;
                time_mean += (float)S1t * r0;
                sp = np > 0 ? fp * rsqrtf(fp) * r0 : 0.f;
                st = nt > 0 ? ft * rsqrtf(ft) * r0 : 0.f;
            }
            uint4 lo4, hi4;
            lo4.x = want_flags ? (w0 | (TPC_CF_F_SHARED << 24)) : w0;
            lo4.y = y;
            lo4.z = (uint32_t)((S0 + 32) >> 6);
            lo4.w = __float_as_uint(pad_mean);
            hi4.x = __float_as_uint(time_mean);
            hi4.y = __float_as_uint(sp);
            hi4.z = __float_as_uint(st);
            hi4.w = 0u;
            out[2 * (size_t)i] = lo4;
            out[2 * (size_t)i + 1] = hi4;
        }
    }
}

// digits != nullptr: sorted digits + ws.line_start (fused paths); else the charge map of the general path (still filled).
int launch_share_charge(const Geo& g, const Workspace& ws, const tpc_digit* digits, tpc_cluster* out, uint64_t capacity,
                        const tpc_cf_status* status, uint32_t q_gate, uint32_t vflags, uint64_t max_digits, cudaStream_t st)
{
    if (capacity == 0) return 0;
    const uint32_t n_lines = g.n_planes * g.LS;
    // n_clusters <= n_digits <= max_digits: the peak list and the queue take 8 of the 32 staging bytes per digit
    uint32_t* peaks_y = (uint32_t*)ws.stage;
    uint32_t* queue = peaks_y + max_digits;
    k_share_index<<<148 * 8, 256, 0, st>>>((const uint4*)out, status, capacity, g, n_lines, ws.line_cnt, peaks_y);
    k_share_find<<<148 * 8, 256, 0, st>>>((const uint4*)out, status, capacity, g, ws.line_cnt, peaks_y, queue, ws.counters);
    const uint32_t want_flags = (vflags & TPC_CF_CLUSTER_FLAGS) ? 1u : 0u;
    if (digits)
        k_share_apply<false><<<148 * 10, kShareThreads, 0, st>>>((uint4*)out, g, ws.line_cnt, peaks_y, queue, ws.counters,
                                                                 (const uint2*)digits, ws.line_start, nullptr, q_gate, want_flags);
    else
        k_share_apply<true><<<148 * 10, kShareThreads, 0, st>>>((uint4*)out, g, ws.line_cnt, peaks_y, queue, ws.counters,
                                                                nullptr, nullptr, ws.map, q_gate, want_flags);
    return 3;
}

}  // namespace tpccf
