// tpc_cf_internal.cuh — internal declarations of the B200 TPC cluster finder (product code, sm_100a).
// Nothing here is shared with oracle/.  Definition implemented: include/tpc_cf.h (BASELINE.json:north_star,
// readings R1..R19 of SURVEY.md §8(c) / DESIGN.md §3; step named in PAPER.md:57).
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tpc_cf.h"

namespace tpccf {

// Geometry as the kernels see it (passed by value as a kernel parameter; 256 + 32 bytes).
struct Geo {
    uint32_t n_sectors, n_rows, max_pads, n_time;
    uint32_t n_planes;   // n_sectors * n_rows
    uint32_t PS;         // map pad stride  = max_pads + 4 (2-cell zero border each side, R2)
    uint32_t TS;         // map time stride = roundup(n_time + 4, 8) uint16 (16-byte multiple)
    uint32_t LS;         // line-index stride per plane = max_pads + 1
    uint8_t  npads[256]; // pads of each row (R19)
};

// Device-side counters of one run (zeroed by a memset node at the start of every run).
struct Counters {
    unsigned long long n_bad;       // R11
    unsigned long long n_used;
    unsigned long long n_clusters;  // total peaks
    unsigned int unsorted;          // 1 if digits[i-1] > digits[i] for some i (key = sector,row,pad,time)
    unsigned int n_share;           // V4: clusters queued for the sharing pass (tpc_cf_share.cu)
};

// Pointers into the caller-owned workspace.
struct Workspace {
    Counters* counters;
    uint16_t* map;        // [n_planes][PS][TS], zero between runs
    uint32_t* peakmask;   // bit j%32 of word j/32: digit j is a peak
    uint32_t* blk_cnt;    // peaks per 256-word block of peakmask
    uint32_t* blk_off;    // exclusive scan of blk_cnt
    uint32_t* scan_part;  // scan partials
    tpc_cluster* stage;   // [max_digits] sparse: cluster of peak digit j at stage[j]
    tpc_cluster* compact; // [max_clusters] digit-order clusters awaiting the key sort (unsorted input only)
    uint64_t* keyA; uint64_t* keyB;   // [max_clusters] radix sort ping-pong
    uint32_t* idxA; uint32_t* idxB;
    uint32_t* ghist;      // [256][n_sort_tiles]
    uint32_t* ghist_part;
    uint32_t* line_start; // [n_planes*LS + 1] first digit of each (plane,pad) line (fused path)
    uint32_t* line_cnt;   // [n_planes*LS + 1] peaks per line (fused path)
    unsigned long long* line_desc;   // [n_lines / 256 + 1] per 256-line block: (flag << 62) | clusters, for the
                                     // single-pass scan of k_scan_gather_lines (fused path); zeroed by k_line_index
    tpc_cf_status* group_status;   // [32] per-group status blocks of the tpc_cf_run_host pipeline
    tpc_digit* sort_tmp;  // [max_digits] digits sorted on the device (any-order input, tpc_cf_sort.cu); absent in sorted-only workspaces
    uint32_t* sort_top;   // [1025] top-level bucket histogram / cursors of the digit sort
    uint32_t* sort_part;  // scan partials of the digit sort
};

// Slot geometry of the block-sparse fused kernels (kernel parameter; all warp-uniform).
struct SlotGeo {
    uint32_t slot_bytes;   // multiple of 16
    uint32_t pool_off;     // header + dir bytes (multiple of 16)
    uint32_t surv_off;     // pool_off + 16 * pcap
    uint32_t pcap;         // blocks in the pool including the zero block 0 (<= 255)
    uint32_t scap;         // survivor entries per slot
    uint32_t n_pass;       // the time axis is covered in n_pass segments, one pass over the unit's lines each
    uint32_t seg_len;      // time bins per segment (multiple of 8); n_pass * seg_len >= n_time
};

// Test / tuning overrides of a handle (tpc_cf_debug_set; all 0 = the library decides).  They never change the result.
struct Tuning {
    int fused_kernel;      // TPC_CF_DEBUG_FUSED_KERNEL: 0 auto, 1 k_fused_pairs, 2 k_fused_blocks, 3 k_fused_lines
    int passes;            // TPC_CF_DEBUG_PASSES: time passes of the block-sparse kernels
    int block_pool;        // TPC_CF_DEBUG_BLOCK_POOL: pool blocks per slot (forces the pool-overflow slow path)
    int surv_cap;          // TPC_CF_DEBUG_SURV_CAP: survivor entries per slot (forces the list-overflow slow path)
    int pads_per_unit;     // TPC_CF_DEBUG_PADS_PER_UNIT: pads per CTA (multiple of 8)
    int ctas_per_sm;       // TPC_CF_DEBUG_CTAS_PER_SM: 2 = never use the 3-CTA instantiation
};

// ---- shared device arithmetic -------------------------------------------------------------------------------

__host__ __device__ inline uint32_t npads_of(const Geo& g, uint32_t row) { return g.npads[row]; }

// R11: a digit is valid iff it addresses an existing cell and carries charge.
__device__ __forceinline__ bool digit_valid(const Geo& g, uint32_t w0, uint32_t w1)
{
    const uint32_t s = w0 & 0xffu, r = (w0 >> 8) & 0xffu, p = (w0 >> 16) & 0xffu;
    const uint32_t t = w1 & 0xffffu, q = w1 >> 16;
    return s < g.n_sectors && r < g.n_rows && p < (uint32_t)g.npads[r < 256u ? r : 0u] && t < g.n_time && q != 0u;
}

// Sort key of a digit / cluster: (sector,row,pad,time) big-endian in 40 bits (R10).
__device__ __forceinline__ uint64_t key40(uint32_t w0, uint32_t w1)
{
    return ((uint64_t)(w0 & 0xffu) << 32) | ((uint64_t)((w0 >> 8) & 0xffu) << 24) |
           ((uint64_t)((w0 >> 16) & 0xffu) << 16) | (uint64_t)(w1 & 0xffffu);
}

// K4: from the 5x5 window c[dp+2][dt+2] around a peak, the gated sums and the 32-byte record.
// Gate of outer cell (dp,dt) is (dp - sgn dp, dt - sgn dt) (R3); compared raw against q_inner_gate (R4).
// Sums are integers taken relative to the peak, |S| <= 25*65535*4 < 2^24 (R8), so any order is exact;
// the variance numerator S0*S2 - S1^2 is formed in int64 and rounded once.
struct ClusterWords { uint4 lo, hi; };
struct ClusterSums { int S0, S1p, S1t, S2p, S2t; };   // integer sums relative to the peak cell (R8)

// Cluster-finder variants (include/tpc_cf.h V1..V3): knobs of one run, warp-uniform kernel parameter.
struct Variant {
    uint32_t q_tot_min;      // V2: minimum qTot (0 = no cut)
    uint32_t q_saturation;   // V1: SATURATED threshold (0 = never)
    uint32_t vflags;         // TPC_CF_CLUSTER_FLAGS | TPC_CF_CUT_SINGLE_PAD | TPC_CF_CUT_SINGLE_TIME
    uint32_t active;         // any of the above set: the default run skips all of it
};

// V1 flags of a cluster from its peak cell and sums; returns false if a cut (V2) drops it.
// P = pads of the peak's row, T = n_time.
__device__ __forceinline__ bool cluster_variant(const ClusterSums& m, uint32_t pad, uint32_t time, uint32_t qmax,
                                                uint32_t P, uint32_t T, const Variant& v, uint32_t* flags)
{
    uint32_t fl = 0u;
    if (pad < 2u || pad + 2u >= P) fl |= TPC_CF_F_EDGE_PAD;
    if (time < 2u || time + 2u >= T) fl |= TPC_CF_F_EDGE_TIME;
    if (m.S2p == 0) fl |= TPC_CF_F_SINGLE_PAD;
    if (m.S2t == 0) fl |= TPC_CF_F_SINGLE_TIME;
    if (v.q_saturation != 0u && qmax >= v.q_saturation) fl |= TPC_CF_F_SATURATED;
    *flags = (v.vflags & TPC_CF_CLUSTER_FLAGS) ? fl : 0u;
    if ((uint32_t)m.S0 < v.q_tot_min) return false;
    if ((v.vflags & TPC_CF_CUT_SINGLE_PAD) && (fl & TPC_CF_F_SINGLE_PAD)) return false;
    if ((v.vflags & TPC_CF_CUT_SINGLE_TIME) && (fl & TPC_CF_F_SINGLE_TIME)) return false;
    return true;
}

// R7: record from the sums.  qmax = charge of the peak cell, flags = V1 byte (0 by default).
__device__ __forceinline__ ClusterWords cluster_finish(const ClusterSums& m, uint32_t w0, uint32_t time, uint32_t qmax,
                                                       uint32_t flags = 0u)
{
    const uint32_t pad = (w0 >> 16) & 0xffu;
    // mean = S1/S0, sigma = sqrt(S0*S2 - S1^2)/S0 with the numerator exact in int64 (R8).  The reciprocal and the
    // square roots use the special-function unit (2 ulp, ~2.4e-7 relative — the parity bar is 1e-5 relative / 1e-4
    // absolute, R18): four IEEE divisions and two IEEE square roots per cluster were ~4 % of the fused kernel.
    const float f0 = (float)m.S0;
    const float r0 = __fdividef(1.f, f0);                     // S0 >= q_peak_min >= 1
    const long long np = (long long)m.S0 * m.S2p - (long long)m.S1p * m.S1p;
    const long long nt = (long long)m.S0 * m.S2t - (long long)m.S1t * m.S1t;
    const float fp = (float)np, ft = (float)nt;
    const float pad_mean = (float)pad + (float)m.S1p * r0;      // R7
    const float time_mean = (float)time + (float)m.S1t * r0;
    const float sp = np > 0 ? fp * rsqrtf(fp) * r0 : 0.f;
    const float st = nt > 0 ? ft * rsqrtf(ft) * r0 : 0.f;
    ClusterWords r;
    r.lo.x = (w0 & 0x00ffffffu) | (flags << 24);              // sector,row,pad,flags
    r.lo.y = time | (qmax << 16);                             // time,qmax
    r.lo.z = (uint32_t)m.S0;                                  // qtot
    r.lo.w = __float_as_uint(pad_mean);
    r.hi.x = __float_as_uint(time_mean);
    r.hi.y = __float_as_uint(sp);
    r.hi.z = __float_as_uint(st);
    r.hi.w = 0u;
    return r;
}

__device__ __forceinline__ ClusterSums cluster_sums(const int (&c)[5][5], uint32_t gate)
{
    ClusterSums m = {0, 0, 0, 0, 0};
#pragma unroll
    for (int a = 0; a < 5; ++a) {
#pragma unroll
        for (int b = 0; b < 5; ++b) {
            const int dp = a - 2, dt = b - 2;
            const bool ring = (dp == 2 || dp == -2 || dt == 2 || dt == -2);
            int v = c[a][b];
            if (ring) {
                const int ga = a - (dp > 0) + (dp < 0), gb = b - (dt > 0) + (dt < 0);
                v = ((uint32_t)c[ga][gb] >= gate) ? v : 0;
            }
            m.S0 += v; m.S1p += v * dp; m.S1t += v * dt; m.S2p += v * dp * dp; m.S2t += v * dt * dt;
        }
    }
    return m;
}

__device__ __forceinline__ ClusterWords cluster_from_window(const int (&c)[5][5], uint32_t w0, uint32_t time,
                                                            uint32_t gate)
{
    return cluster_finish(cluster_sums(c, gate), w0, time, (uint32_t)c[2][2]);
}

// One half of the same sums, for two lanes sharing a peak: the rows on one side of the peak (o: |dp| = 2, m: |dp| = 1,
// sgn = sign of dp) and, if with_center, the peak's own row z.  The gate of an outer cell lies one step towards the
// peak (R3): row o is gated by row m, the dt = +-2 cells of rows m and z by z[1] / z[3] — so a half needs rows o, m, z
// only, and the two halves add up to cluster_from_window's sums exactly (integers).
__device__ __forceinline__ ClusterSums cluster_half_sums(const int (&o)[5], const int (&m)[5], const int (&z)[5],
                                                         int sgn, bool with_center, uint32_t gate)
{
    ClusterSums r = {0, 0, 0, 0, 0};
#pragma unroll
    for (int b = 0; b < 5; ++b) {
        const int dt = b - 2;
        const int gb = b - (dt > 0) + (dt < 0);                       // dt one step towards the peak
        const int vo = ((uint32_t)m[gb] >= gate) ? o[b] : 0;          // |dp| = 2: gate (|dp| = 1, dt -+ 1)
        const bool edge = dt == 2 || dt == -2;
        const int vm = (!edge || (uint32_t)z[gb] >= gate) ? m[b] : 0; // |dp| = 1: only dt = +-2 is gated, by (0, +-1)
        const int vz = (with_center && (!edge || (uint32_t)z[gb] >= gate)) ? z[b] : 0;
        r.S0 += vo + vm + vz;
        r.S1p += sgn * (2 * vo + vm);
        r.S1t += dt * (vo + vm + vz);
        r.S2p += 4 * vo + vm;
        r.S2t += dt * dt * (vo + vm + vz);
    }
    return r;
}

// name of the dominant kernel enqueued last by this host thread (set by the launchers, copied into the handle)
extern thread_local const char* g_last_kernel;

// ---- launchers (each returns the number of kernels it enqueued, or a negative tpc_cf error) -----------------

int launch_general_peaks(const Geo& g, const Workspace& ws, const tpc_digit* digits, uint64_t n,
                         uint32_t q_peak_min, uint32_t q_gate, const Variant& var, cudaStream_t st,
                         cudaEvent_t ev_k0, cudaEvent_t ev_k1);
int launch_unscatter(const Geo& g, const Workspace& ws, const tpc_digit* digits, uint64_t n, cudaStream_t st);
int launch_scatter_only(const Geo& g, const Workspace& ws, const tpc_digit* digits, uint64_t n, cudaStream_t st);
int launch_copy_plane(const Geo& g, const Workspace& ws, uint32_t plane, uint32_t P, uint16_t* dense,
                      cudaStream_t st);

// have_index: ws.line_start already holds the line index and line_cnt / line_desc are zero (the digit sort left them so)
int launch_fused_sorted(const Geo& g, const Workspace& ws, const tpc_digit* digits, uint64_t n, uint64_t shape_n,
                        uint32_t q_peak_min, uint32_t q_gate, const Variant& var, const Tuning& tun, bool have_index,
                        cudaStream_t st, cudaEvent_t ev_k0, cudaEvent_t ev_k1);
// any-order input: digits -> ws.sort_tmp in (sector,row,pad,time) order + the line index (tpc_cf_sort.cu)
int launch_sort_digits(const Geo& g, const Workspace& ws, const tpc_digit* digits, uint64_t n, cudaStream_t st);
cudaError_t sort_set_attributes();

// Block-sparse fused kernels after the line index is in ws.line_start.  Return 1 (launched), 0 (not applicable: the
// caller runs another kernel) or a negative tpc_cf error.  must: no other kernel can take this geometry.
int launch_fused_blocks(const Geo& g, const Workspace& ws, const tpc_digit* digits, uint64_t n, uint64_t shape_n,
                        uint32_t q_peak_min, uint32_t q_gate, const Variant& var, const Tuning& tun, bool must,
                        cudaStream_t st, cudaEvent_t ev_k0, cudaEvent_t ev_k1);
int launch_fused_pairs(const Geo& g, const Workspace& ws, const tpc_digit* digits, uint64_t n, uint64_t shape_n,
                       uint32_t q_peak_min, uint32_t q_gate, const Variant& var, const Tuning& tun, bool must,
                       cudaStream_t st, cudaEvent_t ev_k0, cudaEvent_t ev_k1);
// cudaFuncAttributeMaxDynamicSharedMemorySize of the fused kernels, for the CURRENT device (called by tpc_cf_create:
// the attribute is per device)
cudaError_t fused_lines_set_attributes();
cudaError_t fused_blocks_set_attributes();
cudaError_t fused_pairs_set_attributes();

// compaction of stage[j] by peakmask into dst (= out, or ws.compact when a key sort must follow)
int launch_compact(const Workspace& ws, uint64_t n, tpc_cluster* out, uint64_t capacity, uint64_t max_clusters,
                   int sort_if_unsorted, cudaStream_t st);
// fused path, ONE kernel: single-pass scan of ws.line_cnt (decoupled look-back over blocks of 256 lines), copy
// stage[line_start + k] -> out[offset + k], and the status block (written by the last block).
int launch_compact_lines(const Geo& g, const Workspace& ws, tpc_cluster* out, uint64_t capacity,
                         tpc_cf_status* status, uint64_t n, uint32_t path, cudaStream_t st);
int launch_key_sort(const Workspace& ws, uint64_t max_clusters, uint32_t n_sort_tiles, tpc_cluster* out,
                    uint64_t capacity, cudaStream_t st);
int launch_finalize(const Workspace& ws, tpc_cf_status* status, uint64_t capacity, uint32_t path,
                    int hint_sorted, uint64_t n, uint64_t max_clusters, cudaStream_t st);

// V4 (TPC_CF_SHARE_CHARGE): post-pass over the ordered records in `out` once `status` is written (tpc_cf_share.cu).
// digits != nullptr: the sorted digits the fused path ran on (+ ws.line_start); nullptr: the general path's charge map,
// which must still be filled.  Scratch: ws.line_cnt, ws.stage (8 bytes per digit of it), counters->n_share.
int launch_share_charge(const Geo& g, const Workspace& ws, const tpc_digit* digits, tpc_cluster* out, uint64_t capacity,
                        const tpc_cf_status* status, uint32_t q_gate, uint32_t vflags, uint64_t max_digits, cudaStream_t st);

// exclusive scan of n uint32 (in -> out, may alias); total (optional) receives the sum as 64-bit.
int launch_scan_u32(const uint32_t* in, uint32_t* out, uint64_t n, uint32_t* partials,
                    unsigned long long* total, cudaStream_t st);

static inline uint64_t ceil_div_u64(uint64_t a, uint64_t b) { return (a + b - 1) / b; }

}  // namespace tpccf
