// tpc_cf_sort.cu — any digit order at the speed of the fused path: the digits are SORTED ON THE DEVICE into
// (sector,row,pad,time) order, then the fused sorted path runs on the sorted copy (K5's "deterministic output ordering"
// moved in front of the pipeline).  Measured before this file existed: a randomly ordered config-3 frame took 29.3 ms on
// the general path (random 2-byte map writes: k_scatter / k_unscatter 9.8 ms each, k_peaks_map 6.7 ms, key sort of the
// clusters 2.9 ms) against 1.85 ms for the sorted frame.
//
// The sort uses what the key is: a digit's key is (pad line, time); lines are few (755 k for the full geometry), times are
// unique inside a line (R11: one digit per cell).  So: an UNSTABLE two-level partition of the digits by pad line (order
// inside a line does not matter yet), then one warp per line ranks its digits by time with a bitmap (rank = set bits
// below).  No comparison sort, no stable radix pass:
//   k_sort_count_top   digits per top-level bucket (<= 1024 buckets of 2^shift consecutive lines): a shared-memory
//                      histogram per block; k_sort_top_scan turns the counts into the buckets' first positions
//   k_sort_scatter_top tile of 8192 digits: ranks per bucket by shared-memory atomics, the tile staged in bucket order,
//                      one global atomic per (tile, bucket) reserves the run -> digits grouped by bucket in ws.sort_tmp
//   k_sort_count_grouped digits per pad line, counted on the grouped digits: two blocks per bucket, shared-memory
//                      histogram of the bucket's lines, one global atomic per line
//   scan (n_lines + 1) -> line_start: THE LINE INDEX OF THE FUSED PATH (k_plane_index / k_line_index are not needed)
//   k_sort_scatter_line tile of 4096 digits (one bucket, rarely two): the same per line -> digits grouped by line in the cluster
//                      staging area (idle here)
//   k_sort_rank_lines  one warp per line: time bitmap + rank directory in shared memory -> sorted digits in ws.sort_tmp
// Invalid digits (R11: out-of-range sector / row / pad / time, zero charge) go to an overflow bin behind the last line:
// counted, never seen by the fused kernel.  A duplicate cell shows up as a bit already set in a line's bitmap: reported
// like a false DIGITS_SORTED promise (status.path = 0, no output) — on the general path it was "unspecified".
// Definition: include/tpc_cf.h (R10, R12: exactly one correct output array, independent of the input order).
#include "tpc_cf_internal.cuh"

namespace tpccf {

static constexpr int kSortThreads = 256;
static constexpr int kSortPerThread = 8;
static constexpr uint32_t kSortTopBins = 1024;

// line index of a digit in the fused path's table (plane * LS + pad), or n_lines for an invalid digit (R11)
__device__ __forceinline__ uint32_t sort_line_of(const Geo& g, uint32_t w0, uint32_t w1, uint32_t n_lines)
{
    const uint32_t s = w0 & 0xffu, r = (w0 >> 8) & 0xffu, p = (w0 >> 16) & 0xffu;
    return digit_valid(g, w0, w1) ? (s * g.n_rows + r) * g.LS + p : n_lines;
}

// The same with the pads-per-row table in SHARED memory: g.npads[] lives in the kernel's parameter space, and a load
// from there with a per-lane index (the rows of unordered digits differ from lane to lane) is replayed once per distinct
// row of the warp.
__device__ __forceinline__ uint32_t sort_line_of_s(const Geo& g, const uint8_t* s_np, uint32_t w0, uint32_t w1,
                                                   uint32_t n_lines)
{
    const uint32_t s = w0 & 0xffu, r = (w0 >> 8) & 0xffu, p = (w0 >> 16) & 0xffu;
    const uint32_t t = w1 & 0xffffu, q = w1 >> 16;
    const bool ok = s < g.n_sectors && r < g.n_rows && p < (uint32_t)s_np[r] && t < g.n_time && q != 0u;
    return ok ? (s * g.n_rows + r) * g.LS + p : n_lines;
}

static constexpr int kTopThreads = 1024;                             // top-level pass: tiles of 8192 digits, so that a
static constexpr int kTopTileN = kTopThreads * kSortPerThread;       //   (tile, bucket) run is ~11 digits, not ~3
static constexpr int kSortBlocks = 148 * 2;                          // persistent blocks of the top-level pass
static constexpr int kLineThreads = 512;                             // line-level scatter: tiles of 4096 digits, 4 blocks per SM
static constexpr int kLineTileN = kLineThreads * kSortPerThread;
static constexpr uint32_t kLineBins = 1024;                          // lines a tile may span for the aggregated path (one top-level bucket)

// digits per top-level bucket: a histogram per block in shared memory, one global atomic per (block, bucket)
__global__ void __launch_bounds__(1024)
k_sort_count_top(const uint2* __restrict__ digits, uint32_t n, Geo g, uint32_t n_lines, uint32_t shift,
                 uint32_t* __restrict__ top_cnt)
{
    __shared__ uint32_t s_h[kSortTopBins];
    __shared__ uint8_t s_np[256];
    s_h[threadIdx.x] = 0u;
    if (threadIdx.x < 256) s_np[threadIdx.x] = g.npads[threadIdx.x];
    __syncthreads();
    for (uint64_t i = (uint64_t)blockIdx.x * 1024u + threadIdx.x; i < n; i += (uint64_t)gridDim.x * 1024u) {
        const uint2 d = __ldg(digits + i);
        atomicAdd(&s_h[sort_line_of_s(g, s_np, d.x, d.y, n_lines) >> shift], 1u);
    }
    __syncthreads();
    if (s_h[threadIdx.x]) atomicAdd(&top_cnt[threadIdx.x], s_h[threadIdx.x]);
}

// counts -> first position of every top-level bucket (exclusive scan of 1024 values, one block); a copy stays in
// top_start for the line count
__global__ void __launch_bounds__(1024)
k_sort_top_scan(uint32_t* __restrict__ top_cur)
{
    __shared__ uint32_t s_w[32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t c = top_cur[tid];
    uint32_t inc = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t up = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += up;
    }
    if (lane == 31) s_w[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        const uint32_t w = s_w[lane];
        uint32_t winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t up = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= o) winc += up;
        }
        s_w[lane] = winc - w;
    }
    __syncthreads();
    top_cur[tid] = s_w[warp] + inc - c;
}

// digits per pad line, counted on the digits GROUPED BY BUCKET (after the top-level pass top_cur[b] is the END of bucket
// b): kCountSplit blocks per bucket count their share of the bucket in shared memory (a bucket is 2^shift <= kCountBins
// consecutive lines) and flush with one global atomic per line — 2 M atomics instead of one per digit.  Buckets of more
// lines than the histogram holds (geometries far beyond the TPC's) are counted with one global atomic per digit.
static constexpr uint32_t kCountBins = 2048, kCountSplit = 2, kCountThreads = 512;
__global__ void __launch_bounds__(kCountThreads)
k_sort_count_grouped(const uint2* __restrict__ digits, Geo g, uint32_t n_lines, uint32_t shift,
                     const uint32_t* __restrict__ top_end, uint32_t* __restrict__ line_cnt)
{
    __shared__ uint32_t s_h[kCountBins];
    __shared__ uint8_t s_np[256];                                 // pads per row (see sort_line_of_s)
    if (threadIdx.x < 256) s_np[threadIdx.x] = g.npads[threadIdx.x];
    const uint32_t b = blockIdx.x / kCountSplit, part = blockIdx.x % kCountSplit;
    const uint32_t beg = b ? top_end[b - 1u] : 0u, end = top_end[b];
    if (end <= beg) return;
    const uint32_t len = end - beg, per = (len + kCountSplit - 1u) / kCountSplit;
    const uint32_t lo = beg + part * per, hi = min(end, lo + per);
    const uint32_t l0 = b << shift;
    const bool fits = (1u << shift) <= kCountBins;
    for (uint32_t i = threadIdx.x; i < kCountBins; i += kCountThreads) s_h[i] = 0u;
    __syncthreads();
    for (uint32_t i = lo + threadIdx.x; i < hi; i += kCountThreads) {
        const uint2 d = __ldg(digits + i);
        const uint32_t line = sort_line_of_s(g, s_np, d.x, d.y, n_lines);
        if (fits) atomicAdd(&s_h[line - l0], 1u); else atomicAdd(&line_cnt[line], 1u);
    }
    __syncthreads();
    if (fits)
        for (uint32_t i = threadIdx.x; i < kCountBins; i += kCountThreads)
            if (s_h[i]) atomicAdd(&line_cnt[l0 + i], s_h[i]);
}

// Top level: a tile of 8192 digits; the (tile, bucket) run is reserved by one global atomic on the bucket's cursor.
// The tile is first brought into bucket order in shared memory (ranks by shared-memory atomics, bucket offsets by a block
// scan), then written out in that order: neighbouring lanes write neighbouring addresses of a bucket's run, so a warp's
// store covers a few 32-byte sectors instead of 32 (ncu: 216 M store sectors for 220 M digits without the staging).
__global__ void __launch_bounds__(kTopThreads)
k_sort_scatter_top(const uint2* __restrict__ in, uint2* __restrict__ out, uint32_t n, Geo g,
                   uint32_t n_lines, uint32_t shift, uint32_t* __restrict__ top_cur)
{
    extern __shared__ __align__(16) uint2 s_tile[];              // kTopTileN digits in bucket order
    __shared__ uint32_t s_cnt[kSortTopBins];                     // digits of the tile per bucket
    __shared__ uint32_t s_off[kSortTopBins];                     // first position of the bucket inside the tile
    __shared__ uint32_t s_cur[kSortTopBins];                     // output position of the bucket's run of this tile
    __shared__ uint32_t s_warp[32];
    __shared__ uint8_t s_np[256];                                // pads per row (see sort_line_of_s)
    static_assert(kTopThreads == (int)kSortTopBins, "one thread per bucket in the block scan");
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    s_cnt[tid] = 0u;
    if (tid < 256) s_np[tid] = g.npads[tid];
    __syncthreads();
    const uint32_t n_tiles = (uint32_t)(((uint64_t)n + kTopTileN - 1) / kTopTileN);
    // the digits of the block's next tile are loaded while the present one is ranked, staged and written
    uint2 dn[kSortPerThread];
    auto load_tile = [&](uint32_t tile) {
        const uint64_t t0 = (uint64_t)tile * kTopTileN;
        const uint32_t m = tile < n_tiles ? (uint32_t)min((uint64_t)kTopTileN, (uint64_t)n - t0) : 0u;
#pragma unroll
        for (int j = 0; j < kSortPerThread; ++j) {
            const uint32_t i = (uint32_t)j * kTopThreads + tid;
            if (i < m) dn[j] = __ldg(in + t0 + i);
        }
    };
    load_tile(blockIdx.x);
    for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const uint64_t t0 = (uint64_t)tile * kTopTileN;
        const uint32_t m = (uint32_t)min((uint64_t)kTopTileN, (uint64_t)n - t0);     // digits in this tile
        uint2 d[kSortPerThread];
        uint32_t bin[kSortPerThread], rk[kSortPerThread];
#pragma unroll
        for (int j = 0; j < kSortPerThread; ++j) d[j] = dn[j];
        load_tile(tile + gridDim.x);
#pragma unroll
        for (int j = 0; j < kSortPerThread; ++j) {
            const uint32_t i = (uint32_t)j * kTopThreads + tid;
            bin[j] = 0xffffffffu;
            if (i < m) {
                bin[j] = sort_line_of_s(g, s_np, d[j].x, d[j].y, n_lines) >> shift;
                rk[j] = atomicAdd(&s_cnt[bin[j]], 1u);
            }
        }
        __syncthreads();
        {   // exclusive scan of the 1024 bucket counts, one per thread
            const uint32_t c = s_cnt[tid];
            uint32_t inc = c;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t up = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += up;
            }
            if (lane == 31) s_warp[warp] = inc;
            __syncthreads();
            if (warp == 0) {
                const uint32_t w = s_warp[lane];
                uint32_t winc = w;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t up = __shfl_up_sync(0xffffffffu, winc, o);
                    if (lane >= o) winc += up;
                }
                s_warp[lane] = winc - w;
            }
            __syncthreads();
            s_off[tid] = s_warp[warp] + inc - c;
            if (c) s_cur[tid] = atomicAdd(&top_cur[tid], c);      // one reservation per (tile, bucket)
        }
        __syncthreads();
#pragma unroll
        for (int j = 0; j < kSortPerThread; ++j)
            if (bin[j] != 0xffffffffu) s_tile[s_off[bin[j]] + rk[j]] = d[j];
        __syncthreads();
#pragma unroll
        for (int j = 0; j < kSortPerThread; ++j) {
            const uint32_t i = (uint32_t)j * kTopThreads + tid;
            if (i < m) {
                const uint2 e = s_tile[i];
                const uint32_t b2 = sort_line_of_s(g, s_np, e.x, e.y, n_lines) >> shift;
                out[s_cur[b2] + (i - s_off[b2])] = e;
            }
        }
        __syncthreads();
        s_cnt[tid] = 0u;
        __syncthreads();
    }
}

// Line level: cursor[l] starts at line_start[l].  The input is grouped by top-level bucket, so a tile of 4096 digits spans
// few lines: its digits are ranked per line in shared memory and ONE global atomic per (tile, line) reserves the range
// (a tile spanning more than kLineBins lines — sparse data — takes one atomic per digit instead).
__global__ void __launch_bounds__(kLineThreads)
k_sort_scatter_line(const uint2* __restrict__ in, uint2* __restrict__ out, uint32_t n, Geo g, uint32_t n_lines,
                    uint32_t shift, uint32_t* __restrict__ cursor)
{
    extern __shared__ __align__(16) uint2 s_dyn[];
    uint2* s_tile = s_dyn;                                        // kLineTileN digits in line order
    uint32_t* s_cnt = (uint32_t*)(s_dyn + kLineTileN);            // [kLineBins] digits of the tile per line
    uint32_t* s_off = s_cnt + kLineBins;                          // first position of the line inside the tile
    uint32_t* s_base = s_off + kLineBins;                         // output position of the line's run (global atomic)
    __shared__ uint32_t s_warp[32];
    __shared__ uint32_t s_l0, s_l1;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr uint32_t kPer = kLineBins / kLineThreads;           // bins per thread in the block scan
    const uint32_t n_tiles = (uint32_t)(((uint64_t)n + kLineTileN - 1) / kLineTileN);
    // the digits of the block's next tile are loaded while the present one is ranked, staged and written
    uint2 dn[kSortPerThread];
    auto load_tile = [&](uint32_t tile) {
        const uint64_t t0 = (uint64_t)tile * kLineTileN;
        const uint32_t m = tile < n_tiles ? (uint32_t)min((uint64_t)kLineTileN, (uint64_t)n - t0) : 0u;
#pragma unroll
        for (int j = 0; j < kSortPerThread; ++j) {
            const uint32_t i = (uint32_t)j * kLineThreads + tid;
            if (i < m) dn[j] = __ldg(in + t0 + i);
        }
    };
    load_tile(blockIdx.x);
    for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const uint64_t t0 = (uint64_t)tile * kLineTileN, t1 = min((uint64_t)n, t0 + kLineTileN);
        const uint32_t m = (uint32_t)(t1 - t0);
        // the range of lines the tile spans comes from its digits: the input is grouped by top-level bucket, so the
        // range is one bucket (rarely parts of two)
        uint2 d[kSortPerThread];
        uint32_t bin[kSortPerThread], rk[kSortPerThread];
        uint32_t lmin = 0xffffffffu, lmax = 0u;
        if (tid == 0) { s_l0 = 0xffffffffu; s_l1 = 0u; }
        for (uint32_t i = tid; i < kLineBins; i += kLineThreads) s_cnt[i] = 0u;
#pragma unroll
        for (int j = 0; j < kSortPerThread; ++j) d[j] = dn[j];
        load_tile(tile + gridDim.x);
#pragma unroll
        for (int j = 0; j < kSortPerThread; ++j) {
            const uint32_t i = (uint32_t)j * kLineThreads + tid;
            bin[j] = 0xffffffffu;
            if (i < m) {
                bin[j] = sort_line_of(g, d[j].x, d[j].y, n_lines);
                lmin = min(lmin, bin[j]); lmax = max(lmax, bin[j]);
            }
        }
        __syncthreads();
        lmin = __reduce_min_sync(0xffffffffu, lmin);
        lmax = __reduce_max_sync(0xffffffffu, lmax);
        if (lane == 0) { atomicMin(&s_l0, lmin); atomicMax(&s_l1, lmax); }
        __syncthreads();
        const uint32_t l0 = s_l0, span = s_l1 - l0 + 1u;
        if (span <= kLineBins) {
#pragma unroll
            for (int j = 0; j < kSortPerThread; ++j) {
                if (bin[j] != 0xffffffffu) {
                    bin[j] -= l0;
                    rk[j] = atomicAdd(&s_cnt[bin[j]], 1u);
                }
            }
            __syncthreads();
            {   // exclusive scan of the line counts (kPer consecutive bins per thread) + the runs' output positions
                uint32_t c[kPer], sum = 0u;
#pragma unroll
                for (uint32_t q = 0; q < kPer; ++q) { c[q] = s_cnt[tid * kPer + q]; sum += c[q]; }
                uint32_t inc = sum;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const uint32_t up = __shfl_up_sync(0xffffffffu, inc, o);
                    if (lane >= o) inc += up;
                }
                if (lane == 31) s_warp[warp] = inc;
                __syncthreads();
                if (warp == 0) {
                    const uint32_t w = lane < kLineThreads / 32 ? s_warp[lane] : 0u;
                    uint32_t winc = w;
#pragma unroll
                    for (int o = 1; o < 32; o <<= 1) {
                        const uint32_t up = __shfl_up_sync(0xffffffffu, winc, o);
                        if (lane >= o) winc += up;
                    }
                    s_warp[lane] = winc - w;
                }
                __syncthreads();
                uint32_t run = s_warp[warp] + inc - sum;
#pragma unroll
                for (uint32_t q = 0; q < kPer; ++q) {
                    const uint32_t b = tid * kPer + q;
                    s_off[b] = run;
                    run += c[q];
                    if (c[q]) s_base[b] = atomicAdd(&cursor[l0 + b], c[q]);
                }
            }
            __syncthreads();
#pragma unroll
            for (int j = 0; j < kSortPerThread; ++j)
                if (bin[j] != 0xffffffffu) s_tile[s_off[bin[j]] + rk[j]] = d[j];
            __syncthreads();
#pragma unroll
            for (int j = 0; j < kSortPerThread; ++j) {
                const uint32_t i = (uint32_t)j * kLineThreads + tid;
                if (i < m) {
                    const uint2 e = s_tile[i];
                    const uint32_t b2 = sort_line_of(g, e.x, e.y, n_lines) - l0;
                    out[s_base[b2] + (i - s_off[b2])] = e;
                }
            }
        } else {
            for (uint64_t i = t0 + tid; i < t1; i += kLineThreads) {
                const uint2 d = __ldg(in + i);
                out[atomicAdd(&cursor[sort_line_of(g, d.x, d.y, n_lines)], 1u)] = d;
            }
        }
        __syncthreads();
    }
}

// One warp per pad line: the line's digits (any order) -> time order.  Shared memory per warp: a bitmap over the time
// axis (bm, kept all-zero between lines: a line clears the words it set) and the number of set bits in front of every
// bitmap word (pre).  rank(t) = pre[t / 32] + popc(bm[t / 32] below bit t): the digit's place in the sorted line.
// A bit found already set is a duplicate cell (R11 contract violation): raised as Counters::unsorted.
// The zeroing of line_cnt / line_desc for the fused kernels that follow rides along (line_cnt was the scatter cursor).
static constexpr int kRankRegs = 16;                                 // digits per lane kept in registers: lines up to 512 digits

__global__ void __launch_bounds__(kSortThreads)
k_sort_rank_lines(const uint2* __restrict__ in, uint2* __restrict__ out, const uint32_t* __restrict__ line_start,
                  uint32_t n_lines, uint32_t n_time, uint32_t words, uint32_t* __restrict__ line_cnt,
                  unsigned long long* __restrict__ line_desc, Counters* cnt)
{
    extern __shared__ __align__(16) uint32_t s_sort[];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = kSortThreads / 32;
    uint32_t* bm = s_sort + (size_t)warp * (words + (words + 1) / 2);
    uint16_t* pre = (uint16_t*)(bm + words);
    for (uint32_t w = lane; w < words; w += 32) bm[w] = 0u;
    __syncwarp();
    const uint32_t total_warps = gridDim.x * nwarp;
    uint32_t dup = 0u;
    for (uint32_t l = blockIdx.x * nwarp + warp; l < n_lines; l += total_warps) {
        const uint32_t ls = line_start[l], len = line_start[l + 1] - ls;
        if (lane == 0) line_cnt[l] = 0u;
        if (lane == 1 && (l & 63u) == 0u) line_desc[l >> 6] = 0ull;
        if (len == 0u) continue;
        if (len == 1u) { if (lane == 0) out[ls] = in[ls]; continue; }
        uint32_t wlo = 0xffffffffu, whi = 0u;               // words this line touches
        // a line of up to 32 * kRankRegs digits is read ONCE, all loads in flight together, and kept in registers
        // between the two phases; longer lines are read twice
        const bool in_regs = len <= 32u * (uint32_t)kRankRegs;
        uint2 d[kRankRegs];
        if (in_regs) {
#pragma unroll
            for (int k = 0; k < kRankRegs; ++k) {
                const uint32_t i = (uint32_t)lane + 32u * (uint32_t)k;
                d[k] = i < len ? __ldg(in + ls + i) : make_uint2(0u, 0u);
            }
#pragma unroll
            for (int k = 0; k < kRankRegs; ++k) {
                if ((uint32_t)lane + 32u * (uint32_t)k < len) {
                    const uint32_t t = d[k].y & 0xffffu;             // (valid digits only: t < n_time)
                    const uint32_t old = atomicOr(&bm[t >> 5], 1u << (t & 31u));
                    dup |= (old >> (t & 31u)) & 1u;
                    wlo = min(wlo, t >> 5); whi = max(whi, t >> 5);
                }
            }
        } else {
            for (uint32_t i = lane; i < len; i += 32) {
                const uint32_t t = __ldg(&in[ls + i].y) & 0xffffu;
                const uint32_t old = atomicOr(&bm[t >> 5], 1u << (t & 31u));
                dup |= (old >> (t & 31u)) & 1u;
                wlo = min(wlo, t >> 5); whi = max(whi, t >> 5);
            }
        }
        wlo = __reduce_min_sync(0xffffffffu, wlo);
        whi = __reduce_max_sync(0xffffffffu, whi);
        __syncwarp();
        // set bits in front of every word of [wlo, whi]: every lane takes a contiguous run of words
        const uint32_t span = whi - wlo + 1u, per = (span + 31u) / 32u;
        const uint32_t w0 = wlo + (uint32_t)lane * per, w1 = min(w0 + per, whi + 1u);
        uint32_t mine = 0u;
        for (uint32_t w = w0; w < w1; ++w) mine += (uint32_t)__popc(bm[w]);
        uint32_t inc = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t up = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += up;
        }
        uint32_t run = inc - mine;
        for (uint32_t w = w0; w < w1; ++w) { pre[w] = (uint16_t)run; run += (uint32_t)__popc(bm[w]); }
        __syncwarp();
        if (in_regs) {
#pragma unroll
            for (int k = 0; k < kRankRegs; ++k) {
                if ((uint32_t)lane + 32u * (uint32_t)k < len) {
                    const uint32_t t = d[k].y & 0xffffu;
                    const uint32_t rank = (uint32_t)pre[t >> 5] + (uint32_t)__popc(bm[t >> 5] & ((1u << (t & 31u)) - 1u));
                    out[ls + min(rank, len - 1u)] = d[k];      // (min: stays inside the line if a duplicate broke the ranks)
                }
            }
        } else {
            for (uint32_t i = lane; i < len; i += 32) {
                const uint2 e = __ldg(in + ls + i);
                const uint32_t t = e.y & 0xffffu;
                const uint32_t rank = (uint32_t)pre[t >> 5] + (uint32_t)__popc(bm[t >> 5] & ((1u << (t & 31u)) - 1u));
                out[ls + min(rank, len - 1u)] = e;
            }
        }
        __syncwarp();
        for (uint32_t w = w0; w < w1; ++w) bm[w] = 0u;
        __syncwarp();
    }
    if (lane == 0 && blockIdx.x == 0 && warp == 0) {
        // the overflow bin behind the last line holds the invalid digits (R11): line_cnt was the line-level cursor
        const uint32_t n_bad = line_cnt[n_lines] - line_start[n_lines];
        if (n_bad) atomicAdd(&cnt->n_bad, (unsigned long long)n_bad);
        line_cnt[n_lines] = 0u;
        line_desc[(n_lines >> 6) + 1u] = 0ull;
    }
    if (__any_sync(0xffffffffu, dup != 0u) && lane == 0) atomicOr(&cnt->unsorted, 1u);
}

static uint32_t sort_rank_smem(const Geo& g, uint32_t* words_out)
{
    const uint32_t words = ((g.n_time + 31u) / 32u + 3u) & ~3u;
    *words_out = words;
    return (kSortThreads / 32) * (words + (words + 1) / 2) * 4u;
}

cudaError_t sort_set_attributes()
{
    cudaError_t e = cudaFuncSetAttribute(k_sort_scatter_top, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kTopTileN * sizeof(uint2)));
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(k_sort_scatter_line, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kLineTileN * sizeof(uint2) + 3 * kLineBins * 4));
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_sort_rank_lines, cudaFuncAttributeMaxDynamicSharedMemorySize, 100 * 1024);
}

// Sorts `n` digits into ws.sort_tmp and leaves the fused path's line index in ws.line_start (and line_cnt / line_desc
// zeroed).  The counters must have been zeroed on the stream before.  Returns the number of launches.
int launch_sort_digits(const Geo& g, const Workspace& ws, const tpc_digit* digits, uint64_t n, cudaStream_t st)
{
    const uint32_t n_lines = g.n_planes * g.LS;
    uint32_t shift = 0;
    while (((n_lines + 1u) >> shift) >= kSortTopBins) ++shift;      // top-level bucket = line >> shift, < 1024 buckets
    const uint2* in = (const uint2*)digits;
    uint2* tmp = (uint2*)ws.sort_tmp;
    uint2* tmp2 = (uint2*)ws.stage;                                 // the cluster staging area is idle until the fused kernel
    const int grid = 148 * 8;
    int k = 0;
    cudaMemsetAsync(ws.line_cnt, 0, ((size_t)n_lines + 2) * 4, st);
    cudaMemsetAsync(ws.sort_top, 0, (size_t)kSortTopBins * 4, st);
    k_sort_count_top<<<kSortBlocks, 1024, 0, st>>>(in, (uint32_t)n, g, n_lines, shift, ws.sort_top);
    k_sort_top_scan<<<1, 1024, 0, st>>>(ws.sort_top);
    k_sort_scatter_top<<<kSortBlocks, kTopThreads, kTopTileN * sizeof(uint2), st>>>(in, tmp, (uint32_t)n, g, n_lines, shift, ws.sort_top);
    k_sort_count_grouped<<<kSortTopBins * kCountSplit, kCountThreads, 0, st>>>(tmp, g, n_lines, shift, ws.sort_top, ws.line_cnt);
    k += 4 + launch_scan_u32(ws.line_cnt, ws.line_start, (uint64_t)n_lines + 1, ws.sort_part, nullptr, st);
    // the fused kernels read line_start[n_lines] as the end of the last plane: the overflow bin (invalid digits) starts there
    cudaMemcpyAsync(ws.line_cnt, ws.line_start, ((size_t)n_lines + 1) * 4, cudaMemcpyDeviceToDevice, st);
    k_sort_scatter_line<<<148 * 4, kLineThreads, kLineTileN * sizeof(uint2) + 3 * kLineBins * 4, st>>>(tmp, tmp2, (uint32_t)n, g, n_lines, shift, ws.line_cnt);
    uint32_t words;
    const uint32_t smem = sort_rank_smem(g, &words);
    k_sort_rank_lines<<<grid, kSortThreads, smem, st>>>(tmp2, tmp, ws.line_start, n_lines, g.n_time, words, ws.line_cnt,
                                                        ws.line_desc, ws.counters);
    return k + 2;
}

}  // namespace tpccf
