// tpc_cf_compact.cu — K3 compaction and K5 ordered output, shared by the general and the fused path.
//   Both paths leave the peak set as one bit per digit (peakmask) and the cluster of peak digit j at stage[j].
//   k_count_peaks / scan / k_gather : order-preserving compaction (popc + prefix sums) into the output array.
//     Sorted digits => digit order is (sector,row,pad,time) order => the output is final (R10).
//   Unsorted digits (general path only): the compacted clusters go to ws.compact and an LSD radix sort on the
//     40-bit (sector,row,pad,time) key orders them (keys are unique, so exactly one array is correct, R10).
//   k_finalize writes the status block last.
#include "tpc_cf_internal.cuh"

namespace tpccf {

// ---- block-wide exclusive scan (blockDim.x <= 1024, multiple of 32) ------------------------------------------
__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* total)
{
    __shared__ uint32_t s_warp[32];
    const unsigned lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    uint32_t inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t u = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= (unsigned)o) inc += u;
    }
    if (lane == 31) s_warp[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        uint32_t w = lane < nwarp ? s_warp[lane] : 0u;
        uint32_t winc = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t u = __shfl_up_sync(0xffffffffu, winc, o);
            if (lane >= (unsigned)o) winc += u;
        }
        s_warp[lane] = winc - w;                 // exclusive warp offsets
        if (lane == 31 && total) *total = winc;  // block total
    }
    __syncthreads();
    const uint32_t r = s_warp[warp] + inc - v;
    __syncthreads();                             // s_warp may be reused by the next call
    return r;
}

// ---- generic exclusive scan over uint32 ----------------------------------------------------------------------
static constexpr int kScanThreads = 1024;

__global__ void __launch_bounds__(kScanThreads)
k_scan_reduce(const uint32_t* __restrict__ in, uint64_t n, uint32_t* __restrict__ partial)
{
    __shared__ uint32_t s_total;
    const uint64_t i = (uint64_t)blockIdx.x * kScanThreads + threadIdx.x;
    const uint32_t v = i < n ? in[i] : 0u;
    block_exclusive_scan(v, &s_total);
    __syncthreads();
    if (threadIdx.x == 0) partial[blockIdx.x] = s_total;
}

__global__ void __launch_bounds__(kScanThreads)
k_scan_partials(uint32_t* partial, uint64_t nb, unsigned long long* total)
{
    __shared__ uint32_t s_total;
    unsigned long long carry = 0;
    for (uint64_t base = 0; base < nb; base += kScanThreads) {
        const uint64_t i = base + threadIdx.x;
        const uint32_t v = i < nb ? partial[i] : 0u;
        const uint32_t ex = block_exclusive_scan(v, &s_total);
        __syncthreads();
        if (i < nb) partial[i] = (uint32_t)(carry + ex);
        carry += s_total;
        __syncthreads();
    }
    if (threadIdx.x == 0 && total) *total = carry;
}

__global__ void __launch_bounds__(kScanThreads)
k_scan_apply(const uint32_t* in, uint32_t* out, uint64_t n, const uint32_t* __restrict__ partial)
{
    const uint64_t i = (uint64_t)blockIdx.x * kScanThreads + threadIdx.x;
    const uint32_t v = i < n ? in[i] : 0u;
    const uint32_t ex = block_exclusive_scan(v, nullptr);
    if (i < n) out[i] = partial[blockIdx.x] + ex;
}

int launch_scan_u32(const uint32_t* in, uint32_t* out, uint64_t n, uint32_t* partials,
                    unsigned long long* total, cudaStream_t st)
{
    if (n == 0) return 0;
    const uint64_t nb = ceil_div_u64(n, kScanThreads);
    k_scan_reduce<<<(unsigned)nb, kScanThreads, 0, st>>>(in, n, partials);
    k_scan_partials<<<1, kScanThreads, 0, st>>>(partials, nb, total);
    k_scan_apply<<<(unsigned)nb, kScanThreads, 0, st>>>(in, out, n, partials);
    return 3;
}

// ---- K3: compaction -------------------------------------------------------------------------------------------
static constexpr int kCompactThreads = 256;   // one peakmask word (32 digits) per thread

__global__ void __launch_bounds__(kCompactThreads)
k_count_peaks(const uint32_t* __restrict__ peakmask, uint64_t nwords, uint32_t* __restrict__ blk_cnt)
{
    __shared__ uint32_t s_total;
    const uint64_t w = (uint64_t)blockIdx.x * kCompactThreads + threadIdx.x;
    const uint32_t c = w < nwords ? (uint32_t)__popc(peakmask[w]) : 0u;
    block_exclusive_scan(c, &s_total);
    __syncthreads();
    if (threadIdx.x == 0) blk_cnt[blockIdx.x] = s_total;
}

__global__ void __launch_bounds__(kCompactThreads)
k_gather(const uint32_t* __restrict__ peakmask, uint64_t nwords, const uint32_t* __restrict__ blk_off,
         const uint4* __restrict__ stage, uint4* out, uint64_t capacity, uint4* compact, uint64_t max_clusters,
         int sort_if_unsorted, const Counters* cnt)
{
    // A block owns 256 mask words = 8192 digits.  Its peaks are first listed in shared memory in output order
    // (local digit index), then copied by all threads: independent 32-byte loads, fully coalesced stores.
    __shared__ uint16_t s_list[kCompactThreads * 32];
    __shared__ uint32_t s_count;
    const uint64_t w = (uint64_t)blockIdx.x * kCompactThreads + threadIdx.x;
    uint32_t m = w < nwords ? peakmask[w] : 0u;
    uint32_t pos = block_exclusive_scan((uint32_t)__popc(m), &s_count);
    while (m) {
        const int b = __ffs(m) - 1;
        m &= m - 1;
        s_list[pos++] = (uint16_t)(threadIdx.x * 32 + b);
    }
    __syncthreads();
    uint4* dst = out;
    uint64_t cap = capacity;
    if (sort_if_unsorted && cnt->unsorted) { dst = compact; cap = max_clusters; }
    const uint64_t base = blk_off[blockIdx.x];
    const uint64_t j0 = (uint64_t)blockIdx.x * kCompactThreads * 32;
    const uint32_t total = s_count;
    // two 16-byte halves per record: thread pairs (2i, 2i+1) move one record, so a warp writes 512 contiguous bytes
    for (uint32_t i = threadIdx.x; i < 2 * total; i += kCompactThreads) {
        const uint32_t r = i >> 1, h = i & 1u;
        const uint64_t p = base + r;
        if (p < cap) __stcs(dst + 2 * p + h, __ldcs(stage + 2 * (j0 + s_list[r]) + h));
    }
}

int launch_compact(const Workspace& ws, uint64_t n, tpc_cluster* out, uint64_t capacity, uint64_t max_clusters,
                   int sort_if_unsorted, cudaStream_t st)
{
    if (n == 0) return 0;
    const uint64_t nwords = ceil_div_u64(n, 32);
    const uint64_t nblk = ceil_div_u64(nwords, kCompactThreads);
    k_count_peaks<<<(unsigned)nblk, kCompactThreads, 0, st>>>(ws.peakmask, nwords, ws.blk_cnt);
    int k = 1 + launch_scan_u32(ws.blk_cnt, ws.blk_off, nblk, ws.scan_part, &ws.counters->n_clusters, st);
    k_gather<<<(unsigned)nblk, kCompactThreads, 0, st>>>(ws.peakmask, nwords, ws.blk_off, (const uint4*)ws.stage,
                                                         (uint4*)out, capacity, (uint4*)ws.compact, max_clusters,
                                                         sort_if_unsorted, ws.counters);
    return k + 1;
}

// ---- K3 + K5 for the fused path: the peaks of a line are already packed, in time order, at the start of the
// line's own digit range in `stage`; a scan over the per-line counts gives each line its place in the output.
// ONE kernel: a block owns 256 consecutive lines; it scans their counts, publishes its total in line_desc[block] and
// finds the clusters in front of it by a decoupled look-back (a warp reads the 32 descriptors before it at a time:
// flag 1 = this block's total, flag 2 = total of everything up to and including this block), then copies its records:
// they are consecutive in the output, so the block copies one contiguous output range, every thread moving 16-byte
// halves and finding the source line of a record by a binary search in the block's prefix sums (shared memory).
// The last block knows the frame's cluster count and writes the status block.
static constexpr unsigned long long kDescMask = (1ull << 62) - 1ull;

template <int LINES>      // lines per block: 256, or 64 for small geometries (a single sector has only 21 k lines)
__global__ void __launch_bounds__(256)
k_scan_gather_lines(const uint32_t* __restrict__ line_cnt, const uint32_t* __restrict__ line_start, uint32_t n_lines,
                    const uint4* __restrict__ stage, uint4* __restrict__ out, uint64_t capacity,
                    unsigned long long* line_desc, Counters* cnt, tpc_cf_status* status, uint64_t n, uint32_t path)
{
    __shared__ uint32_t s_pref[LINES + 1];
    __shared__ uint32_t s_src[LINES];
    __shared__ unsigned long long s_excl;
    const uint32_t line = blockIdx.x * LINES + threadIdx.x;
    const bool mine = threadIdx.x < LINES && line < n_lines;
    const uint32_t c = mine ? line_cnt[line] : 0u;
    uint32_t total;
    {
        __shared__ uint32_t s_total;
        const uint32_t ex = block_exclusive_scan(c, &s_total);
        if (threadIdx.x < LINES) {
            s_pref[threadIdx.x] = ex;
            s_src[threadIdx.x] = mine ? line_start[line] : 0u;
        }
        __syncthreads();
        total = s_total;
        if (threadIdx.x == 0) s_pref[LINES] = total;
    }
    if (threadIdx.x < 32) {
        volatile unsigned long long* desc = line_desc;
        const unsigned lane = threadIdx.x;
        unsigned long long excl = 0ull;
        if (blockIdx.x == 0) {
            if (lane == 0) desc[0] = (2ull << 62) | (unsigned long long)total;
        } else {
            if (lane == 0) desc[blockIdx.x] = (1ull << 62) | (unsigned long long)total;
            int j = (int)blockIdx.x - 1;                      // descriptor lane 0 looks at
            while (true) {
                const int idx = j - (int)lane;
                unsigned long long v = idx >= 0 ? desc[idx] : (2ull << 62);      // in front of block 0: prefix 0
                while (__any_sync(0xffffffffu, (v >> 62) == 0ull)) v = idx >= 0 ? desc[idx] : (2ull << 62);
                const unsigned full = __ballot_sync(0xffffffffu, (v >> 62) == 2ull);
                const unsigned upto = full ? (unsigned)__ffs(full) : 32u;       // lanes < upto contribute
                unsigned long long part = lane < upto ? (v & kDescMask) : 0ull;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
                excl += part;
                if (full) break;
                j -= 32;
            }
            if (lane == 0) desc[blockIdx.x] = (2ull << 62) | (excl + (unsigned long long)total);
        }
        if (lane == 0) {
            s_excl = excl;
            if (blockIdx.x == gridDim.x - 1) {               // the frame's count is known here: status, written last
                tpc_cf_status s;
                s.n_clusters = excl + total;
                s.n_digits_used = n - cnt->n_bad;
                s.n_bad_digits = cnt->n_bad;
                s.overflow = s.n_clusters > capacity ? 1u : 0u;
                s.path = path;
                if (cnt->unsorted) {      // false DIGITS_SORTED promise: detected, no output (include/tpc_cf.h)
                    s.n_clusters = 0;
                    s.overflow = 0;
                    s.path = 0;
                }
                cnt->n_clusters = excl + total;
                *status = s;
            }
        }
    }
    __syncthreads();
    if (total == 0) return;
    const uint64_t dst0 = s_excl;
    // four 16-byte halves per thread and step: the four loads are in flight together (eight were slower again)
    for (uint32_t i0 = threadIdx.x; i0 < 2 * total; i0 += 4 * 256) {
        uint4 v[4];
        bool ok[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint32_t i = i0 + (uint32_t)k * 256u, r = i >> 1;
            ok[k] = i < 2 * total && dst0 + r < capacity;
            if (ok[k]) {
                uint32_t lo = 0, hi = LINES;             // last line with s_pref[line] <= r
                while (hi - lo > 1) { const uint32_t mid = (lo + hi) >> 1; if (s_pref[mid] <= r) lo = mid; else hi = mid; }
                const uint64_t src = (uint64_t)s_src[lo] + (r - s_pref[lo]);
                v[k] = __ldcs(stage + 2 * src + (i & 1u));
            }
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint32_t i = i0 + (uint32_t)k * 256u;
            if (ok[k]) __stcs(out + 2 * (dst0 + (i >> 1)) + (i & 1u), v[k]);
        }
    }
}

int launch_compact_lines(const Geo& g, const Workspace& ws, tpc_cluster* out, uint64_t capacity,
                         tpc_cf_status* status, uint64_t n, uint32_t path, cudaStream_t st)
{
    const uint32_t n_lines = g.n_planes * g.LS;
    // (line_desc holds one descriptor per 64 lines: tpc_cf_api.cu carve, k_line_index)
    if (n_lines >= 64u * 148u * 16u)
        k_scan_gather_lines<256><<<(n_lines + 255) / 256, 256, 0, st>>>(ws.line_cnt, ws.line_start, n_lines,
                                                                        (const uint4*)ws.stage, (uint4*)out, capacity,
                                                                        ws.line_desc, ws.counters, status, n, path);
    else
        k_scan_gather_lines<64><<<(n_lines + 63) / 64, 256, 0, st>>>(ws.line_cnt, ws.line_start, n_lines,
                                                                     (const uint4*)ws.stage, (uint4*)out, capacity,
                                                                     ws.line_desc, ws.counters, status, n, path);
    return 1;
}

// ---- K5 for unsorted input: LSD radix sort of (key40, index), 8 bits per pass, warp-private tiles -------------
static constexpr int kSortTile = 2048;     // elements per warp
static constexpr int kSortWarps = 8;

__device__ __forceinline__ uint64_t sort_count(const Counters* cnt, uint64_t max_clusters)
{
    const uint64_t c = cnt->n_clusters;
    return c < max_clusters ? c : max_clusters;
}

__global__ void k_sort_init(const uint4* __restrict__ compact, const Counters* cnt, uint64_t max_clusters,
                            uint64_t* __restrict__ key, uint32_t* __restrict__ idx)
{
    if (!cnt->unsorted) return;
    const uint64_t N = sort_count(cnt, max_clusters);
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const uint4 lo = compact[2 * i];
    key[i] = key40(lo.x, lo.y);
    idx[i] = (uint32_t)i;
}

__global__ void __launch_bounds__(kSortWarps * 32)
k_radix_hist(const uint64_t* __restrict__ key, const Counters* cnt, uint64_t max_clusters, int shift,
             uint32_t* __restrict__ ghist, uint32_t n_tiles)
{
    if (!cnt->unsorted) return;
    __shared__ uint32_t s_hist[kSortWarps][256];
    const unsigned lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t tile = blockIdx.x * kSortWarps + warp;
    const uint64_t N = sort_count(cnt, max_clusters);
    for (int d = lane; d < 256; d += 32) s_hist[warp][d] = 0;
    __syncwarp();
    if (tile < n_tiles) {
        const uint64_t b = (uint64_t)tile * kSortTile;
        for (int it = 0; it < kSortTile / 32; ++it) {
            const uint64_t i = b + (uint64_t)it * 32 + lane;
            if (i < N) atomicAdd(&s_hist[warp][(key[i] >> shift) & 0xffu], 1u);
        }
        __syncwarp();
        for (int d = lane; d < 256; d += 32) ghist[(size_t)d * n_tiles + tile] = s_hist[warp][d];
    }
}

__global__ void __launch_bounds__(kSortWarps * 32)
k_radix_scatter(const uint64_t* __restrict__ key_in, const uint32_t* __restrict__ idx_in,
                uint64_t* __restrict__ key_out, uint32_t* __restrict__ idx_out, const Counters* cnt,
                uint64_t max_clusters, int shift, const uint32_t* __restrict__ goff, uint32_t n_tiles)
{
    if (!cnt->unsorted) return;
    __shared__ uint32_t s_base[kSortWarps][256];
    const unsigned lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t tile = blockIdx.x * kSortWarps + warp;
    if (tile >= n_tiles) return;
    const uint64_t N = sort_count(cnt, max_clusters);
    for (int d = lane; d < 256; d += 32) s_base[warp][d] = goff[(size_t)d * n_tiles + tile];
    __syncwarp();
    const uint64_t b = (uint64_t)tile * kSortTile;
    for (int it = 0; it < kSortTile / 32; ++it) {
        const uint64_t i = b + (uint64_t)it * 32 + lane;
        const bool act = i < N;
        const unsigned am = __ballot_sync(0xffffffffu, act);
        if (am == 0) break;
        if (act) {
            const uint64_t k = key_in[i];
            const uint32_t d = (uint32_t)(k >> shift) & 0xffu;
            const unsigned peers = __match_any_sync(am, d);
            const uint32_t rank = (uint32_t)__popc(peers & ((1u << lane) - 1u));
            const uint32_t pos = s_base[warp][d] + rank;
            key_out[pos] = k;
            idx_out[pos] = idx_in[i];
            __syncwarp(am);
            if (rank == 0) s_base[warp][d] += (uint32_t)__popc(peers);
        }
        __syncwarp();
    }
}

__global__ void k_sort_gather(const uint4* __restrict__ compact, const uint32_t* __restrict__ idx,
                              const Counters* cnt, uint64_t max_clusters, uint4* __restrict__ out, uint64_t capacity)
{
    if (!cnt->unsorted) return;
    uint64_t N = sort_count(cnt, max_clusters);
    if (N > capacity) N = capacity;
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const uint32_t j = idx[i];
    out[2 * i] = compact[2 * (uint64_t)j];
    out[2 * i + 1] = compact[2 * (uint64_t)j + 1];
}

int launch_key_sort(const Workspace& ws, uint64_t max_clusters, uint32_t n_sort_tiles, tpc_cluster* out,
                    uint64_t capacity, cudaStream_t st)
{
    if (max_clusters == 0) return 0;
    int k = 0;
    const unsigned g256 = (unsigned)ceil_div_u64(max_clusters, 256);
    k_sort_init<<<g256, 256, 0, st>>>((const uint4*)ws.compact, ws.counters, max_clusters, ws.keyA, ws.idxA);
    ++k;
    uint64_t* kin = ws.keyA; uint64_t* kout = ws.keyB;
    uint32_t* iin = ws.idxA; uint32_t* iout = ws.idxB;
    const unsigned gt = (unsigned)ceil_div_u64(n_sort_tiles, kSortWarps);
    for (int pass = 0; pass < 5; ++pass) {
        const int shift = pass * 8;
        k_radix_hist<<<gt, kSortWarps * 32, 0, st>>>(kin, ws.counters, max_clusters, shift, ws.ghist, n_sort_tiles);
        k += 1 + launch_scan_u32(ws.ghist, ws.ghist, (uint64_t)256 * n_sort_tiles, ws.ghist_part, nullptr, st);
        k_radix_scatter<<<gt, kSortWarps * 32, 0, st>>>(kin, iin, kout, iout, ws.counters, max_clusters, shift,
                                                        ws.ghist, n_sort_tiles);
        ++k;
        uint64_t* tk = kin; kin = kout; kout = tk;
        uint32_t* ti = iin; iin = iout; iout = ti;
    }
    k_sort_gather<<<g256, 256, 0, st>>>((const uint4*)ws.compact, iin, ws.counters, max_clusters, (uint4*)out,
                                        capacity);
    return k + 1;
}

// ---- status ---------------------------------------------------------------------------------------------------
__global__ void k_finalize(const Counters* cnt, tpc_cf_status* status, uint64_t capacity, uint32_t path,
                           int hint_sorted, uint64_t n, uint64_t max_clusters)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    tpc_cf_status s;
    s.n_clusters = cnt->n_clusters;
    s.n_digits_used = n - cnt->n_bad;
    s.n_bad_digits = cnt->n_bad;
    s.overflow = s.n_clusters > capacity ? 1u : 0u;
    // unsorted input goes through the key sort, which holds at most the workspace's max_clusters records (A2): beyond
    // that only the first max_clusters peaks in digit order were kept (sorted), whatever the caller's capacity
    if (!hint_sorted && cnt->unsorted && s.n_clusters > max_clusters) s.overflow = 1u;
    s.path = path;
    if (hint_sorted && cnt->unsorted) {   // false DIGITS_SORTED promise: detected, no output (include/tpc_cf.h)
        s.n_clusters = 0;
        s.overflow = 0;
        s.path = 0;
    }
    *status = s;
}

int launch_finalize(const Workspace& ws, tpc_cf_status* status, uint64_t capacity, uint32_t path,
                    int hint_sorted, uint64_t n, uint64_t max_clusters, cudaStream_t st)
{
    k_finalize<<<1, 32, 0, st>>>(ws.counters, status, capacity, path, hint_sorted, n, max_clusters);
    return 1;
}

// ---- exclusive scan without any allocation: scratch in a file-scope device array ----------------------------------
// For callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
// the same three scan kernels as launch_scan_u32, with the per-block partial sums in a static device array instead of
// a caller-owned workspace.  Every GPU that loads the library holds the array (257 KB) until exit.
// In HOST code the array's name is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, resolved once per device with that device current (tpc_cf_scan_static_setup).
// All calls on a device share the array: it keeps the last call's partials, every call overwrites the entries it will
// read (partials [0, ceil(n / 1024)) by k_scan_reduce) before it reads them, so nothing has to start at zero — but two
// calls that overlap on the GPU (different streams, or graphs replayed concurrently) race on it.
static constexpr uint64_t kScanStaticMaxN = 1ull << 26;                       // elements per call
static constexpr uint32_t kScanStaticPartials = (uint32_t)(kScanStaticMaxN / kScanThreads) + 256u;
static __device__ __align__(256) uint32_t g_scan_static_partials[kScanStaticPartials];

static constexpr int kMaxDevices = 64;
static uint32_t* g_scan_static_ptr[kMaxDevices];     // device address of the array, per device (0 = not resolved)

}  // namespace tpccf

using namespace tpccf;

extern "C" uint64_t tpc_cf_scan_static_max_n(void) { return kScanStaticMaxN; }

extern "C" int tpc_cf_scan_static_setup(void)
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return TPC_CF_E_CUDA;
    if (g_scan_static_ptr[dev]) return TPC_CF_OK;
    uint32_t* p = nullptr;
    if (cudaGetSymbolAddress((void**)&p, g_scan_static_partials) != cudaSuccess || !p) {
        (void)cudaGetLastError();
        return TPC_CF_E_CUDA;
    }
    g_scan_static_ptr[dev] = p;
    return TPC_CF_OK;
}

extern "C" int tpc_cf_scan_u32_static(const uint32_t* in, uint32_t* out, uint64_t n, unsigned long long* total,
                                      void* stream)
{
    if (n && (!in || !out)) return TPC_CF_E_NULL;
    if (n > kScanStaticMaxN) return TPC_CF_E_CAPACITY;        // beyond the static scratch: use a handle's workspace
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) return TPC_CF_E_CUDA;
    if (!g_scan_static_ptr[dev]) {
        const int rc = tpc_cf_scan_static_setup();            // (callers that capture graphs call the set-up beforehand)
        if (rc != TPC_CF_OK) return rc;
    }
    cudaStream_t st = (cudaStream_t)stream;
    if (n == 0) {
        if (total && cudaMemsetAsync(total, 0, sizeof *total, st) != cudaSuccess) return TPC_CF_E_CUDA;
        return TPC_CF_OK;
    }
    (void)cudaGetLastError();
    launch_scan_u32(in, out, n, g_scan_static_ptr[dev], total, st);
    return cudaGetLastError() == cudaSuccess ? TPC_CF_OK : TPC_CF_E_CUDA;
}
