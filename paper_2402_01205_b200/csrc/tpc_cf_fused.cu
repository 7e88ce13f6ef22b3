// tpc_cf_fused.cu — fused path ("T3") for digits sorted by (sector,row,pad,time): the charge map never exists in HBM.
//
//   k_line_index   lower_bound of every (plane,pad) line in the digit array -> ws.line_start
//   k_fused_lines  one CTA per (plane, pad range).  The pad lines of the range stream through a ring of line slots in
//                  shared memory.  A line slot is the line of the charge map in compressed form:
//                     bm[w]   presence bitmap over time bins (bit t+32; one guard word each side = zero border, R2)
//                     pre[w]  index within the line of the first digit of bitmap word w (rank directory)
//                     tq[i]   (time | charge << 16) of the i-th digit of the line = upper word of the input record
//                  K1 (scatter) = building a slot from the line's digits, K2 = digit-centric 3x3 test against the
//                  slots of lines p-1, p, p+1, K4 = 5x5 window gathered from the five slots p-2..p+2, K0 = clearing
//                  the bitmap of the slot that leaves the ring.  Per step: S lines are processed, the next S lines
//                  are built and the S lines retired one step earlier are cleared, with ONE __syncthreads.
//                  Peaks are recorded as one bit per digit (peakmask) and their cluster at stage[j]; the shared
//                  compaction (tpc_cf_compact.cu) turns that into the ordered output (K3, K5).
//   The DIGITS_SORTED promise is verified here for free: every digit is checked once against the line (or gap) it
//   was found in; any violation raises Counters::unsorted and the run reports path 0.
#include "tpc_cf_internal.cuh"

namespace tpccf {

static constexpr int kFThreads = 256;
static constexpr int kS = 2;                    // lines per step
static constexpr int kSlots = 3 * kS + 4;       // process window S+4, build S, clear S
static constexpr int kPeakQ = 512;              // CTA peak queue entries per step

__device__ __forceinline__ uint32_t key24_of(uint32_t w0)
{
    return ((w0 & 0xffu) << 16) | (w0 & 0xff00u) | ((w0 >> 16) & 0xffu);
}

__global__ void __launch_bounds__(256)
k_line_index(const uint2* __restrict__ digits, uint32_t n, Geo g, uint32_t* __restrict__ line_start)
{
    const uint32_t total = g.n_planes * g.LS + 1;
    const uint32_t e = blockIdx.x * 256 + threadIdx.x;
    if (e >= total) return;
    if (e == total - 1) { line_start[e] = n; return; }
    const uint32_t plane = e / g.LS, p = e % g.LS;
    const uint32_t s = plane / g.n_rows, r = plane % g.n_rows;
    const uint32_t target = (s << 16) | (r << 8) | p;
    uint32_t lo = 0, hi = n;
    while (lo < hi) {
        const uint32_t mid = lo + ((hi - lo) >> 1);
        if (key24_of(__ldg(&digits[mid].x)) < target) lo = mid + 1; else hi = mid;
    }
    line_start[e] = lo;
}

struct SlotView {
    uint32_t* bm;
    uint32_t* tq;
    uint16_t* pre;
};

// charges of the window t-H..t+H of one line slot (0 where no digit), c[k] for time t-H+k
template <int H>
__device__ __forceinline__ void window(const SlotView& sv, uint32_t cap, const uint2* __restrict__ digits,
                                       uint32_t lbeg, uint32_t n, int t, int (&c)[2 * H + 1])
{
    const int b = t + 32 - H;
    const int w = b >> 5, s = b & 31;
    const uint32_t lo = sv.bm[w], hi = sv.bm[w + 1];
    uint32_t bits = __funnelshift_r(lo, hi, s) & ((1u << (2 * H + 1)) - 1u);
#pragma unroll
    for (int k = 0; k < 2 * H + 1; ++k) c[k] = 0;
    if (!bits) return;
    uint32_t idx = (lo >> s) ? (uint32_t)sv.pre[w] + (uint32_t)__popc(lo & ((1u << s) - 1u)) : (uint32_t)sv.pre[w + 1];
#pragma unroll
    for (int k = 0; k < 2 * H + 1; ++k) {
        if (bits & (1u << k)) {
            uint32_t v;
            if (idx < cap) v = sv.tq[idx];
            else { uint32_t gi = lbeg + idx; gi = gi < n ? gi : n - 1; v = __ldg(&digits[gi].y); }
            c[k] = (int)(v >> 16);
            ++idx;
        }
    }
}

__global__ void __launch_bounds__(kFThreads, 4)
k_fused_lines(const uint2* __restrict__ digits, uint32_t n, Geo g, const uint32_t* __restrict__ line_start,
              uint32_t pads_per_unit, uint32_t units_per_plane, uint32_t wpl, uint32_t cap,
              uint32_t q_peak_min, uint32_t q_gate, Counters* cnt, uint32_t* __restrict__ peakmask,
              uint4* __restrict__ stage)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t s_ls[260];       // line starts of this plane: s_ls[p] for p = 0..max_pads, then next plane's start
    __shared__ int s_unsorted;
    __shared__ uint32_t s_wq[kFThreads / 32][64];   // per-warp survivor queues (stage A -> B)
    __shared__ uint32_t s_pq[kPeakQ];               // CTA peak queue (stage B -> C)
    __shared__ uint32_t s_npk[2];                   // its fill count, double-buffered by step parity

    const uint32_t plane = blockIdx.x / units_per_plane, unit = blockIdx.x % units_per_plane;
    const uint32_t sector = plane / g.n_rows, row = plane % g.n_rows;
    const int P = (int)g.npads[row];
    const int pa = (int)(unit * pads_per_unit);
    const int pb = min(pa + (int)pads_per_unit, P);
    const int T = (int)g.n_time;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t w0_base = sector | (row << 8);

    // slot views
    const uint32_t slot_words = wpl + cap + ((wpl + 1) >> 1);
    uint32_t* sm = reinterpret_cast<uint32_t*>(smem_raw);
    auto slot_of = [&](int p) -> SlotView {
        const int v = (p - pa + 2 + kSlots) % kSlots;     // p >= pa - 2 - kSlots always
        uint32_t* base = sm + (uint32_t)v * slot_words;
        SlotView sv;
        sv.bm = base; sv.tq = base + wpl; sv.pre = reinterpret_cast<uint16_t*>(base + wpl + cap);
        return sv;
    };

    for (int i = tid; i <= (int)g.LS; i += kFThreads) s_ls[i] = line_start[plane * g.LS + i];
    if (tid == 0) { s_unsorted = 0; s_npk[0] = 0u; s_npk[1] = 0u; }
    for (uint32_t i = tid; i < kSlots * slot_words; i += kFThreads) sm[i] = 0u;
    __syncthreads();

    if (pa >= P && unit != 0) return;    // nothing in this pad range (rows with fewer pads)

    bool bad_order = false;
    // monotone line starts: a garbage index from unsorted input must not produce negative lengths or unbounded work
    for (int i = tid; i < (int)g.LS; i += kFThreads) if (s_ls[i] > s_ls[i + 1]) bad_order = true;
    if (__syncthreads_or(bad_order ? 1 : 0)) {
        if (tid == 0) atomicOr(&cnt->unsorted, 1u);
        return;
    }

    // gap of the plane: digits with pad >= npads[row] (or a row/sector beyond the geometry) — all invalid (R11)
    if (unit == 0) {
        const uint32_t gb = s_ls[P], ge = s_ls[g.LS];
        if (ge > gb) {
            for (uint32_t j = gb + tid; j < ge; j += kFThreads) {
                const uint2 d = __ldg(digits + j);
                if (digit_valid(g, d.x, d.y)) bad_order = true;     // a valid digit outside every line: not sorted
            }
            if (tid == 0) atomicAdd(&cnt->n_bad, (unsigned long long)(ge - gb));
        }
    }

    // ---- K1: build the slots of lines [b0,b1) (clipped to existing lines) ---------------------------------------
    auto build = [&](int b0, int b1) {
        b0 = max(b0, 0); b1 = min(b1, min(P, pb + 2));
        if (b0 >= b1) return;
        const uint32_t jb = s_ls[b0], je = s_ls[b1];
        if (je <= jb) return;
        for (uint32_t j0 = jb; j0 < je; j0 += kFThreads) {      // uniform trip count: the shuffles need whole warps
            const uint32_t j = j0 + tid;
            const bool act = j < je;
            uint2 d = make_uint2(0, 0);
            if (act) d = __ldg(digits + j);
            // previous digit (lane-1, or a load for lane 0 / first of the range)
            uint32_t pw0 = __shfl_up_sync(0xffffffffu, d.x, 1), pw1 = __shfl_up_sync(0xffffffffu, d.y, 1);
            if (act && lane == 0 && j > jb) { const uint2 e = __ldg(digits + j - 1); pw0 = e.x; pw1 = e.y; }
            if (!act) continue;
            const int p = (int)((d.x >> 16) & 0xffu);
            const uint32_t t = d.y & 0xffffu;
            const bool owner = p >= pa && p < pb;
            if ((d.x & 0xffffu) != w0_base || p < b0 || p >= b1) { bad_order = true; continue; }
            const uint32_t lbeg = s_ls[p];
            if (j < lbeg || j >= s_ls[p + 1]) { bad_order = true; continue; }
            const uint32_t jl = j - lbeg;
            const bool first_of_line = (jl == 0);
            const uint32_t pt = pw1 & 0xffffu;
            if (!first_of_line && pt >= t) bad_order = true;          // not strictly ascending (or a duplicate cell)
            if (t >= (uint32_t)T || (d.y >> 16) == 0u) { if (owner) atomicAdd(&cnt->n_bad, 1ull); }
            if (t >= (uint32_t)T) continue;
            const SlotView sv = slot_of(p);
            const uint32_t bw = (t + 32u) >> 5;
            atomicOr(&sv.bm[bw], 1u << (t & 31u));
            if (first_of_line || ((pt + 32u) >> 5) != bw) sv.pre[bw] = (uint16_t)jl;
            if (jl < cap) sv.tq[jl] = d.y;
        }
    };

    // ---- K0: clear the bitmaps of lines [c0,c1) ------------------------------------------------------------------
    auto clear = [&](int c0, int c1) {
        for (int p = c0; p < c1; ++p) {
            if (p < pa - 2) continue;
            const SlotView sv = slot_of(p);
            for (uint32_t i = tid; i < wpl; i += kFThreads) sv.bm[i] = 0u;
        }
    };

    // ---- K2 + K4: digit-centric peak test and moments for lines [l0,l1) -------------------------------------------
    // Peaks are ~1 in 20 digits, so the work is done in three dense stages instead of one divergent pass:
    //   A (every digit)     own-line test against the adjacent digits of the line; survivors -> per-warp queue
    //   B (survivors, ~25%) lines p-1 / p+1 through the bitmap windows; peaks -> CTA queue + peakmask bit
    //   C (peaks, ~5%)      5x5 window from the five slots, gated sums, record -> stage[j]   (after a barrier)
    auto locate = [&](uint32_t j, int l0, int l1, int& p, uint32_t& jl, uint32_t& len) {
        p = l0;
#pragma unroll
        for (int i = 1; i < kS; ++i) if (l0 + i < l1 && j >= s_ls[l0 + i]) p = l0 + i;
        const uint32_t lbeg = s_ls[p];
        jl = j - lbeg;
        len = s_ls[p + 1] - lbeg;
    };
    auto fetch = [&](const SlotView& sv, uint32_t j, uint32_t jl) -> uint32_t {
        if (jl < cap) return sv.tq[jl];
        return __ldg(&digits[min(j, n - 1)].y);
    };
    auto moments = [&](uint32_t j, int p, int t) {
        int c[5][5];
#pragma unroll
        for (int a = 0; a < 5; ++a) {
            const int pp = p + a - 2;
            if (pp >= 0 && pp < P) {
                window<2>(slot_of(pp), cap, digits, s_ls[pp], n, t, c[a]);
            } else {
#pragma unroll
                for (int b = 0; b < 5; ++b) c[a][b] = 0;
            }
        }
        const ClusterWords r = cluster_from_window(c, w0_base | ((uint32_t)p << 16), (uint32_t)t, q_gate);
        stage[2 * (size_t)j] = r.lo;
        stage[2 * (size_t)j + 1] = r.hi;
    };
    auto stage_b = [&](bool act, uint32_t j, int l0, int l1, int par) {
        bool peak = false;
        int p = l0, t = 0;
        if (act) {
            uint32_t jl, len;
            locate(j, l0, l1, p, jl, len);
            const uint32_t self = fetch(slot_of(p), j, jl);
            t = (int)(self & 0xffffu);
            const uint32_t q = self >> 16;
            peak = true;
            if (p > 0) {                                                    // line p-1: earlier, strict (R1)
                int c[3];
                window<1>(slot_of(p - 1), cap, digits, s_ls[p - 1], n, t, c);
                peak = q > (uint32_t)c[0] && q > (uint32_t)c[1] && q > (uint32_t)c[2];
            }
            if (peak && p + 1 < P) {                                        // line p+1: later, >=
                int c[3];
                window<1>(slot_of(p + 1), cap, digits, s_ls[p + 1], n, t, c);
                peak = q >= (uint32_t)c[0] && q >= (uint32_t)c[1] && q >= (uint32_t)c[2];
            }
        }
        const unsigned pm = __ballot_sync(0xffffffffu, peak);
        if (pm == 0) return;
        const int leader = __ffs(pm) - 1;
        uint32_t base = 0;
        if (lane == leader) base = atomicAdd(&s_npk[par], (uint32_t)__popc(pm));
        base = __shfl_sync(0xffffffffu, base, leader);
        if (peak) {
            atomicOr(&peakmask[j >> 5], 1u << (j & 31u));
            const uint32_t slot = base + (uint32_t)__popc(pm & ((1u << lane) - 1u));
            if (slot < kPeakQ) s_pq[slot] = j;
            else moments(j, p, t);                                          // queue full: do it here (rare)
        }
    };
    auto phase1 = [&](int l0, int l1, int par) {
        l1 = min(l1, pb);
        if (l0 >= l1) return;
        const uint32_t jb = s_ls[l0], je = s_ls[l1];
        if (je <= jb) return;
        uint32_t* wq = s_wq[warp];
        uint32_t wcount = 0;                                                // warp-uniform
        for (uint32_t j0 = (jb & ~31u) + 32u * warp; j0 < je; j0 += kFThreads) {
            const uint32_t j = j0 + lane;
            bool surv = false;
            if (j >= jb && j < je) {
                int p; uint32_t jl, len;
                locate(j, l0, l1, p, jl, len);
                const SlotView sv = slot_of(p);
                const uint32_t self = fetch(sv, j, jl);
                const int t = (int)(self & 0xffffu);
                const uint32_t q = self >> 16;
                if (q >= q_peak_min && t < T) {
                    // own line: the neighbours in time are the adjacent digits of the line
                    const uint32_t prev = jl > 0 ? fetch(sv, j - 1, jl - 1) : 0u;
                    const uint32_t next = jl + 1 < len ? fetch(sv, j + 1, jl + 1) : 0u;
                    const uint32_t qm = (jl > 0 && (int)(prev & 0xffffu) == t - 1) ? (prev >> 16) : 0u;
                    const uint32_t qp = (jl + 1 < len && (int)(next & 0xffffu) == t + 1 && t + 1 < T) ? (next >> 16) : 0u;
                    surv = q > qm && q >= qp;                               // R1: (0,-1) strict, (0,+1) >=
                }
            }
            const unsigned m = __ballot_sync(0xffffffffu, surv);
            if (surv) wq[wcount + (uint32_t)__popc(m & ((1u << lane) - 1u))] = j;
            wcount += (uint32_t)__popc(m);
            __syncwarp();
            if (wcount >= 32u) {
                stage_b(true, wq[lane], l0, l1, par);
                const uint32_t mv = (lane + 32u < wcount) ? wq[lane + 32u] : 0u;
                __syncwarp();
                if (lane + 32u < wcount) wq[lane] = mv;
                wcount -= 32u;
                __syncwarp();
            }
        }
        if (wcount) stage_b((uint32_t)lane < wcount, (uint32_t)lane < wcount ? wq[lane] : 0u, l0, l1, par);
    };
    auto phase2 = [&](int l0, int l1, int par) {
        l1 = min(l1, pb);
        const uint32_t np = min(s_npk[par], (uint32_t)kPeakQ);
        for (uint32_t i = tid; i < np; i += kFThreads) {
            const uint32_t j = s_pq[i];
            int p; uint32_t jl, len;
            locate(j, l0, l1, p, jl, len);
            const uint32_t self = fetch(slot_of(p), j, jl);
            moments(j, p, (int)(self & 0xffffu));
        }
        if (tid == 0) s_npk[par ^ 1] = 0u;
    };

    // prologue: lines needed by step 0
    build(pa - 2, pa + kS + 2);
    __syncthreads();
    int par = 0;
    for (int l0 = pa; l0 < pb; l0 += kS, par ^= 1) {
        phase1(l0, l0 + kS, par);
        __syncthreads();
        phase2(l0, l0 + kS, par);
        build(l0 + kS + 2, l0 + 2 * kS + 2);
        clear(l0 - kS - 2, l0 - 2);
        __syncthreads();
    }
    if (bad_order) s_unsorted = 1;
    __syncthreads();
    if (tid == 0 && s_unsorted) atomicOr(&cnt->unsorted, 1u);
}

int launch_fused_sorted(const Geo& g, const Workspace& ws, const tpc_digit* digits, uint64_t n,
                        uint32_t q_peak_min, uint32_t q_gate, cudaStream_t st,
                        cudaEvent_t ev_k0, cudaEvent_t ev_k1)
{
    if (n == 0) return 0;
    int k = 0;
    const uint32_t entries = g.n_planes * g.LS + 1;
    cudaMemsetAsync(ws.peakmask, 0, (size_t)ceil_div_u64(n, 32) * 4, st);
    k_line_index<<<(entries + 255) / 256, 256, 0, st>>>((const uint2*)digits, (uint32_t)n, g, ws.line_start);
    ++k;

    // launch shape: pad range per unit, tq capacity per slot from the mean line length (host-known)
    uint64_t total_pads = 0;
    for (uint32_t r = 0; r < g.n_rows; ++r) total_pads += g.npads[r];
    total_pads *= g.n_sectors;
    const double mean_len = (double)n / (double)(total_pads ? total_pads : 1);
    const uint32_t wpl = (g.n_time + 31) / 32 + 3;          // guard word below, >= 2 words above the last bin
    uint32_t cap = (uint32_t)(mean_len * 1.5) + 64;
    cap = (cap + 31u) & ~31u;
    const uint32_t max_smem = 52 * 1024;                     // 4 CTAs per SM (+ ~1 KB static + 1 KB reserved each)
    const uint32_t fixed = kSlots * (wpl * 4 + ((wpl + 1) / 2) * 4);
    if (fixed + kSlots * cap * 4 > max_smem) cap = fixed < max_smem ? ((max_smem - fixed) / (kSlots * 4)) & ~31u : 0;
    const uint32_t smem = fixed + kSlots * cap * 4;
    const uint32_t pads_per_unit = (g.max_pads + 1) / 2;
    const uint32_t upp = (g.max_pads + pads_per_unit - 1) / pads_per_unit;
    static bool attr_set = false;
    if (!attr_set) {
        cudaError_t e = cudaFuncSetAttribute(k_fused_lines, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e != cudaSuccess) return TPC_CF_E_CUDA;
        attr_set = true;
    }
    if (ev_k0) cudaEventRecord(ev_k0, st);
    k_fused_lines<<<g.n_planes * upp, kFThreads, smem, st>>>((const uint2*)digits, (uint32_t)n, g, ws.line_start,
                                                             pads_per_unit, upp, wpl, cap, q_peak_min, q_gate,
                                                             ws.counters, ws.peakmask, (uint4*)ws.stage);
    if (ev_k1) cudaEventRecord(ev_k1, st);
    ++k;
    return k;
}

}  // namespace tpccf
