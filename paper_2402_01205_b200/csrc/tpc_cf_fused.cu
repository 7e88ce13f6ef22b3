// tpc_cf_fused.cu — fused path ("T3") for digits sorted by (sector,row,pad,time): the charge map never exists in HBM.
//
//   k_plane_index, k_line_index   two-level lower_bound of every (plane,pad) line in the digit array -> ws.line_start
//   k_fused_lines  one CTA (8 warps) per (plane, pad range).  The pad lines of the range stream through a ring of line
//                  slots in shared memory.  A line slot is one line of the charge map in compressed form:
//                     bm[w]   presence bitmap over time bins (bit t+32; guard words = zero border in time, R2)
//                     pre[w]  index within the line of the first digit of bitmap word w (rank directory)
//                     tq[i]   (time | charge << 16) of the i-th digit of the line = upper word of the input record
//                  One WARP owns one LINE at a time, so line geometry and slot pointers are warp-uniform:
//                   K1 build    the warp zeroes its slot's bitmap, then streams the line's digits into bm/pre/tq
//                               (this is also K0: a slot is cleaned by the warp that reuses it)
//                   K2 stage A  own-line test of every digit against the adjacent digits of the line (shuffles)
//                      stage B  survivors (~25 %) against lines p-1 / p+1 through 3-bit bitmap windows
//                   K4 stage C  peaks (~5 %) gathered into a per-warp queue; 5x5 window from the five slots p-2..p+2,
//                               gated sums, record -> stage[j]
//                  Step = 8 lines, one barrier: each warp prefetches (cp.async) the line it will build, runs A+B+C on
//                  its current line, then rebuilds the slot of a line that left the ring.
//                  The k-th peak of a line (time order) goes to stage[line_start + k] and the line's peak count to
//                  line_cnt[]; a scan over the line counts and a per-line copy give the ordered output (K3, K5).
//   The DIGITS_SORTED promise is verified here for free: every digit is checked once against the line (or gap) it
//   was found in; any violation raises Counters::unsorted and the run reports path 0.
#include "tpc_cf_internal.cuh"

namespace tpccf {

static constexpr int kFThreads = 256;
static constexpr int kWarps = kFThreads / 32;
static constexpr int kS = kWarps;               // lines per step: one per warp
static constexpr int kSlots = 2 * kS + 4;       // lines l0-2 .. l0+S+1 in use, next S being built

__device__ __forceinline__ uint32_t key24_of(uint32_t w0)
{
    return ((w0 & 0xffu) << 16) | (w0 & 0xff00u) | ((w0 >> 16) & 0xffu);
}

// lower_bound of a 24-bit (sector,row,pad) key in digits[lo, hi)
__device__ __forceinline__ uint32_t lower_bound_key(const uint2* __restrict__ digits, uint32_t lo, uint32_t hi,
                                                    uint32_t target)
{
    while (lo < hi) {
        const uint32_t mid = lo + ((hi - lo) >> 1);
        if (key24_of(__ldg(&digits[mid].x)) < target) lo = mid + 1; else hi = mid;
    }
    return lo;
}

// the same result by an 8-ary search: 7 independent probes per step instead of one (the search is bound by the latency
// of dependent loads: 6 steps instead of 16 for a plane of 40 k digits)
__device__ __forceinline__ uint32_t lower_bound_key8(const uint2* __restrict__ digits, uint32_t lo, uint32_t hi,
                                                     uint32_t target)
{
    while (hi - lo > 8u) {
        const uint32_t step = (hi - lo) >> 3;
        uint32_t k[7];
#pragma unroll
        for (int i = 0; i < 7; ++i) k[i] = key24_of(__ldg(&digits[lo + (uint32_t)(i + 1) * step].x));
        // first pivot whose key is >= target bounds the answer from above; the one before it from below
        uint32_t nlo = lo, nhi = hi;
#pragma unroll
        for (int i = 6; i >= 0; --i) if (k[i] >= target) nhi = lo + (uint32_t)(i + 1) * step;
#pragma unroll
        for (int i = 0; i < 7; ++i) if (k[i] < target) nlo = lo + (uint32_t)(i + 1) * step + 1u;
        if (nlo > nhi) nlo = nhi;        // keys not ascending (false DIGITS_SORTED promise): stay in bounds, terminate
        lo = nlo; hi = nhi;
    }
    return lower_bound_key(digits, lo, hi, target);
}

// level 1: first digit of every plane (entry p = 0 of each plane; the final entry is n)
__global__ void __launch_bounds__(256)
k_plane_index(const uint2* __restrict__ digits, uint32_t n, Geo g, uint32_t* __restrict__ line_start, Counters* cnt)
{
    const uint32_t plane = blockIdx.x * 256 + threadIdx.x;
    if (plane == 0) { cnt->n_bad = 0ull; cnt->n_used = 0ull; cnt->n_clusters = 0ull; cnt->unsorted = 0u; cnt->n_share = 0u; }
    if (plane > g.n_planes) return;
    if (plane == g.n_planes) { line_start[(size_t)g.n_planes * g.LS] = n; return; }
    const uint32_t s = plane / g.n_rows, r = plane % g.n_rows;
    line_start[(size_t)plane * g.LS] = lower_bound_key8(digits, 0, n, (s << 16) | (r << 8));
}

// level 2: the lines of a plane, searched inside the plane's own range
__global__ void __launch_bounds__(256)
k_line_index(const uint2* __restrict__ digits, uint32_t n, Geo g, uint32_t* __restrict__ line_start,
             uint32_t* __restrict__ line_cnt, unsigned long long* __restrict__ line_desc, Counters* cnt)
{
    // cnt != NULL: small input, no k_plane_index in front: every line is searched in the whole array (as many probes as
    // the two-level search for small n, one launch less), and this kernel zeroes the run's counters as well
    const bool direct = cnt != nullptr;
    const uint32_t total = g.n_planes * g.LS;
    const uint32_t e = blockIdx.x * 256 + threadIdx.x;
    if (direct && e == 0) { cnt->n_bad = 0ull; cnt->n_used = 0ull; cnt->n_clusters = 0ull; cnt->unsorted = 0u; cnt->n_share = 0u; }
    if (direct && e == total) line_start[total] = n;
    // per-run state of the compaction: peak counts (pads beyond npads[row] stay 0) and scan descriptors
    if (e <= total) line_cnt[e] = 0u;
    if (e <= (total + 63u) / 64u) line_desc[e] = 0ull;
    if (e >= total) return;
    const uint32_t plane = e / g.LS, p = e % g.LS;
    if (p == 0 && !direct) return;                        // written by k_plane_index
    const uint32_t s = plane / g.n_rows, r = plane % g.n_rows;
    uint32_t lo = 0, hi = n;
    if (!direct) {
        lo = line_start[(size_t)plane * g.LS]; hi = line_start[(size_t)(plane + 1) * g.LS];
        if (hi < lo || hi > n) { lo = 0; hi = n; }        // unsorted input: stay in bounds, the fused kernel reports it
    }
    line_start[e] = lower_bound_key(digits, lo, hi, (s << 16) | (r << 8) | p);   // (8-ary measured slower here: 122 vs 100 us — request-bound, not latency-bound)
}

// Slot layout (warp-uniform).
struct Ring {
    uint32_t* sm;          // base of the dynamic shared memory
    uint32_t slot_words;   // words per slot (multiple of 4)
    uint32_t wpl;          // bitmap words per line (multiple of 4)
    uint32_t cap;          // tq entries per slot (multiple of 128; longer lines read their tail from global memory)
    uint32_t pre_words;    // words of the rank directory (wpl uint16, padded to a multiple of 4 words)
    __device__ __forceinline__ uint32_t* slot(int v) const { return sm + (uint32_t)v * slot_words; }
};

// ring index of the line at distance d (|d| < kSlots) from the line whose ring index is v0
__device__ __forceinline__ int ring_at(int v0, int d)
{
    int v = v0 + d;
    v += (v < 0) ? kSlots : 0;
    v -= (v >= kSlots) ? kSlots : 0;
    return v;
}

// charges of the window t-H..t+H of one line slot (0 where no digit): c[k] is time t-H+k.  Branch-free except for the
// rare tail of a line longer than cap, read from the digit array (gl = global index of the line's first digit).
template <int H>
__device__ __forceinline__ void window(const Ring& rg, const uint32_t* __restrict__ slot,
                                       const uint2* __restrict__ digits, uint32_t gl, uint32_t n, int t,
                                       int (&c)[2 * H + 1])
{
    const uint32_t* tq = slot + rg.wpl;
    const uint16_t* pre = reinterpret_cast<const uint16_t*>(slot + rg.wpl + rg.cap);
    const int b = t + 32 - H;
    const int w = b >> 5, s = b & 31;
    const uint32_t lo = slot[w], hi = slot[w + 1];
    const uint32_t bits = __funnelshift_r(lo, hi, s) & ((1u << (2 * H + 1)) - 1u);
    const uint32_t p0 = pre[w], p1 = pre[w + 1];
    const uint32_t idx = (lo >> s) ? p0 + (uint32_t)__popc(lo & ((1u << s) - 1u)) : p1;
    if (bits == 0u) {
#pragma unroll
        for (int k = 0; k < 2 * H + 1; ++k) c[k] = 0;
    } else if (idx + (uint32_t)__popc(bits) <= rg.cap) {          // all present cells are in the staged tq area
#pragma unroll
        for (int k = 0; k < 2 * H + 1; ++k) {
            const uint32_t v = tq[idx + (uint32_t)__popc(bits & ((1u << k) - 1u))];
            c[k] = ((bits >> k) & 1u) ? (int)(v >> 16) : 0;
        }
    } else {
#pragma unroll
        for (int k = 0; k < 2 * H + 1; ++k) {
            const uint32_t ik = idx + (uint32_t)__popc(bits & ((1u << k) - 1u));
            uint32_t v = tq[min(ik, rg.cap - 1u)];
            const bool present = (bits >> k) & 1u;
            if (present && ik >= rg.cap) v = __ldg(&digits[min(gl + ik, n - 1u)].y);
            c[k] = present ? (int)(v >> 16) : 0;
        }
    }
}

__global__ void __launch_bounds__(kFThreads, 2)
k_fused_lines(const uint2* __restrict__ digits, uint32_t n, Geo g, const uint32_t* __restrict__ line_start,
              uint32_t pads_per_unit, uint32_t units_per_plane, uint32_t wpl, uint32_t cap,
              uint32_t q_peak_min, uint32_t q_gate, Variant var, Counters* cnt, uint32_t* __restrict__ line_cnt,
              uint4* __restrict__ stage)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t s_ls[260];          // line starts of this plane: s_ls[p], p = 0..max_pads, then next plane's start
    __shared__ uint32_t s_wq[kWarps][64];   // per-warp survivor queues (stage A -> B): index within the warp's line
    __shared__ uint32_t s_pq[kWarps][64];   // per-warp peak queues (stage B -> C): index within the warp's line
    __shared__ int s_unsorted;

    const uint32_t plane = blockIdx.x / units_per_plane, unit = blockIdx.x % units_per_plane;
    const uint32_t sector = plane / g.n_rows, row = plane % g.n_rows;
    const int P = (int)g.npads[row];
    const int pa = (int)(unit * pads_per_unit);
    const int pb = min(pa + (int)pads_per_unit, P);
    const int T = (int)g.n_time;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t w0_base = sector | (row << 8);

    Ring rg;
    rg.sm = reinterpret_cast<uint32_t*>(smem_raw);
    rg.wpl = wpl; rg.cap = cap;
    rg.pre_words = ((wpl >> 1) + 3u) & ~3u;
    rg.slot_words = wpl + cap + rg.pre_words + (cap >> 5);   // bm | tq | pre | stage-A bits

    for (int i = tid; i <= (int)g.LS; i += kFThreads) s_ls[i] = line_start[plane * g.LS + i];
    if (tid == 0) s_unsorted = 0;
    {   // every slot starts as an empty line (lines outside the plane keep this state: zero border in pad, R2)
        uint4* z = reinterpret_cast<uint4*>(rg.sm);
        const uint32_t nz = (kSlots * rg.slot_words) >> 2;
        for (uint32_t i = tid; i < nz; i += kFThreads) z[i] = make_uint4(0, 0, 0, 0);
    }
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

    const int blo = max(pa - 2, 0), bhi = min(P, pb + 2);   // lines this unit ever builds

    // tq entry jl of line p (slot given); the tail beyond cap comes from the digit array
    auto fetch = [&](const uint32_t* slot, uint32_t gl, uint32_t jl) -> uint32_t {
        if (jl < rg.cap) return slot[rg.wpl + jl];
        return __ldg(&digits[min(gl + jl, n - 1u)].y);
    };

    // ---- prefetch for K1: the (time|charge) words of line p go straight into the tq area of slot v with cp.async ----
    // (issued at the top of a step by the warp that builds the line after the step's first barrier)
    // The key words (sector,row,pad) are staged too, into this warp's own buffer, when with_x is set: the build then
    // verifies every digit's line without a single exposed global load.
    uint32_t* xst = rg.sm + kSlots * rg.slot_words + (uint32_t)warp * rg.cap;
    auto prefetch_line = [&](int p, int v, bool with_x) {
        if (p < blo || p >= bhi) return;
        const uint32_t lbeg = s_ls[p], len = s_ls[p + 1] - lbeg;
        const uint32_t m = min(len, rg.cap);
        const uint32_t dst = (uint32_t)__cvta_generic_to_shared(rg.slot(v) + rg.wpl);
        const uint32_t dsx = (uint32_t)__cvta_generic_to_shared(xst);
        for (uint32_t jl = lane; jl < m; jl += 32) {
            asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst + 4u * jl), "l"(&digits[lbeg + jl].y) : "memory");
            if (with_x)
                asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dsx + 4u * jl), "l"(&digits[lbeg + jl].x) : "memory");
        }
        asm volatile("cp.async.commit_group;" ::: "memory");
    };

    // ---- K0 + K1: this warp (re)builds the slot v of line p from the line's digits -----------------------------------
    // staged: the tq words [0, min(len,cap)) were already copied by prefetch_line.
    auto build_line = [&](int p, int v, bool staged, bool xstaged) {
        uint32_t* slot = rg.slot(v);
        {
            uint4* z = reinterpret_cast<uint4*>(slot);
            for (uint32_t x = lane; x < (rg.wpl >> 2); x += 32) z[x] = make_uint4(0, 0, 0, 0);
        }
        if (staged) asm volatile("cp.async.wait_all;" ::: "memory");
        __syncwarp();
        if (p < blo || p >= bhi) return;                    // a line outside the plane / the halo: stays empty
        const uint32_t lbeg = s_ls[p], len = s_ls[p + 1] - lbeg;
        // 32-bit shared-window addresses for the bitmap and the rank directory (red.shared / st.shared below)
        const uint32_t a_bm = (uint32_t)__cvta_generic_to_shared(slot);
        const uint32_t a_pre = a_bm + 4u * (rg.wpl + rg.cap);
        const uint32_t w0_line = w0_base | ((uint32_t)p << 16);
        const bool owner = p >= pa && p < pb;
        uint32_t* sbm = slot + rg.wpl + rg.cap + rg.pre_words;   // stage-A result: one bit per digit index < cap
        // (time|charge) word of digit jl: from the staged tq area, else from the digit array (and into tq)
        const bool fast = staged && xstaged && len <= rg.cap;   // the common case: both words of every digit are staged
        auto load_y = [&](uint32_t jl) -> uint32_t {
            if (fast) return jl < len ? slot[rg.wpl + jl] : 0u;
            if (jl >= len) return 0u;
            if (staged && jl < rg.cap) return slot[rg.wpl + jl];
            const uint32_t y = __ldg(&digits[lbeg + jl].y);
            if (jl < rg.cap) slot[rg.wpl + jl] = y;
            return y;
        };
        auto load_x = [&](uint32_t jl) -> uint32_t {
            if (fast) return jl < len ? xst[jl] : 0u;
            if (jl >= len) return 0u;
            if (xstaged && jl < rg.cap) return xst[jl];
            return __ldg(&digits[lbeg + jl].x);
        };
        uint32_t carry = 0;                                 // tq word of the digit before this chunk
        uint32_t mysbm = 0u;
        uint32_t xn = load_x(lane);                         // both words are loaded one chunk ahead
        uint32_t yn = load_y(lane);
        for (uint32_t c0 = 0; c0 < len; c0 += 32) {
            const uint32_t jl = c0 + lane;
            const bool act = jl < len;
            const uint32_t dx = xn, dy = yn;
            xn = load_x(jl + 32);
            yn = load_y(jl + 32);
            uint32_t prevy = __shfl_up_sync(0xffffffffu, dy, 1);
            uint32_t nexty = __shfl_down_sync(0xffffffffu, dy, 1);
            const uint32_t ny0 = __shfl_sync(0xffffffffu, yn, 0);
            if (lane == 0) prevy = carry;
            if (lane == 31) nexty = ny0;
            carry = __shfl_sync(0xffffffffu, dy, 31);
            const uint32_t t = dy & 0xffffu, pt = prevy & 0xffffu, q = dy >> 16;
            const bool first = (jl == 0);
            const bool ok = act && (dx & 0x00ffffffu) == w0_line;
            if (act && (!ok || (!first && pt >= t))) bad_order = true;   // wrong line, not ascending, or duplicate cell
            const bool valid = ok && t < (uint32_t)T;
            const unsigned mbad = __ballot_sync(0xffffffffu, ok && (!valid || q == 0u));   // R11, rare
            if (mbad != 0u && owner && lane == 0) atomicAdd(&cnt->n_bad, (unsigned long long)__popc(mbad));
            if (valid) {
                const uint32_t bw = (t + 32u) >> 5;
                asm volatile("red.shared.or.b32 [%0], %1;" ::"r"(a_bm + 4u * bw), "r"(1u << (t & 31u)) : "memory");
                if (first || ((pt + 32u) >> 5) != bw)
                    asm volatile("st.shared.u16 [%0], %1;" ::"r"(a_pre + 2u * bw), "h"((unsigned short)jl) : "memory");
            }
            // K2 stage A, done here because only the line itself is needed: the neighbours in time are the adjacent
            // digits of the line (an absent one reads as charge 0).  R1: (0,-1) strict, (0,+1) >=
            const uint32_t qm = (pt + 1u == t && !first) ? (prevy >> 16) : 0u;
            const uint32_t qp = ((nexty & 0xffffu) == t + 1u && t + 1u < (uint32_t)T) ? (nexty >> 16) : 0u;
            const unsigned sm = __ballot_sync(0xffffffffu, valid && q >= q_peak_min && q > qm && q >= qp);
            if ((uint32_t)lane == ((c0 >> 5) & 31u)) mysbm = sm;            // lane k keeps the word of chunk k (mod 32)
            if (((c0 >> 5) & 31u) == 31u || c0 + 32u >= len) {              // flush 32 chunk words at a time
                const uint32_t wbase = (c0 >> 5) & ~31u;
                if (wbase + lane <= (c0 >> 5) && wbase + lane < (rg.cap >> 5)) sbm[wbase + lane] = mysbm;
            }
        }
    };

    // ---- K4 (stage C): 5x5 window from the slots of lines p-2..p+2, gated sums, record -> stage[j] ----------------
    // vp = ring index of line p.  Slots of lines outside the plane are empty (R2).
    // sl[a] / gls[a]: slot and first-digit index of line p+a-2 (warp-uniform: a warp's peaks are all on its line)
    // valid lanes hold one queued peak each (jl = its index in the line); clusters that pass the cuts (V2; all of them
    // by default) are written in lane order from ordinal k0 on; returns how many.
    auto moments = [&](bool valid, int p, uint32_t jl, uint32_t k0, const uint32_t* const (&sl)[5],
                       const uint32_t (&gls)[5]) -> uint32_t {
        bool keep = false;
        ClusterSums sums = {0, 0, 0, 0, 0};
        uint32_t fl = 0u, t = 0u, qmax = 0u;
        if (valid) {
            const uint32_t self = fetch(sl[2], gls[2], jl);
            t = self & 0xffffu;
            qmax = self >> 16;
            int c[5][5];
#pragma unroll
            for (int a = 0; a < 5; ++a) window<2>(rg, sl[a], digits, gls[a], n, (int)t, c[a]);
            sums = cluster_sums(c, q_gate);
            keep = var.active ? cluster_variant(sums, (uint32_t)p, t, qmax, (uint32_t)P, (uint32_t)T, var, &fl) : true;
        }
        const unsigned km = __ballot_sync(0xffffffffu, keep);
        if (keep) {
            const ClusterWords r = cluster_finish(sums, w0_base | ((uint32_t)p << 16), t, qmax, fl);
            const size_t j = (size_t)gls[2] + k0 + (uint32_t)__popc(km & ((1u << lane) - 1u));
            stage[2 * j] = r.lo;
            stage[2 * j + 1] = r.hi;
        }
        return (uint32_t)__popc(km);
    };

    // ---- K2: stages A and B for line p (ring index vp), owned by this warp; lo = p - l0 ------------------------------
    auto stage_ab = [&](int p, int vp) {
        const uint32_t gl = s_ls[p], len = s_ls[p + 1] - gl;
        if (len == 0) { if (lane == 0) line_cnt[plane * g.LS + p] = 0u; return; }
        const uint32_t* sl[5];
        uint32_t gls[5];
#pragma unroll
        for (int a = 0; a < 5; ++a) {
            sl[a] = rg.slot(ring_at(vp, a - 2));
            gls[a] = s_ls[min(max(p + a - 2, 0), P)];
        }
        const uint32_t* sp = sl[2];
        const uint32_t* sm1 = sl[1];
        const uint32_t* sp1 = sl[3];
        const uint32_t glm = gls[1], glp = gls[3];
        uint32_t* wq = s_wq[warp];
        uint32_t* pq = s_pq[warp];
        uint32_t pcount = 0, pdone = 0;                         // warp-uniform: queued / already written peaks

        auto stage_b = [&](bool act, uint32_t jl) {
            bool peak = false;
            int t = 0;
            if (act) {
                const uint32_t self = fetch(sp, gl, jl);
                t = (int)(self & 0xffffu);
                const uint32_t q = self >> 16;
                int cm[3], cp[3];
                window<1>(rg, sm1, digits, glm, n, t, cm);      // line p-1: earlier, strict (R1)
                window<1>(rg, sp1, digits, glp, n, t, cp);      // line p+1: later, >=
                peak = q > (uint32_t)cm[0] && q > (uint32_t)cm[1] && q > (uint32_t)cm[2] &&
                       q >= (uint32_t)cp[0] && q >= (uint32_t)cp[1] && q >= (uint32_t)cp[2];
            }
            // peaks -> this warp's peak queue; stage C runs on every full 32 (dense lanes) and once at the end
            const unsigned pm = __ballot_sync(0xffffffffu, peak);
            if (pm == 0) return;
            if (peak) pq[pcount + (uint32_t)__popc(pm & ((1u << lane) - 1u))] = jl;
            pcount += (uint32_t)__popc(pm);
            __syncwarp();
            if (pcount >= 32u) {
                pdone += moments(true, p, pq[lane], pdone, sl, gls);
                const uint32_t mv = (lane + 32u < pcount) ? pq[lane + 32u] : 0u;
                __syncwarp();
                if (lane + 32u < pcount) pq[lane] = mv;
                pcount -= 32u;
                __syncwarp();
            }
        };

        uint32_t wcount = 0;                                    // warp-uniform
        auto enqueue_m = [&](unsigned m, uint32_t jl) {         // m = ballot of survivors; stage B on every full 32
            if (m == 0) return;
            const bool surv = (m >> lane) & 1u;
            if (surv) wq[wcount + (uint32_t)__popc(m & ((1u << lane) - 1u))] = jl;
            wcount += (uint32_t)__popc(m);
            __syncwarp();
            if (wcount >= 32u) {
                stage_b(true, wq[lane]);
                const uint32_t mv = (lane + 32u < wcount) ? wq[lane + 32u] : 0u;
                __syncwarp();
                if (lane + 32u < wcount) wq[lane] = mv;
                wcount -= 32u;
                __syncwarp();
            }
        };
        // stage A was done when the line was built: one bit per digit index below cap
        const uint32_t* sbm = sp + rg.wpl + rg.cap + rg.pre_words;
        const uint32_t nstaged = min(len, rg.cap);
        auto enqueue = [&](bool surv, uint32_t jl) { enqueue_m(__ballot_sync(0xffffffffu, surv), jl); };
        {   // expand all stage-A words at once: lane k owns word k (cap <= 1024 => at most 32 words); prefix sums of
            // the popcounts give every lane its place in the list, then stage B runs over dense groups of 32
            const uint32_t nw = (nstaged + 31u) >> 5;
            uint32_t word = (uint32_t)lane < nw ? sbm[lane] : 0u;
            const uint32_t cw = (uint32_t)__popc(word);
            uint32_t inc = cw;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t u = __shfl_up_sync(0xffffffffu, inc, o);
                if (lane >= o) inc += u;
            }
            const uint32_t total = __shfl_sync(0xffffffffu, inc, 31);
            uint16_t* lst = reinterpret_cast<uint16_t*>(rg.sm + kSlots * rg.slot_words + kWarps * rg.cap) +
                            (size_t)warp * (rg.cap + 32);         // every staged digit may survive
            uint32_t o = inc - cw;
            while (word) {
                const uint32_t b = (uint32_t)__ffs(word) - 1u;
                word &= word - 1u;
                lst[o++] = (uint16_t)(32u * lane + b);
            }
            __syncwarp();
            for (uint32_t i = 0; i < total; i += 32)
                stage_b(i + lane < total, i + lane < total ? (uint32_t)lst[i + lane] : 0u);
        }
        // tail of a line longer than cap: the own-line test from the digit array
        uint32_t carry = nstaged < len ? fetch(sp, gl, nstaged - 1) : 0u;
        for (uint32_t c0 = nstaged; c0 < len; c0 += 32) {
            const uint32_t jl = c0 + lane;
            const bool act = jl < len;
            const uint32_t self = act ? fetch(sp, gl, jl) : 0u;
            uint32_t prev = __shfl_up_sync(0xffffffffu, self, 1);
            uint32_t next = __shfl_down_sync(0xffffffffu, self, 1);
            if (lane == 0) prev = carry;
            if (lane == 31) next = (jl + 1 < len) ? fetch(sp, gl, jl + 1) : 0u;
            carry = __shfl_sync(0xffffffffu, self, 31);
            const int t = (int)(self & 0xffffu);
            const uint32_t q = self >> 16;
            const uint32_t qm = ((int)(prev & 0xffffu) == t - 1) ? (prev >> 16) : 0u;
            const uint32_t qp = ((int)(next & 0xffffu) == t + 1 && t + 1 < T) ? (next >> 16) : 0u;
            enqueue(act && q >= q_peak_min && t < T && q > qm && q >= qp, jl);   // R1: (0,-1) strict, (0,+1) >=
        }
        if (wcount) stage_b((uint32_t)lane < wcount, (uint32_t)lane < wcount ? wq[lane] : 0u);
        if (pcount) pdone += moments((uint32_t)lane < pcount, p, pq[lane], pdone, sl, gls);
        if (lane == 0) line_cnt[plane * g.LS + p] = pdone;   // clusters of this line, in time order
    };

    // ---- main loop -------------------------------------------------------------------------------------------------
    // Ring index of line p is (p - (pa - 2)) mod kSlots.  Prologue: lines pa-2 .. pa+S+1.
    for (int i = warp; i < kS + 4; i += kWarps) prefetch_line(pa - 2 + i, i, i < kWarps);
    for (int i = warp; i < kS + 4; i += kWarps) build_line(pa - 2 + i, i, true, i < kWarps);
    __syncthreads();
    // Step (ONE barrier): every warp prefetches the line it will build, runs stages A+B+C on its current line
    // (lines l0-2 .. l0+S+1 are complete), then rebuilds the slot of a line that left the ring (l0-S-2 .. l0-3).
    int vl0 = 2;                                                // ring index of line l0
    for (int l0 = pa; l0 < pb; l0 += kS) {
        const bool more = l0 + kS < pb;                         // lines l0+S+2 .. l0+2S+1 enter the ring in this step
        const int pnew = l0 + kS + 2 + warp, vnew = ring_at(vl0, kS + 2 + warp - kSlots);
        if (more) prefetch_line(pnew, vnew, true);
        if (l0 + warp < pb) stage_ab(l0 + warp, ring_at(vl0, warp));
        if (more) build_line(pnew, vnew, true, true);
        __syncthreads();
        vl0 = ring_at(vl0, kS);
    }
    if (bad_order) s_unsorted = 1;
    __syncthreads();
    if (tid == 0 && s_unsorted) atomicOr(&cnt->unsorted, 1u);
}

cudaError_t fused_lines_set_attributes()
{
    return cudaFuncSetAttribute(k_fused_lines, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
}

int launch_fused_sorted(const Geo& g, const Workspace& ws, const tpc_digit* digits, uint64_t n, uint64_t shape_n,
                        uint32_t q_peak_min, uint32_t q_gate, const Variant& var, const Tuning& tun, bool have_index,
                        cudaStream_t st, cudaEvent_t ev_k0, cudaEvent_t ev_k1)
{
    const uint32_t entries = g.n_planes * g.LS + 1;
    if (n == 0) {     // nothing to index: only the per-run state of the compaction (the caller zeroed the counters)
        cudaMemsetAsync(ws.line_cnt, 0, (size_t)entries * 4, st);
        cudaMemsetAsync(ws.line_desc, 0, ((size_t)(entries + 63) / 64 + 1) * 8, st);
        return 0;
    }
    int k = 0;
    if (!have_index) {
        const bool direct = n < (1u << 20);             // small input: one index launch instead of two
        if (!direct) {
            k_plane_index<<<(g.n_planes + 1 + 255) / 256, 256, 0, st>>>((const uint2*)digits, (uint32_t)n, g, ws.line_start,
                                                                         ws.counters);
            ++k;
        }
        k_line_index<<<(entries + 255) / 256, 256, 0, st>>>((const uint2*)digits, (uint32_t)n, g, ws.line_start,
                                                            ws.line_cnt, ws.line_desc, direct ? ws.counters : nullptr);
        ++k;
    }

    // Kernel choice.  Block-sparse line slots when the mean line fits their pool (k_fused_pairs, tpc_cf_pairs.cu; its
    // first generation k_fused_blocks, tpc_cf_blocks.cu, only on request), else the bitmap slots below.
    // tun.fused_kernel (tests, profiling): 1 pairs, 2 blocks, 3 lines.
    if (tun.fused_kernel != 3) {
        const int r = tun.fused_kernel == 2
            ? launch_fused_blocks(g, ws, digits, n, shape_n, q_peak_min, q_gate, var, tun, false, st, ev_k0, ev_k1)
            : launch_fused_pairs(g, ws, digits, n, shape_n, q_peak_min, q_gate, var, tun, tun.fused_kernel == 1, st, ev_k0, ev_k1);
        if (r < 0) return r;
        if (r > 0) return k + r;
    }

    // launch shape: pad range per unit, tq capacity per slot from the mean line length (host-known)
    uint64_t total_pads = 0;
    for (uint32_t r = 0; r < g.n_rows; ++r) total_pads += g.npads[r];
    total_pads *= g.n_sectors;
    const double mean_len = (double)(shape_n ? shape_n : n) / (double)(total_pads ? total_pads : 1);
    const uint32_t wpl = (((g.n_time + 31) / 32 + 3) + 3u) & ~3u;   // guard word below, >= 2 above; multiple of 4
    const uint32_t pre_words = ((wpl >> 1) + 3u) & ~3u;
    uint32_t cap = ((uint32_t)(mean_len * 1.5) + 64u + 127u) & ~127u;
    const uint32_t max_smem = 106 * 1024;                    // 2 CTAs per SM (+ ~5 KB static + 1 KB reserved each)
    const uint32_t fixed = kSlots * (wpl + pre_words) * 4 + kWarps * 64;
    const uint32_t per_cap0 = kSlots * 4 + kSlots / 8 + 1 + kWarps * 4 + kWarps * 2;   // tq, stage-A bit, key staging, survivor list
    if (fixed + per_cap0 * 128 > 200 * 1024) {
        // the bitmap slots of 20 lines do not fit (n_time above ~50 k): the block kernel covers the time axis in passes
        int r = launch_fused_pairs(g, ws, digits, n, shape_n, q_peak_min, q_gate, var, tun, true, st, ev_k0, ev_k1);
        if (r == 0)     // (k_fused_pairs declines n_time above its sentinel times; its first generation takes any geometry)
            r = launch_fused_blocks(g, ws, digits, n, shape_n, q_peak_min, q_gate, var, tun, true, st, ev_k0, ev_k1);
        if (r < 0) return r;
        return r > 0 ? k + r : TPC_CF_E_GEOMETRY;
    }
    const uint32_t limit = fixed + per_cap0 * 128 <= max_smem ? max_smem : 200 * 1024;
    const uint32_t per_cap = per_cap0;
    if (cap > 1024u) cap = 1024u;                            // the stage-A words of a line must fit one warp (32 words)
    if (fixed + per_cap * cap > limit) cap = ((limit - fixed) / per_cap) & ~127u;
    const uint32_t smem = fixed + kSlots * (cap * 4 + (cap >> 5) * 4) + kWarps * cap * 4 + kWarps * (cap + 32) * 2;
    // One CTA per whole plane when there are enough planes to fill the GPU (no halo lines, one prologue per plane:
    // measured 2.94 ms vs 3.16 ms at 48 pads on config 3); smaller pad ranges for small problems.
    const uint32_t whole = (g.max_pads + kS - 1) / kS * kS;
    uint32_t pads_per_unit = g.n_planes >= 1184 ? whole : (g.n_planes >= 296 ? 6 * kS : 3 * kS);
    if (pads_per_unit > whole) pads_per_unit = whole;
    if (tun.pads_per_unit >= kS && tun.pads_per_unit <= 256) pads_per_unit = (uint32_t)(tun.pads_per_unit / kS * kS);
    const uint32_t upp = (g.max_pads + pads_per_unit - 1) / pads_per_unit;
    if (ev_k0) cudaEventRecord(ev_k0, st);
    g_last_kernel = "k_fused_lines";
    k_fused_lines<<<g.n_planes * upp, kFThreads, smem, st>>>((const uint2*)digits, (uint32_t)n, g, ws.line_start,
                                                             pads_per_unit, upp, wpl, cap, q_peak_min, q_gate, var,
                                                             ws.counters, ws.line_cnt, (uint4*)ws.stage);
    if (ev_k1) cudaEventRecord(ev_k1, st);
    return k + 1;
}

}  // namespace tpccf
