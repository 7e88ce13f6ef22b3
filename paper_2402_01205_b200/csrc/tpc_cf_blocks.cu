// tpc_cf_blocks.cu — fused path, block-sparse line slots ("T3b"): same streaming scheme as tpc_cf_fused.cu (one CTA per
// (plane, pad range), one WARP per pad LINE, a ring of line slots in shared memory, one barrier per step of 8 lines),
// but a line slot holds the line of the charge map as 8-cell blocks instead of a bitmap + rank directory:
//     hdr      [16 B]   word 0: number of stage-A survivors of the line
//     dir[b]   uint8    pool index of the block of time bins 8b-8 .. 8b-1 (0 = the all-zero block, 0xFF = the line has
//                       this block but the pool was full: the cell is then looked up in the digit array)
//     pool[i]  16 B     eight uint16 charges; block 0 stays zero (zero border in time and empty cells, R2)
//     surv[k]  uint32   (time | charge << 16) of the k-th digit that passed the own-line test (stage A), time order
// A cell lookup is dir byte -> 16-bit load, without bit counting or divergence; a 3- or 5-cell window costs two dir
// bytes and 3 / 5 charge loads.  Digits stream through a per-warp staging ring of four 32-digit chunks (cp.async),
// so a line of any length is handled by the same code.
//   K0  the warp that reuses a slot zeroes its dir + pool          K1  build: block allocation by ballot/popc
//   K2  stage A at build time (shuffles), stage B from the survivor list against lines p-1 / p+1
//   K4  stage C: peaks queued per warp, 5x5 window from the five slots p-2..p+2 -> stage[line_start + k]
// Selected by launch_fused_sorted when the mean line fits the block pool (<= 254 blocks); otherwise the bitmap
// kernel of tpc_cf_fused.cu runs.  Definition: include/tpc_cf.h (BASELINE.json:north_star; step named in PAPER.md:57).
#include "tpc_cf_internal.cuh"

namespace tpccf {

static constexpr int kBThreads = 256;
static constexpr int kBWarps = kBThreads / 32;
static constexpr int kBS = kBWarps;              // lines per step: one per warp
static constexpr int kBSlots = 2 * kBS + 4;      // lines l0-2 .. l0+S+1 in use, next S being built
static constexpr int kStageDepth = 4;            // staging ring: chunks of 32 digits (256 B each) per warp
static constexpr uint32_t kDirOff = 16;          // dir starts after the header
#ifndef TPC_CF_BALANCE
#define TPC_CF_BALANCE 1
#endif
static constexpr bool kBalance = TPC_CF_BALANCE != 0;   // in-step load balancing by line length

// ---- shared-window accessors (32-bit addresses: no generic-address arithmetic in the hot loops) ------------------
__device__ __forceinline__ uint32_t lds32(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint2 lds64(uint32_t a)
{
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ uint32_t lds16(uint32_t a)
{
    uint16_t v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint32_t lds8(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts32(uint32_t a, uint32_t v)
{
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ void sts16(uint32_t a, uint32_t v)
{
    asm volatile("st.shared.u16 [%0], %1;" ::"r"(a), "h"((uint16_t)v) : "memory");
}
__device__ __forceinline__ void sts8(uint32_t a, uint32_t v)
{
    asm volatile("st.shared.u8 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ void sts128z(uint32_t a)
{
    asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(a), "r"(0u) : "memory");
}

// ring index of the line at distance d (|d| < kBSlots) from the line whose ring index is v0
__device__ __forceinline__ int bring_at(int v0, int d)
{
    int v = v0 + d;
    v += (v < 0) ? kBSlots : 0;
    v -= (v >= kBSlots) ? kBSlots : 0;
    return v;
}

// K2 stage A (R1, own line): the neighbours in time are the adjacent digits of the line; an absent one reads 0.
// (0,-1) is lexicographically earlier: strict; (0,+1) later: >=.
__device__ __forceinline__ bool stage_a(uint32_t y, uint32_t prevy, bool has_prev, uint32_t nexty, bool has_next,
                                        uint32_t T, uint32_t q_peak_min)
{
    const uint32_t t = y & 0xffffu, q = y >> 16;
    const uint32_t qm = (has_prev && (prevy & 0xffffu) + 1u == t) ? (prevy >> 16) : 0u;
    const uint32_t qp = (has_next && (nexty & 0xffffu) == t + 1u && t + 1u < T) ? (nexty >> 16) : 0u;
    return q >= q_peak_min && q > qm && q >= qp;
}

// charge of cell (line, tt) from the digit array (slow path: the line's block pool was full).  Binary search on time.
// Cells outside [0, T) read 0 (R2) whatever the digit array holds there (a digit with time >= T is invalid, R11).
__device__ __noinline__ uint32_t cell_from_digits(const uint2* __restrict__ digits, uint32_t gl, uint32_t glen,
                                                  uint32_t tt, uint32_t T)
{
    if (tt >= T) return 0u;
    uint32_t lo = 0, hi = glen;
    while (lo < hi) {
        const uint32_t mid = lo + ((hi - lo) >> 1);
        if ((__ldg(&digits[gl + mid].y) & 0xffffu) < tt) lo = mid + 1; else hi = mid;
    }
    if (lo >= glen) return 0u;
    const uint32_t y = __ldg(&digits[gl + lo].y);
    return (y & 0xffffu) == tt ? (y >> 16) : 0u;
}

// Slow path of bwindow (rare: a block of the window is not in the pool): cells of missing blocks come from the digit
// array.  Out of line, result in registers, to keep the hot code small.
struct Win5 { int c[5]; };
__device__ __noinline__ Win5 bwindow_slow(uint32_t aA, uint32_t aB, uint32_t dA, uint32_t dB, uint32_t o, int t0, int n,
                                          const uint2* __restrict__ digits, uint32_t gl, uint32_t glen, uint32_t T)
{
    Win5 r;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const bool inA = o + (uint32_t)k < 8u;
        const uint32_t d = inA ? dA : dB;
        r.c[k] = k >= n ? 0
               : (d != 0xFFu ? (int)lds16((inA ? aA : aB) + 2u * (uint32_t)k)
                             : (int)cell_from_digits(digits, gl, glen, (uint32_t)(t0 + k), T));
    }
    return r;
}

// charges of the window t-H..t+H of the line in slot `slot` (0 where no digit): c[k] is time t-H+k.
// dsub = first time bin of the pass / 8.  lidx = pad index of that line, used only by the slow path (line_start
// lookups in s_ls).
template <int H>
__device__ __forceinline__ void bwindow(uint32_t slot, uint32_t dsub, const SlotGeo& sg, int t, int (&c)[2 * H + 1],
                                        const uint2* __restrict__ digits, const uint32_t* s_ls, int lidx, int P,
                                        uint32_t T)
{
    const uint32_t u = (uint32_t)(t + 8 - H);                 // first cell, shifted by the 8-bin guard block
    const uint32_t dir = slot + kDirOff - dsub;
    const uint32_t dA = lds8(dir + (u >> 3));
    const uint32_t dB = lds8(dir + ((u + 2 * H) >> 3));
    const uint32_t o = u & 7u;
    const uint32_t base = slot + sg.pool_off + 2u * o;
    const uint32_t aA = base + (dA << 4), aB = base + (dB << 4) - 16u;
    if (dA != 0xFFu && dB != 0xFFu) {
#pragma unroll
        for (int k = 0; k < 2 * H + 1; ++k) c[k] = (int)lds16((o + (uint32_t)k < 8u ? aA : aB) + 2u * (uint32_t)k);
    } else {
        const bool inside = lidx >= 0 && lidx < P;
        const uint32_t gl = inside ? s_ls[lidx] : 0u;
        const uint32_t glen = inside ? s_ls[lidx + 1] - gl : 0u;
        const Win5 r = bwindow_slow(aA, aB, dA, dB, o, t - H, 2 * H + 1, digits, gl, glen, T);
#pragma unroll
        for (int k = 0; k < 2 * H + 1; ++k) c[k] = r.c[k];
    }
}

// MULTI: the time axis is covered in sg.n_pass > 1 passes (long lines).  VAR: flags / cuts requested (V1..V3); the
// default instantiation carries none of that code.
// MINB: CTAs per SM the registers are limited for (3 when the slots are small enough for a third CTA).
template <bool MULTI, bool VAR, int MINB>
__global__ void __launch_bounds__(kBThreads, MINB)
k_fused_blocks(const uint2* __restrict__ digits, uint32_t n, Geo g, const uint32_t* __restrict__ line_start,
               uint32_t pads_per_unit, uint32_t units_per_plane, SlotGeo sg, uint32_t q_peak_min, uint32_t q_gate,
               Variant var, Counters* cnt, uint32_t* __restrict__ line_cnt, uint4* __restrict__ stage)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t s_ls[260];          // line starts of this plane: s_ls[p], p = 0..max_pads, then next plane's start
    __shared__ uint32_t s_pos[260];         // first digit of line p that the current pass needs (time >= pass start - 2)
    __shared__ uint32_t s_cnt[260];         // peaks of line p found by the passes so far
    __shared__ int s_unsorted;

    const uint32_t plane = blockIdx.x / units_per_plane, unit = blockIdx.x % units_per_plane;
    const uint32_t sector = plane / g.n_rows, row = plane % g.n_rows;
    const int P = (int)g.npads[row];
    const int pa = (int)(unit * pads_per_unit);
    const int pb = min(pa + (int)pads_per_unit, P);
    const uint32_t T = g.n_time;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t w0_base = sector | (row << 8);
    const uint32_t lt_mask = (1u << lane) - 1u;

    const uint32_t sm0 = (uint32_t)__cvta_generic_to_shared(smem_raw);
    const uint32_t stg = sm0 + kBSlots * sg.slot_bytes + (uint32_t)warp * (kStageDepth * 256u);   // staging ring
    const uint32_t pqa = sm0 + kBSlots * sg.slot_bytes + kBWarps * (kStageDepth * 256u) + (uint32_t)warp * 256u;

    for (int i = tid; i <= (int)g.LS; i += kBThreads) {
        const uint32_t v = line_start[plane * g.LS + i];
        s_ls[i] = v; s_pos[i] = v; s_cnt[i] = 0u;
    }
    if (tid == 0) s_unsorted = 0;
    // every slot starts as an empty line (lines outside the plane keep this state: zero border in pad, R2)
    for (uint32_t x = (uint32_t)tid * 16u; x < kBSlots * sg.slot_bytes; x += kBThreads * 16u) sts128z(sm0 + x);
    __syncthreads();

    if (pa >= P && unit != 0) return;    // nothing in this pad range (rows with fewer pads)

    uint32_t bad_order = 0u;
    // monotone line starts: a garbage index from unsorted input must not produce negative lengths or unbounded work
    for (int i = tid; i < (int)g.LS; i += kBThreads) if (s_ls[i] > s_ls[i + 1]) bad_order = 1u;
    if (__syncthreads_or((int)bad_order)) {
        if (tid == 0) atomicOr(&cnt->unsorted, 1u);
        return;
    }

    // gap of the plane: digits with pad >= npads[row] (or a row/sector beyond the geometry) — all invalid (R11)
    if (unit == 0) {
        const uint32_t gb = s_ls[P], ge = s_ls[g.LS];
        if (ge > gb) {
            for (uint32_t j = gb + tid; j < ge; j += kBThreads) {
                const uint2 d = __ldg(digits + j);
                if (digit_valid(g, d.x, d.y)) bad_order = 1u;     // a valid digit outside every line: not sorted
            }
            if (tid == 0) atomicAdd(&cnt->n_bad, (unsigned long long)(ge - gb));
        }
    }

    const int blo = max(pa - 2, 0), bhi = min(P, pb + 2);   // lines this unit ever builds

    // Time window of the current pass (set in the pass loop below).  Owned cells [tlo, thi): their peaks are found
    // in this pass.  Stored cells [wlo, whi) = owned +- 2 bins: the 5x5 windows of owned peaks stay inside.
    // With a single pass (MULTI = false) these are constants and the pass logic folds away.
    uint32_t tlo = 0u, thi = T, wlo = 0u, whi = T, dsub = 0u;
    bool last_pass = true;

    // ---- staging: chunk c (digits 32c .. 32c+31) of a line -> ring entry c mod kStageDepth (cp.async, 8 B per lane) --
    // one commit group per chunk, empty or not, so that wait_group counts chunks.  Prefetch distance: kAhead chunks.
    constexpr uint32_t kAhead = kStageDepth - 1;
    const uint32_t stg_lane = stg + 8u * (uint32_t)lane;
    auto cp_async8 = [&](uint32_t dst, const uint2* src) {
        asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
    };
    // the first kAhead chunks of the line this warp builds next (issued before the warp processes its current line,
    // so the global latency is covered)
    auto stage_head = [&](int p) {
        if (p < blo || p >= bhi) return;
        const uint32_t lbeg = s_pos[p], len = s_ls[p + 1] - lbeg;
#pragma unroll
        for (uint32_t c = 0; c < kAhead; ++c) {
            if (32u * c + (uint32_t)lane < len) cp_async8(stg_lane + 256u * c, digits + lbeg + 32u * c + lane);
            asm volatile("cp.async.commit_group;" ::: "memory");
        }
    };

    // ---- K0 + K1 + stage A: this warp (re)builds slot v as line p ---------------------------------------------------
    auto build_line = [&](int p, int v) {
        const uint32_t slot = sm0 + (uint32_t)v * sg.slot_bytes;
        for (uint32_t x = (uint32_t)lane * 16u; x < sg.surv_off; x += 512u) sts128z(slot + x);   // hdr, dir, pool
        __syncwarp();
        if (p < blo || p >= bhi) return;                    // a line outside the plane / the halo: stays empty
        const uint32_t lbeg = s_pos[p], lend = s_ls[p + 1], len = lend - lbeg;
        if (lane == 0) sts32(slot + 4u, lbeg);              // hdr word 1: where this pass started in the line
        if (len == 0) return;
        const uint32_t w0_line = w0_base | ((uint32_t)p << 16);
        const uint32_t a_dir1 = slot + kDirOff + 1u - (MULTI ? dsub : 0u); // dir byte of the block of time t: a_dir1 + (t >> 3)
        const uint32_t a_pool = slot + sg.pool_off, a_surv = slot + sg.surv_off;
        const uint32_t qmin_y = q_peak_min << 16;           // y >= qmin_y  <=>  charge >= q_peak_min
        const uint32_t le_mask = lt_mask | (1u << lane);
        const uint32_t own_span = thi - tlo, win_span = whi - wlo;
        const uint32_t nlo = thi - 2u;                      // the next pass needs the line from this time on
        const uint2* gp = digits + lbeg + 32u * kAhead + lane;   // this lane's digit of chunk c + kAhead
        uint32_t ro = 0u;                                   // ring offset of chunk c
        const uint32_t off_own = (8u * (uint32_t)lane + kStageDepth * 256u - 8u) & (kStageDepth * 256u - 1u);
        const uint32_t off_prev = (8u * (uint32_t)lane + kStageDepth * 256u - 16u) & (kStageDepth * 256u - 1u);
        uint32_t nblk = 0u, nsurv = 0u;                     // warp-uniform running counts
        uint32_t nbad = 0u;                                 // per lane
        uint32_t next_pos = lend;                           // first digit with time >= nlo (warp-uniform)
        bool found = false;
        // Iteration c works on the digits 32c-1 .. 32c+30 (lane i: digit 32c+i-1): with this one-digit shift the
        // successor of the last digit of the iteration is still in chunk c, so only chunk c has to have landed and
        // the copies of chunks c+1, c+2 stay in flight (one more chunk of slack than with a look-ahead into chunk c+1).
        for (uint32_t c0 = 0; c0 <= len; c0 += 32u) {
            const uint32_t jl = c0 + (uint32_t)lane - 1u;   // 0xffffffff for the digit before the line: inactive
            // chunks 0 .. c+2 are committed at this point; all but the two newest have landed: chunks <= c
            asm volatile("cp.async.wait_group %0;" ::"n"(kAhead - 1) : "memory");
            __syncwarp();
            // this digit and its neighbours in the line, straight from the staging ring (one contiguous 1 KB window per
            // warp, so "previous / next digit" is -8 / +8 bytes modulo 1 KB): three independent loads.  Chunk c-1 is
            // still there: its entry is recycled by the cp.async below, after these loads.
            const uint2 d = lds64(stg + ((off_own + ro) & (kStageDepth * 256u - 1u)));
            const uint32_t prevy = lds32(stg + ((off_prev + ro) & (kStageDepth * 256u - 1u)) + 4u);
            const uint32_t nexty = lds32(stg_lane + ro + 4u);
            const uint32_t y = d.y;
            if (32u * kAhead + c0 + (uint32_t)lane < len)
                cp_async8(stg_lane + ((ro + 256u * kAhead) & (256u * (kStageDepth - 1))), gp);
            gp += 32;
            asm volatile("cp.async.commit_group;" ::: "memory");
            ro = (ro + 256u) & (256u * (kStageDepth - 1));
            const bool act = jl < len, nf = jl != 0u;
            const uint32_t t = y & 0xffffu;
            const uint32_t xkey = (d.x ^ w0_line) & 0x00ffffffu;
            const bool ok = act && xkey == 0u;
            // wrong line, not ascending, or duplicate cell: the DIGITS_SORTED promise is false
            bad_order |= (act && (xkey != 0u || (nf && (prevy & 0xffffu) >= t))) ? 1u : 0u;
            const bool inb = MULTI ? (ok && (t - wlo) < win_span) : (ok && t < T);    // a cell this pass stores
            const bool own = MULTI ? (ok && (t - tlo) < own_span) : inb;   // a cell this pass decides (ends at T at the latest)
            // R11: time out of range or zero charge, counted by the pass that owns the digit's time
            if ((!MULTI ? ok : (last_pass ? (ok && t >= tlo) : own)) && !(own && y >= 0x10000u)) ++nbad;
            // K1: blocks are allocated in time order: a digit opens a block iff the digit before it is in another one
            const bool head = inb && (!nf || ((y ^ prevy) & 0xfff8u) != 0u);
            const unsigned hm = __ballot_sync(0xffffffffu, head);
            const uint32_t idx = nblk + (uint32_t)__popc(hm & le_mask);   // 1-based; 0 = zero block
            nblk += (uint32_t)__popc(hm);
            const bool in_pool = idx < sg.pcap;
            if (head) sts8(a_dir1 + (t >> 3), in_pool ? idx : 0xFFu);
            if (inb && in_pool) sts16(a_pool + (idx << 4) + ((y & 7u) << 1), y >> 16);
            // K2 stage A (R1, own line) on the packed words: with equal time fields, comparing the words compares
            // the charges.  (0,-1) is earlier: the digit loses to an adjacent previous charge >= its own;
            // (0,+1) is later: it loses to an adjacent next charge > its own (cells at time >= T read 0).
            const uint32_t A = prevy + 1u, B = nexty - 1u;
            const bool kill_prev = nf && ((A ^ y) & 0xffffu) == 0u && A >= y;
            const bool kill_next = jl + 1u < len && ((B ^ y) & 0xffffu) == 0u && B > y && (nexty & 0xffffu) < T;
            const bool surv = own && y >= qmin_y && !kill_prev && !kill_next;
            const unsigned smk = __ballot_sync(0xffffffffu, surv);
            const uint32_t pos = nsurv + (uint32_t)__popc(smk & lt_mask);
            if (surv && pos < sg.scap) sts32(a_surv + (pos << 2), y);
            nsurv += (uint32_t)__popc(smk);
            if (MULTI && !last_pass) {
                // where the next pass starts in this line, and whether this pass has seen all it stores
                const bool tail = c0 + 31u >= len;           // this iteration reaches the last digit of the line
                const uint32_t t31 = __shfl_sync(0xffffffffu, y, 31) & 0xffffu;   // time of the iteration's last digit (if not tail)
                if (!found && (tail || t31 >= nlo)) {
                    const unsigned m = __ballot_sync(0xffffffffu, act && t >= nlo);
                    if (m) { next_pos = lbeg + c0 + (uint32_t)__ffs(m) - 2u; found = true; }   // digit of lane i: c0+i-1
                }
                if (!tail && t31 >= whi) {                  // every later digit is beyond the window
                    asm volatile("cp.async.wait_group 0;" ::: "memory");   // the ring is reused by the next line
                    break;
                }
            }
        }
        if (lane == 0) {
            sts32(slot, nsurv);
            if (MULTI && !last_pass) s_pos[p] = next_pos;
        }
        if (p >= pa && p < pb) {                            // halo lines are counted by the unit that owns them
            const uint32_t tot = __reduce_add_sync(0xffffffffu, nbad);
            if (tot != 0u && lane == 0) atomicAdd(&cnt->n_bad, (unsigned long long)tot);
        }
    };

    // ---- K2 stage B + K4 stage C for line p (ring index vp), owned by this warp -------------------------------------
    auto process_line = [&](int p, int vp) {
        const uint32_t gl = s_ls[p], lend = s_ls[p + 1];
        if (lend == gl) return;                             // line_cnt stays 0 (cleared per run)
        uint32_t sl[5];                                     // slots of lines p-2 .. p+2 (empty outside the plane, R2)
        {
            const uint32_t ring_end = sm0 + kBSlots * sg.slot_bytes;
            uint32_t a0 = sm0 + (uint32_t)bring_at(vp, -2) * sg.slot_bytes;
#pragma unroll
            for (int a = 0; a < 5; ++a) {
                sl[a] = a0;
                a0 += sg.slot_bytes;
                if (a0 == ring_end) a0 = sm0;
            }
        }
        const uint32_t w0_line = w0_base | ((uint32_t)p << 16);
        uint32_t pcount = 0, pdone = MULTI ? s_cnt[p] : 0u; // warp-uniform: queued / already written peaks of the line

        // stage C for up to 32 queued peaks (one per lane): y = (time | qmax << 16).  Clusters that pass the cuts (V2;
        // all of them by default) are written in lane order from ordinal `pdone` on; returns how many.
        auto moments = [&](bool valid, uint32_t y) -> uint32_t {
            bool keep = false;
            ClusterSums sums = {0, 0, 0, 0, 0};
            uint32_t fl = 0u;
            const uint32_t t = y & 0xffffu;
            if (valid) {
                int c[5][5];
#pragma unroll
                for (int a = 0; a < 5; ++a) bwindow<2>(sl[a], MULTI ? dsub : 0u, sg, (int)t, c[a], digits, s_ls, p + a - 2, P, T);
                sums = cluster_sums(c, q_gate);
                keep = VAR ? cluster_variant(sums, (uint32_t)p, t, y >> 16, (uint32_t)P, T, var, &fl) : true;
            }
            const unsigned km = __ballot_sync(0xffffffffu, keep);
            if (keep) {
                const ClusterWords r = cluster_finish(sums, w0_line, t, y >> 16, fl);
                const size_t j = (size_t)gl + pdone + (uint32_t)__popc(km & lt_mask);   // line's range, time order
                stage[2 * j] = r.lo;
                stage[2 * j + 1] = r.hi;
            }
            return (uint32_t)__popc(km);
        };
        // stage B for up to 32 survivors (one per lane); peaks go to the warp's queue, stage C runs on full warps
        auto stage_b = [&](bool act, uint32_t y) {
            bool peak = false;
            if (act) {
                const int t = (int)(y & 0xffffu);
                const uint32_t q = y >> 16;
                int cm[3], cp[3];
                bwindow<1>(sl[1], MULTI ? dsub : 0u, sg, t, cm, digits, s_ls, p - 1, P, T);   // line p-1: earlier, strict (R1)
                bwindow<1>(sl[3], MULTI ? dsub : 0u, sg, t, cp, digits, s_ls, p + 1, P, T);   // line p+1: later, >=
                peak = q > (uint32_t)cm[0] && q > (uint32_t)cm[1] && q > (uint32_t)cm[2] &&
                       q >= (uint32_t)cp[0] && q >= (uint32_t)cp[1] && q >= (uint32_t)cp[2];
            }
            const unsigned pm = __ballot_sync(0xffffffffu, peak);
            if (pm == 0u) return;
            if (peak) sts32(pqa + ((pcount + (uint32_t)__popc(pm & lt_mask)) << 2), y);
            pcount += (uint32_t)__popc(pm);
            __syncwarp();
            if (pcount >= 32u) {
                pdone += moments(true, lds32(pqa + ((uint32_t)lane << 2)));
                const uint32_t mv = lds32(pqa + (((uint32_t)lane + 32u) << 2));
                __syncwarp();
                sts32(pqa + ((uint32_t)lane << 2), mv);
                pcount -= 32u;
                __syncwarp();
            }
        };

        const uint32_t ns = lds32(sl[2]);
        const uint32_t nst = min(ns, sg.scap);
        for (uint32_t i = 0; i < nst; i += 32u) {
            const bool act = i + (uint32_t)lane < nst;
            stage_b(act, act ? lds32(sl[2] + sg.surv_off + ((i + (uint32_t)lane) << 2)) : 0u);
        }
        if (ns > sg.scap) {
            // rare: more survivors than the slot's list holds.  Stage A again from the digit array, from where this
            // pass started in the line; survivors whose ordinal is >= scap were not listed and are tested here
            // (still in time order).
            const uint32_t lbeg = lds32(sl[2] + 4u), len = lend - lbeg;
            uint32_t seen = 0;
            for (uint32_t c0 = 0; c0 < len; c0 += 32u) {
                const uint32_t jl = c0 + (uint32_t)lane;
                const bool act = jl < len;
                const uint32_t y = act ? __ldg(&digits[lbeg + jl].y) : 0u;
                const uint32_t prevy = jl > 0u && act ? __ldg(&digits[lbeg + jl - 1u].y) : 0u;
                const uint32_t nexty = jl + 1u < len ? __ldg(&digits[lbeg + jl + 1u].y) : 0u;
                const bool surv = act && (MULTI ? ((y & 0xffffu) - tlo) < (thi - tlo) : (y & 0xffffu) < T) &&
                                  stage_a(y, prevy, jl > 0u, nexty, jl + 1u < len, T, q_peak_min);
                const unsigned smk = __ballot_sync(0xffffffffu, surv);
                const uint32_t ord = seen + (uint32_t)__popc(smk & lt_mask);
                seen += (uint32_t)__popc(smk);
                if (seen > sg.scap) stage_b(surv && ord >= sg.scap, y);
                if (seen >= ns) break;                      // all survivors of this pass have been seen
            }
        }
        if (pcount > 16u) {
            pdone += moments((uint32_t)lane < pcount, lds32(pqa + (((uint32_t)lane & 31u) << 2)));
        } else if (pcount > 0u) {
            // the usual case (a line has ~14 peaks): two lanes per peak, each gathers the rows on one side of the
            // peak plus the peak's row (3 windows instead of 5); the halves of the integer sums are added by shuffle
            const uint32_t i = (uint32_t)lane & 15u;
            const bool neg = lane >= 16;                        // this lane takes dp < 0 (lines p-2, p-1)
            const bool valid = i < pcount;
            ClusterSums h = {0, 0, 0, 0, 0};
            uint32_t y = 0u;
            if (valid) {
                y = lds32(pqa + (i << 2));
                const int t = (int)(y & 0xffffu);
                int o[5], m[5], z[5];
                bwindow<2>(neg ? sl[0] : sl[4], MULTI ? dsub : 0u, sg, t, o, digits, s_ls, neg ? p - 2 : p + 2, P, T);
                bwindow<2>(neg ? sl[1] : sl[3], MULTI ? dsub : 0u, sg, t, m, digits, s_ls, neg ? p - 1 : p + 1, P, T);
                bwindow<2>(sl[2], MULTI ? dsub : 0u, sg, t, z, digits, s_ls, p, P, T);
                h = cluster_half_sums(o, m, z, neg ? -1 : 1, !neg, q_gate);
            }
            h.S0 += __shfl_xor_sync(0xffffffffu, h.S0, 16);
            h.S1p += __shfl_xor_sync(0xffffffffu, h.S1p, 16);
            h.S1t += __shfl_xor_sync(0xffffffffu, h.S1t, 16);
            h.S2p += __shfl_xor_sync(0xffffffffu, h.S2p, 16);
            h.S2t += __shfl_xor_sync(0xffffffffu, h.S2t, 16);
            bool keep = valid && !neg;
            uint32_t fl = 0u;
            if (VAR && keep)
                keep = cluster_variant(h, (uint32_t)p, y & 0xffffu, y >> 16, (uint32_t)P, T, var, &fl);
            const unsigned km = __ballot_sync(0xffffffffu, keep);
            if (keep) {
                const ClusterWords r = cluster_finish(h, w0_line, y & 0xffffu, y >> 16, fl);
                const size_t j = (size_t)gl + pdone + (uint32_t)__popc(km & lt_mask);
                stage[2 * j] = r.lo;
                stage[2 * j + 1] = r.hi;
            }
            pdone += (uint32_t)__popc(km);
        }
        if (lane == 0) {
            if (MULTI) s_cnt[p] = pdone;                    // clusters of this line so far, in time order
            if (!MULTI || last_pass) line_cnt[plane * g.LS + p] = pdone;
        }
    };

    // ---- main loop -------------------------------------------------------------------------------------------------
    // The time axis is covered in sg.n_pass passes over the unit's lines (smaller slots -> more CTAs per SM).
    for (uint32_t pass = 0; pass < (MULTI ? sg.n_pass : 1u); ++pass) {
    if (MULTI) {
        last_pass = pass + 1u == sg.n_pass;
        tlo = pass * sg.seg_len;
        thi = last_pass ? T : min(tlo + sg.seg_len, T);
        wlo = tlo >= 2u ? tlo - 2u : 0u;
        whi = min(thi + 2u, T);
        dsub = tlo >> 3;
    }
    // Ring index of line p is (p - (pa - 2)) mod kBSlots.  Prologue: lines pa-2 .. pa+S+1.
    for (int i = warp; i < kBS + 4; i += kBWarps) {
        stage_head(pa - 2 + i);
        build_line(pa - 2 + i, i);
    }
    __syncthreads();
    // Step (ONE barrier): every warp stages the head of the line it will build, runs stages B+C on its current line
    // (lines l0-2 .. l0+S+1 are complete), then rebuilds the slot of a line that left the ring (l0-S-2 .. l0-3).
    int vl0 = 2;                                                // ring index of line l0
    for (int l0 = pa; l0 < pb; l0 += kBS) {
        const bool more = l0 + kBS < pb;                        // lines l0+S+2 .. l0+2S+1 enter the ring in this step
        // Load balance inside the step: a warp's work is one line to process plus one line to build, both
        // proportional to the line lengths (known from the index).  The warp with the longest line to process gets
        // the shortest line to build, and so on: the 8 sums come out nearly equal and the barrier waits less.
        int ip = warp, ib = warp;                               // which of the 8 lines this warp processes / builds
        if (kBalance) {
            uint32_t lp = 0u, lb = 0u;
            if (lane < kBS) {
                const int p = l0 + lane, q = l0 + kBS + 2 + lane;
                if (p < pb) lp = min(s_ls[p + 1] - s_ls[p], 0xfffeu) + 1u;
                if (more && q >= blo && q < bhi) lb = min(s_ls[q + 1] - s_ls[q], 0xfffeu) + 1u;
            }
            const uint32_t mine = lp | (lb << 16);
            // ranks of the 8 lines by all-pairs comparison, two pairs per lane: lane L compares line i = L & 7 with
            // lines j = L >> 3 and j + 4; the four partial counts of a line are added across lanes i, i+8, i+16, i+24.
            // rp: rank of line i among the lines to process, longest first; rb: among the lines to build, shortest first.
            const int i = lane & 7, j0 = lane >> 3;
            const uint32_t vi = __shfl_sync(0xffffffffu, mine, i);
            const uint32_t va = __shfl_sync(0xffffffffu, mine, j0), vb = __shfl_sync(0xffffffffu, mine, j0 + 4);
            const uint32_t pi = vi & 0xffffu, bi = vi >> 16;
            uint32_t cnt = 0u;                                  // process count | build count << 8
            cnt += ((va & 0xffffu) > pi || ((va & 0xffffu) == pi && j0 < i)) ? 1u : 0u;
            cnt += ((vb & 0xffffu) > pi || ((vb & 0xffffu) == pi && j0 + 4 < i)) ? 1u : 0u;
            cnt += ((va >> 16) < bi || ((va >> 16) == bi && j0 < i)) ? 256u : 0u;
            cnt += ((vb >> 16) < bi || ((vb >> 16) == bi && j0 + 4 < i)) ? 256u : 0u;
            cnt += __shfl_xor_sync(0xffffffffu, cnt, 8);
            cnt += __shfl_xor_sync(0xffffffffu, cnt, 16);
            const uint32_t rp = cnt & 0xffu, rb = cnt >> 8;
            const unsigned mp = __ballot_sync(0xffffffffu, lane < kBS && rp == (uint32_t)warp);
            const unsigned mb = __ballot_sync(0xffffffffu, lane < kBS && rb == (uint32_t)warp);
            ip = __ffs(mp) - 1;
            ib = __ffs(mb) - 1;
        }
        const int pnew = l0 + kBS + 2 + ib, vnew = bring_at(vl0, kBS + 2 + ib - kBSlots);
        if (more) stage_head(pnew);
        if (l0 + ip < pb) process_line(l0 + ip, bring_at(vl0, ip));
        if (more) build_line(pnew, vnew);
        __syncthreads();
        vl0 = bring_at(vl0, kBS);
    }
    }   // passes
    if (bad_order) s_unsorted = 1;
    __syncthreads();
    if (tid == 0 && s_unsorted) atomicOr(&cnt->unsorted, 1u);
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device attribute: tpc_cf_create sets it for its device.
cudaError_t fused_blocks_set_attributes()
{
    cudaError_t e = cudaSuccess;
    auto set = [&](const void* f, int bytes) {
        if (e == cudaSuccess) e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    };
    set((const void*)k_fused_blocks<false, false, 2>, 112 * 1024); set((const void*)k_fused_blocks<true, false, 2>, 112 * 1024);
    set((const void*)k_fused_blocks<false, true, 2>, 112 * 1024);  set((const void*)k_fused_blocks<true, true, 2>, 112 * 1024);
    set((const void*)k_fused_blocks<false, false, 3>, 72 * 1024);  set((const void*)k_fused_blocks<true, false, 3>, 72 * 1024);
    set((const void*)k_fused_blocks<false, true, 3>, 72 * 1024);   set((const void*)k_fused_blocks<true, true, 3>, 72 * 1024);
    return e;
}

// Launches k_fused_blocks after the line index is in ws.line_start.  Returns 1 (launched), 0 (not applicable: the
// mean line would not fit the block pool; the caller runs the bitmap kernel instead) or a negative tpc_cf error.
//
// Launch shape: 2 CTAs of 8 warps per SM (the kernel is latency bound — 8 -> 16 warps per SM is 1.67x faster — but
// 20 line slots of ~5 KB leave no room for a third CTA).  Lines too long for the 254-block pool are covered in several
// passes over the time axis (dir, pool and survivor list all scale with the segment length).
int launch_fused_blocks(const Geo& g, const Workspace& ws, const tpc_digit* digits, uint64_t n, uint64_t shape_n,
                        uint32_t q_peak_min, uint32_t q_gate, const Variant& var, const Tuning& tun, bool must,
                        cudaStream_t st, cudaEvent_t ev_k0, cudaEvent_t ev_k1)
{
    uint64_t total_pads = 0;
    for (uint32_t r = 0; r < g.n_rows; ++r) total_pads += g.npads[r];
    total_pads *= g.n_sectors;
    // shape_n: digits of the whole frame when this run covers only some of its sectors (tpc_cf_run_host pipeline)
    const double mean_len = (double)(shape_n ? shape_n : n) / (double)(total_pads ? total_pads : 1);
    // measured on the synthetic frames: 0.38 blocks and 0.16 stage-A survivors per digit
    const double mean_blocks = 0.38 * mean_len, mean_surv = 0.16 * mean_len;

    const bool forced = must || tun.fused_kernel == 2;        // must: the bitmap kernel cannot take this geometry
    const int env_pass = tun.passes;

    const uint32_t fixed = kBWarps * (kStageDepth * 256u + 256u);
    const uint32_t budget = 227u * 1024u / 2u - 1024u - 3328u;     // 2 CTAs per SM: - 1 KB reserved - ~3.2 KB static
    auto shape = [&](uint32_t n_pass, bool must, SlotGeo* out) -> bool {
        SlotGeo sg;
        sg.n_pass = n_pass;
        sg.seg_len = (((g.n_time + n_pass - 1u) / n_pass) + 7u) & ~7u;
        const uint32_t dir_bytes = ((sg.seg_len >> 3) + 2u + 15u) & ~15u;
        sg.pool_off = kDirOff + dir_bytes;
        const double mb = mean_blocks / n_pass + (n_pass > 1 ? 1.0 : 0.0), ms = mean_surv / n_pass;
        sg.scap = (((uint32_t)(ms * 1.6) + 16u) + 3u) & ~3u;
        uint32_t want = (uint32_t)(mb * 1.5) + 24u;                // blocks incl. the zero block
        if (want > 255u) want = 255u;
        const uint32_t per_slot_fixed = sg.pool_off + 4u * sg.scap;
        if (fixed + kBSlots * (per_slot_fixed + 16u * 8u) > budget) return false;
        const uint32_t fit = ((budget - fixed) / kBSlots - per_slot_fixed) / 16u;
        sg.pcap = want < fit ? want : fit;
        if (!must && (double)sg.pcap < mb * 1.25 + 8.0) return false;   // too many lines would overflow the pool
        *out = sg;
        return true;
    };
    // Passes: 1 when the mean line fits the pool, else the fewest that do (each pass costs a partly used chunk and a
    // partly filled survivor / peak batch per line, so fewer is better: measured 1.90 -> 2.87 ms at 2 passes on config 3).
    SlotGeo sg;
    bool have = false;
    for (uint32_t np = 1; np <= 6 && !have; ++np) {
        if (env_pass && (int)np != env_pass) continue;
        if (np > 1 && g.n_time < 64u * np) break;
        have = shape(np, false, &sg);
    }
    if (!have) {
        if (!forced) return 0;
        if (env_pass >= 1 && env_pass <= 8 && g.n_time >= 64u * (uint32_t)env_pass) have = shape((uint32_t)env_pass, true, &sg);
        for (uint32_t np = 1; np <= 8 && !have; ++np) have = (np == 1 || g.n_time >= 64u * np) && shape(np, true, &sg);
        if (!have) return 0;
    }
    if (tun.block_pool >= 2 && tun.block_pool <= 255 && (uint32_t)tun.block_pool <= sg.pcap) sg.pcap = (uint32_t)tun.block_pool;
    if (tun.surv_cap >= 4 && (uint32_t)tun.surv_cap <= sg.scap) sg.scap = (uint32_t)tun.surv_cap & ~3u;
    sg.surv_off = sg.pool_off + 16u * sg.pcap;
    sg.slot_bytes = sg.surv_off + 4u * sg.scap;
    const uint32_t smem = kBSlots * sg.slot_bytes + fixed;

    const uint32_t whole = (g.max_pads + kBS - 1) / kBS * kBS;
    uint32_t pads_per_unit = g.n_planes >= 1184 ? whole : (g.n_planes >= 296 ? 6 * kBS : 3 * kBS);
    if (pads_per_unit > whole) pads_per_unit = whole;
    if (tun.pads_per_unit >= kBS && tun.pads_per_unit <= 256) pads_per_unit = (uint32_t)(tun.pads_per_unit / kBS * kBS);
    const uint32_t upp = (g.max_pads + pads_per_unit - 1) / pads_per_unit;
    if (ev_k0) cudaEventRecord(ev_k0, st);
    g_last_kernel = "k_fused_blocks";
    // a third CTA per SM when the slots are small (short lines): the kernel is latency bound
    const uint32_t budget3 = 227u * 1024u / 3u - 1024u - 3328u;
    const bool three = smem <= budget3 && tun.ctas_per_sm != 2;
    const bool m = sg.n_pass > 1, v = var.active != 0u;
    auto kern = three ? (m ? (v ? k_fused_blocks<true, true, 3> : k_fused_blocks<true, false, 3>)
                           : (v ? k_fused_blocks<false, true, 3> : k_fused_blocks<false, false, 3>))
                      : (m ? (v ? k_fused_blocks<true, true, 2> : k_fused_blocks<true, false, 2>)
                           : (v ? k_fused_blocks<false, true, 2> : k_fused_blocks<false, false, 2>));
    kern<<<g.n_planes * upp, kBThreads, smem, st>>>((const uint2*)digits, (uint32_t)n, g, ws.line_start,
                                                    pads_per_unit, upp, sg, q_peak_min, q_gate, var,
                                                    ws.counters, ws.line_cnt, (uint4*)ws.stage);
    if (ev_k1) cudaEventRecord(ev_k1, st);
    return 1;
}

}  // namespace tpccf
