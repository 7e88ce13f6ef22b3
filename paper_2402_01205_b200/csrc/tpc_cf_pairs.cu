// tpc_cf_pairs.cu — fused path, second generation ("T3c"): block-sparse line slots in shared memory as in
// tpc_cf_blocks.cu (one CTA per (plane, pad range), one WARP per pad LINE, a ring of line slots, one barrier per step
// of 8 lines), rebuilt around the instruction count (profiles/r2a_*: the build loop was 54 % of all issued
// instructions, 95 SASS instructions per 32 digits, 60 % of them on the ALU pipe):
//   * the digit stream reaches shared memory by 1-D bulk copies (cp.async.bulk + mbarrier transaction counts; SASS
//     UBLKCP), 128 digits = 1 KB per copy, issued by one lane into a two-piece ring, two iterations ahead;
//   * every lane works on TWO consecutive digits per iteration (64 digits per warp iteration): one of the two neighbour
//     relations of a digit is in-register, ballots / rank arithmetic / loop control are paid once per 64 digits;
//   * neighbours in the line are read from the staging ring at immediate offsets of one address (no shuffles, no
//     carried state between iterations): lane i holds digits 2i-1 and 2i of the chunk, so that the successor of the
//     last digit is still in the same chunk and the predecessor of the first one is the tail of the chunk before
//     (a 16-byte guard in front of the ring carries it across the wrap);
//   * the in-step load balance (which warp builds / processes which line) is computed once per CTA, not per step;
//   * a slot is cleaned by what its last line used (directory + allocated blocks), not by its capacity;
//   * windows skip the "block not in the pool" test when none of the five lines overflowed its pool.
// Slot of one pad line (all offsets multiples of 16):
//     hdr   [16 B]  word 0: stage-A survivors of the line; 1: first digit this pass streamed; 2: blocks the line opened;
//                   3: 1 if a block did not fit the pool (its dir byte is 0xFF: cells come from the digit array)
//     dir[b] uint8  pool index of the block of time bins 8b-8 .. 8b-1 (0 = the all-zero block)
//     pool[i] 16 B  eight uint16 charges; block 0 stays zero (zero border in time and empty cells, R2)
//     surv[k] u32   (time | charge << 16) of the k-th digit that passed the own-line test (stage A), time order
//   K0 the warp that reuses a slot zeroes it      K1 build: block allocation by ballot / popc, in time order
//   K2 stage A at build time, stage B from the survivor list against lines p-1 / p+1
//   K4 stage C: peaks queued per warp, 5x5 window from the five slots p-2..p+2 -> stage[line_start + k]
// Definition: include/tpc_cf.h (BASELINE.json:north_star; step named in PAPER.md:57).  Readings R1..R19: DESIGN.md §3.
#include <algorithm>

#include "tpc_cf_internal.cuh"

namespace tpccf {

static constexpr int kPThreads = 256;
static constexpr int kPBuild = 4;                 // builder warps (warps 0..3): K0 + K1 + stage A of one line per step each
static constexpr int kPProc = 4;                  // processor warps (warps 4..7): stages B + C of one line per step each
static constexpr int kPS = kPProc;                // lines per step
static constexpr int kPSlots = 2 * kPS + 4;       // lines l0-2 .. l0+S+1 in use, next S being built
static constexpr int kRegsBuild = 72;             // registers per thread after setmaxnreg (launch: 80 = 65536 / (3 * 256));
static constexpr int kRegsProc = 88;              //   4 * 72 + 4 * 88 = 8 * 80.  (ptxas allocates per region: without the
                                                  //   split it spills at 80; at 56 the builder re-computes its lane masks)
static constexpr uint32_t kChunkBytes = 512;      // one build iteration: 64 digits
static constexpr uint32_t kPieceBytes = 1024;     // one bulk copy: 128 digits = two iterations
static constexpr uint32_t kNH = 2;                // staging ring of one line: two pieces, one mbarrier each
static constexpr uint32_t kGuard = 16;            // in front of the ring: copy of the ring's last 16 bytes
static constexpr uint32_t kBufBytes = kGuard + kNH * kPieceBytes;
static constexpr uint32_t kStgBytes = 2 * kBufBytes;   // per builder: the line being built and the head of the next one
static constexpr uint32_t kPqBytes = 256;         // per-processor peak queue (64 entries)
static constexpr uint32_t kHdrBytes = 16;
static constexpr uint32_t kSentT0 = 65470u;       // time of the first trailing sentinel digit (+ up to 63); n_time <= this

// ---- shared-memory accessors on 32-bit addresses -------------------------------------------------------------------
__device__ __forceinline__ uint32_t p_lds32(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint2 p_lds64(uint32_t a)
{
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ uint4 p_lds128(uint32_t a)
{
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ uint32_t p_lds16(uint32_t a)
{
    uint16_t v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint32_t p_lds8(uint32_t a)
{
    uint32_t v;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void p_sts32(uint32_t a, uint32_t v)
{
    asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ void p_sts16(uint32_t a, uint32_t v)
{
    asm volatile("st.shared.u16 [%0], %1;" ::"r"(a), "h"((uint16_t)v) : "memory");
}
__device__ __forceinline__ void p_sts8(uint32_t a, uint32_t v)
{
    asm volatile("st.shared.u8 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ void p_sts128(uint32_t a, uint4 v)
{
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void p_sts128z(uint32_t a)
{
    asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(a), "r"(0u) : "memory");
}

// ---- mbarrier + 1-D bulk copy (global -> shared, completion counted in bytes) ----------------------------------------
__device__ __forceinline__ void p_mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ bool p_mbar_try(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0u;
}
__device__ __forceinline__ void p_mbar_wait(uint32_t bar, uint32_t parity)
{
    while (!p_mbar_try(bar, parity)) { }
}
__device__ __forceinline__ void p_mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void p_bulk_load(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

// ring index of the line at distance d (|d| < kPSlots) from the line whose ring index is v0
__device__ __forceinline__ int pring_at(int v0, int d)
{
    int v = v0 + d;
    v += (v < 0) ? kPSlots : 0;
    v -= (v >= kPSlots) ? kPSlots : 0;
    return v;
}

// K2 stage A (R1, own line) from the digit array (slow path only): the neighbours in time are the adjacent digits of the
// line; an absent one reads 0.  (0,-1) is lexicographically earlier: strict; (0,+1) later: >=.
__device__ __forceinline__ bool p_stage_a(uint32_t y, uint32_t prevy, bool has_prev, uint32_t nexty, bool has_next,
                                          uint32_t T, uint32_t q_peak_min)
{
    const uint32_t t = y & 0xffffu, q = y >> 16;
    const uint32_t qm = (has_prev && (prevy & 0xffffu) + 1u == t) ? (prevy >> 16) : 0u;
    const uint32_t qp = (has_next && (nexty & 0xffffu) == t + 1u && t + 1u < T) ? (nexty >> 16) : 0u;
    return q >= q_peak_min && q > qm && q >= qp;
}

// charge of cell (line, tt) from the digit array (slow path: the line's block pool was full).  Binary search on time.
// Cells outside [0, T) read 0 (R2) whatever the digit array holds there (a digit with time >= T is invalid, R11).
__device__ __noinline__ uint32_t p_cell_from_digits(const uint2* __restrict__ digits, uint32_t gl, uint32_t glen,
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

// Slow path of pwindow (rare: a block of the window is not in the pool): cells of missing blocks come from the digit
// array.  Out of line, result in registers, to keep the hot code small.
struct PWin5 { int c[5]; };
__device__ __noinline__ PWin5 pwindow_slow(uint32_t aA, uint32_t aB, uint32_t dA, uint32_t dB, uint32_t o, int t0, int n,
                                           const uint2* __restrict__ digits, uint32_t gl, uint32_t glen, uint32_t T)
{
    PWin5 r;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
        const bool inA = o + (uint32_t)k < 8u;
        const uint32_t d = inA ? dA : dB;
        r.c[k] = k >= n ? 0
               : (d != 0xFFu ? (int)p_lds16((inA ? aA : aB) + 2u * (uint32_t)k)
                             : (int)p_cell_from_digits(digits, gl, glen, (uint32_t)(t0 + k), T));
    }
    return r;
}

// charges of the window t-H..t+H of the line in slot `slot` (0 where no digit): c[k] is time t-H+k.
// dsub = first time bin of the pass / 8.  OVF (warp-uniform): some line of the neighbourhood has blocks outside its
// pool (their dir byte is 0xFF): only then are the directory bytes tested.  lidx = pad index of the line, slow path only.
template <int H>
__device__ __forceinline__ void pwindow(uint32_t slot, uint32_t dsub, const SlotGeo& sg, int t, int (&c)[2 * H + 1],
                                        const uint2* __restrict__ digits, const uint32_t* s_ls, int lidx, int P,
                                        uint32_t T, bool OVF)
{
    const uint32_t u = (uint32_t)(t + 8 - H);                 // first cell, shifted by the 8-bin guard block
    const uint32_t dir = slot + kHdrBytes - dsub;
    const uint32_t dA = p_lds8(dir + (u >> 3));
    const uint32_t dB = p_lds8(dir + ((u + 2 * H) >> 3));
    const uint32_t o = u & 7u;
    const uint32_t base = slot + sg.pool_off + 2u * o;
    const uint32_t aA = base + (dA << 4), aB = base + (dB << 4) - 16u;
    if (!OVF || (dA != 0xFFu && dB != 0xFFu)) {
        c[0] = (int)p_lds16(aA);
#pragma unroll
        for (int k = 1; k < 2 * H + 1; ++k) c[k] = (int)p_lds16((o < (uint32_t)(8 - k) ? aA : aB) + 2u * (uint32_t)k);
    } else {
        const bool inside = lidx >= 0 && lidx < P;
        const uint32_t gl = inside ? s_ls[lidx] : 0u;
        const uint32_t glen = inside ? s_ls[lidx + 1] - gl : 0u;
        const PWin5 r = pwindow_slow(aA, aB, dA, dB, o, t - H, 2 * H + 1, digits, gl, glen, T);
#pragma unroll
        for (int k = 0; k < 2 * H + 1; ++k) c[k] = r.c[k];
    }
}

// Piece k of a line that touches a ragged end of the digit array (called by one lane; rare: at most two lines of a
// run).  Bulk copies move the 16-byte aligned part [bs, be) of the piece, cut at the line's end rounded out to 16 bytes;
// the first / last digit of the whole array, where it is ragged, is copied by hand before the barrier is armed (the
// arrive releases those stores to the lanes that wait on the barrier).
__device__ __noinline__ void p_issue_piece_slow(const uint2* __restrict__ digits, uint32_t base, uint32_t lend, uint32_t k,
                                            uint32_t ring, uint32_t bar0, uint32_t gpar, uint32_t al_lo, uint32_t al_hi)
{
    const int s = (int)base + 128 * (int)k;             // -1: the piece in front of digit 0 of a buffer 8 bytes off
    const uint32_t e = min((uint32_t)(s + 128), lend);
    const uint32_t dst = ring + (k & 1u) * kPieceBytes;
    const uint32_t bar = bar0 + 8u * (k & 1u);
    uint32_t bs = (uint32_t)s, be = e + ((e + gpar) & 1u);
    if (s < (int)al_lo) {
        bs = al_lo;
        if (e > 0u && bs > 0u) {
            const uint2 d = __ldg(digits);
            asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(dst + 8u), "r"(d.x), "r"(d.y) : "memory");
        }
    }
    if (be > al_hi) {
        be = al_hi;
        if (e > be && (int)be >= s) {
            const uint2 d = __ldg(digits + be);
            asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(dst + 8u * (uint32_t)((int)be - s)), "r"(d.x), "r"(d.y) : "memory");
        }
    }
    if (be > bs) p_bulk_load(dst + 8u * (uint32_t)((int)bs - s), digits + bs, 8u * (be - bs), bar);
    else p_mbar_arrive(bar);
}

// MULTI: the time axis is covered in sg.n_pass > 1 passes (long lines).  VAR: flags / cuts requested (V1..V3); the
// default instantiation carries none of that code.
template <bool MULTI, bool VAR>
__global__ void __launch_bounds__(kPThreads, 3)
k_fused_pairs(const uint2* __restrict__ digits, uint32_t n, Geo g, const uint32_t* __restrict__ line_start,
              uint32_t pads_per_unit, uint32_t units_per_plane, SlotGeo sg, uint32_t q_peak_min, uint32_t q_gate,
              Variant var, Counters* cnt, uint32_t* __restrict__ line_cnt, uint4* __restrict__ stage)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ uint32_t s_ls[260];          // line starts of this plane: s_ls[p], p = 0..max_pads, then next plane's start
    __shared__ uint32_t s_pos[260];         // first digit of line p that the current pass needs (time >= pass start - 2)
    __shared__ uint32_t s_cnt[260];         // peaks of line p found by the passes so far
    __shared__ __align__(8) unsigned long long s_bar[kPBuild * 2 * kNH];   // per builder, buffer and piece
    __shared__ int s_unsorted;

    const uint32_t plane = blockIdx.x / units_per_plane, unit = blockIdx.x % units_per_plane;
    const uint32_t sector = plane / g.n_rows, row = plane % g.n_rows;
    const int P = (int)g.npads[row];
    const int pa = (int)(unit * pads_per_unit);
    const int pb = min(pa + (int)pads_per_unit, P);
    const uint32_t T = g.n_time;
    const int tid = threadIdx.x, lane = tid & 31;
    const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);    // (the shuffle tells the compiler it is warp-uniform)
    const uint32_t w0_base = sector | (row << 8);
    const uint32_t lt_mask = (1u << lane) - 1u;
    const uint32_t le_mask = lt_mask | (1u << lane);

    const uint32_t sm0 = (uint32_t)__cvta_generic_to_shared(smem_raw);
    const bool builder = warp < kPBuild;
    const int rw = builder ? warp : warp - kPBuild;            // index within the role
    // staging of builder rw: two buffers (guard + two pieces each); the line in hand uses buffer `buf`
    const uint32_t stg0 = sm0 + kPSlots * sg.slot_bytes + (uint32_t)rw * kStgBytes + kGuard;
    const uint32_t pqa = sm0 + kPSlots * sg.slot_bytes + kPBuild * kStgBytes + (uint32_t)rw * kPqBytes;
    const uint32_t barb = (uint32_t)__cvta_generic_to_shared(&s_bar[rw * 2 * kNH]);
    uint32_t ring = stg0, bar0 = barb, pbit = 0u;              // of the buffer in hand (set_buf)
    auto set_buf = [&](uint32_t buf) { ring = stg0 + buf * kBufBytes; bar0 = barb + buf * (8u * kNH); pbit = buf * kNH; };
    // 16-byte alignment of digit j in global memory: (j + gpar) even
    const uint32_t gpar = (uint32_t)((reinterpret_cast<uintptr_t>(digits) >> 3) & 1u);
    const uint32_t al_lo = gpar;                                  // first and one-past-last digit a bulk copy may touch
    const uint32_t al_hi = n - ((n + gpar) & 1u);

    for (int i = tid; i <= (int)g.LS; i += kPThreads) {
        const uint32_t v = line_start[plane * g.LS + i];
        s_ls[i] = v; s_pos[i] = v; s_cnt[i] = 0u;
    }
    if (tid == 0) s_unsorted = 0;
    if (tid < kPBuild * 2 * (int)kNH) p_mbar_init((uint32_t)__cvta_generic_to_shared(&s_bar[tid]), 1u);
    // every slot starts as an empty line (lines outside the plane keep this state: zero border in pad, R2)
    for (uint32_t x = (uint32_t)tid * 16u; x < kPSlots * sg.slot_bytes; x += kPThreads * 16u) p_sts128z(sm0 + x);
    __syncthreads();

    if (pa >= P && unit != 0) return;    // nothing in this pad range (rows with fewer pads)

    uint32_t bad_order = 0u;
    // monotone line starts: a garbage index from unsorted input must not produce negative lengths or unbounded work
    for (int i = tid; i < (int)g.LS; i += kPThreads) if (s_ls[i] > s_ls[i + 1]) bad_order = 1u;
    if (s_ls[g.LS] > n) bad_order = 1u;
    if (__syncthreads_or((int)bad_order)) {
        if (tid == 0) atomicOr(&cnt->unsorted, 1u);
        return;
    }

    // gap of the plane: digits with pad >= npads[row] (or a row/sector beyond the geometry) — all invalid (R11)
    if (unit == 0) {
        const uint32_t gb = s_ls[P], ge = s_ls[g.LS];
        if (ge > gb) {
            for (uint32_t j = gb + tid; j < ge; j += kPThreads) {
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
    uint32_t phase = 0u;                    // bit 2 buf + h: parity the next wait on piece h of staging buffer buf expects

    // ---- staging: piece k of a line = digit slots [base + 128k, base + 128k + 128), base = first digit of the pass in
    // the line, rounded down to a 16-byte boundary of global memory; ring half k mod 2.  Only lane 0 issues.
    // Bulk copies move the 16-byte aligned part [bs, be) of the piece, cut at the line's end rounded out to 16 bytes; the
    // first / last digit of the whole array, where it is ragged (at most one each), is copied by hand before the barrier
    // is armed (the arrive releases those stores to the lanes that wait on the barrier).
    // The usual case (warp-uniform test): the line touches neither ragged end of the array, so piece k is one copy of
    // [base + 128k, min(base + 128k + 128, lend rounded out to 16 bytes)).  Called by all lanes; lane 0 issues.
    auto issue_piece = [&](uint32_t base, uint32_t lend, uint32_t k) {
        const uint32_t lend_al = lend + ((lend + gpar) & 1u);
        if ((int)base >= (int)al_lo && lend_al <= al_hi) {
            const uint32_t s = base + 128u * k;
            const uint32_t bytes = 8u * (min(s + 128u, lend_al) - s);
            if (lane == 0) p_bulk_load(ring + (k & 1u) * kPieceBytes, digits + s, bytes, bar0 + 8u * (k & 1u));
        } else if (lane == 0) {
            p_issue_piece_slow(digits, base, lend, k, ring, bar0, gpar, al_lo, al_hi);
        }
    };
    // The head of the line this warp builds next: its first two pieces, issued a step ahead (so the global latency is
    // covered) as ONE copy of up to 256 digits that completes on the barrier of piece 0; a line at a ragged end of the
    // array gets two separate pieces instead (head_split below).
    auto stage_head = [&](int p) {
        if (p < blo || p >= bhi) return;
        const uint32_t lbeg = s_pos[p], lend = s_ls[p + 1];
        if (lend == lbeg) return;
        const uint32_t base = lbeg - ((lbeg + gpar) & 1u);
        const uint32_t lend_al = lend + ((lend + gpar) & 1u);
        if ((int)base >= (int)al_lo && lend_al <= al_hi) {
            if (lane == 0) p_bulk_load(ring, digits + base, 8u * (min(base + 256u, lend_al) - base), bar0);
        } else if (lane == 0) {
            p_issue_piece_slow(digits, base, lend, 0u, ring, bar0, gpar, al_lo, al_hi);
            if (lend - base > 128u) p_issue_piece_slow(digits, base, lend, 1u, ring, bar0, gpar, al_lo, al_hi);
        }
    };

    // ---- K0 + K1 + stage A: this warp (re)builds slot v as line p ---------------------------------------------------
    // The loop body carries no "does this digit exist" logic: the digit slots in front of the line's first digit and
    // behind its last one are overwritten in the staging ring with SENTINEL digits (right key word, charge 1, a time
    // >= n_time + 1: 0xffff in front, kSentT0 + k behind, ascending) once their chunk has landed.  A sentinel stores no
    // cell, opens no block, survives no test, is adjacent to no real digit and keeps the order check quiet.
    // (n_time < kSentT0 is a condition of this kernel's launcher.)
    auto build_line = [&](int p, int v) {
        const uint32_t slot = sm0 + (uint32_t)v * sg.slot_bytes;
        {
            // K0: header + directory, and the pool blocks the slot's last line opened
            const uint32_t oldn = __shfl_sync(0xffffffffu, p_lds32(slot + 8u), 0);
            const uint32_t pend = sg.pool_off + 16u * (min(oldn, sg.pcap - 1u) + 1u);
            for (uint32_t x = (uint32_t)lane * 16u; x < pend; x += 512u) p_sts128z(slot + x);
            __syncwarp();
        }
        if (p < blo || p >= bhi) return;                    // a line outside the plane / the halo: stays empty
        const uint32_t lbeg = s_pos[p], lend = s_ls[p + 1], len = lend - lbeg;
        if (lane == 0) p_sts32(slot + 4u, lbeg);            // hdr word 1: where this pass started in the line
        if (len == 0) return;
        const uint32_t lk = w0_base | ((uint32_t)p << 16);  // key word of the line's digits
        const uint32_t a_dir1 = slot + kHdrBytes + 1u - (MULTI ? dsub : 0u); // dir byte of the block of time t: a_dir1 + (t >> 3)
        const uint32_t a_pool = slot + sg.pool_off, a_surv = slot + sg.surv_off;
        const uint32_t own_span = thi - tlo, win_span = whi - wlo;
        const uint32_t nlo = thi - 2u;                      // the next pass needs the line from this time on
        const uint32_t odd = (lbeg + gpar) & 1u;
        const uint32_t base = lbeg - odd;
        const uint32_t L = len + odd;                       // digit slots from base to the end of the line
        const uint32_t np = (L + 127u) >> 7;                // pieces of the line
        // was the head issued as two pieces (stage_head's rule)?  Else piece 1 came with piece 0: no wait of its own
        const bool head_split = !((int)base >= (int)al_lo && lend + ((lend + gpar) & 1u) <= al_hi);
        const uint32_t c_last = L >> 6;                     // iteration c works on slots 64c-1 .. 64c+62
        const uint32_t pcap = sg.pcap, scap = sg.scap;
        uint32_t nblk = 0u, nsurv = 0u;                     // warp-uniform running counts
        uint32_t ymin = 0xffffffffu;                        // per lane: smallest (time | charge << 16) seen: < 0x10000 = a zero charge
        const uint32_t ylast = __ldg(&digits[lend - 1u].y);  // the line's last digit: is its time in range? (R11)
        uint32_t next_pos = lend;                           // first digit with time >= nlo (warp-uniform)
        bool found = false;
        uint32_t iters = 0u;                                // iterations run
        // order check of the pairs (prev, a) and (a, b): off in iteration 0 where the earlier one is a leading sentinel
        uint32_t m_pa = (lane == 0 || (lane == 1 && odd)) ? 0u : 0x80000000u, m_ab = lane == 0 ? 0u : 0x80000000u;
        uint32_t bad = 0u;
        // piece k = chunks 2k, 2k+1 (ring half k & 1); iteration c reads chunk c and the tail of chunk c - 1
        uint32_t c = 0u;
        bool done = false;
        for (uint32_t k = 0; !done; ++k) {
            const uint32_t h = k & 1u;
            if (k < np && (k != 1u || head_split)) {        // has the piece landed?
                p_mbar_wait(bar0 + 8u * h, (phase >> (pbit + h)) & 1u);
                phase ^= 1u << (pbit + h);
            }
#pragma unroll
            for (uint32_t j = 0; j < 2u; ++j) {
            if (done) break;
            const uint32_t ent = ring + h * kPieceBytes + j * kChunkBytes;
            ++iters;
            if (c == 0u) {
                // leading sentinels: slots -2, -1 (the guard) and, if the line starts 8 bytes off a boundary, slot 0
                if (lane == 0) {
                    p_sts128(ring - kGuard, make_uint4(lk, 0x1ffffu, lk, 0x1ffffu));
                    if (odd) asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(ring), "r"(lk), "r"(0x1ffffu) : "memory");
                }
            }
            if (c == c_last) {
                // trailing sentinels: slots L .. 64 c + 63 of this (the last) chunk
                const uint32_t k0 = L - 64u * c;            // first sentinel slot within the chunk (0 .. 63)
#pragma unroll
                for (uint32_t r = 0; r < 2u; ++r) {
                    const uint32_t kk = k0 + (uint32_t)lane + 32u * r;
                    if (kk < 64u)
                        asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(ent + 8u * kk), "r"(lk), "r"(0x10000u + kSentT0 + kk - k0) : "memory");
                }
            }
            if (c == 0u || c == c_last) __syncwarp();
            const uint32_t addr = ent + 16u * (uint32_t)lane;      // digit b; a at -8; chunk 0 of the ring: lane 0 reads the guard
            const uint2 A = p_lds64(addr - 8u), B = p_lds64(addr);
            const uint32_t prevy = p_lds32(addr - 12u), nexty = p_lds32(addr + 12u);
            // the ring's last 16 bytes are kept in the guard for lane 0 of the next iteration (chunk 0 of the ring)
            if (h == 1u && j == 1u && lane == 31) p_sts128(ring - kGuard, p_lds128(addr));
            __syncwarp();
            // the piece in front of this one is dead now: its half receives the piece after this one
            if (j == 0u && k >= 1u && k + 1u < np) issue_piece(base, lend, k + 1u);
            const uint32_t ya = A.y, yb = B.y;
            const uint32_t ta = ya & 0xffffu, tb = yb & 0xffffu, tp = prevy & 0xffffu, tn = nexty & 0xffffu;
            const uint32_t qa = ya >> 16, qb = yb >> 16, qp = prevy >> 16, qn = nexty >> 16;
            // DIGITS_SORTED promise: right line, strictly ascending times (a duplicate cell breaks it too)
            const uint32_t d_pa = ta - tp - 1u, d_ab = tb - ta - 1u, d_bn = tn - tb - 1u;   // 0: adjacent cells; < 0: not ascending
            bad |= ((A.x ^ lk) | (B.x ^ lk)) & 0x00ffffffu;
            bad |= (d_pa & m_pa) | (d_ab & m_ab);
            m_pa = 0x80000000u; m_ab = 0x80000000u;
            const bool inb_a = MULTI ? (ta - wlo) < win_span : ta < T;    // a cell this pass stores
            const bool inb_b = MULTI ? (tb - wlo) < win_span : tb < T;
            const bool own_a = MULTI ? (ta - tlo) < own_span : inb_a;     // a cell this pass decides
            const bool own_b = MULTI ? (tb - tlo) < own_span : inb_b;
            ymin = min(ymin, min(ya, yb));                  // R11: zero charges are looked for here, counted below
            // All four ballots and their bit counts come first (independent of each other: the builder warps are bound by
            // the latency of dependent chains, not by issue slots), the stores after.
            // K1: blocks are allocated in time order: a digit opens a block iff the digit before it is in another one
            const bool head_a = inb_a && (ta ^ tp) > 7u;
            const bool head_b = inb_b && (tb ^ ta) > 7u;
            // K2 stage A (R1, own line).  (0,-1) is earlier: the digit loses to an adjacent previous charge >= its
            // own; (0,+1) is later: it loses to an adjacent next charge > its own (cells at time >= T read 0).
            // With qe = charge of the adjacent cell (0 if there is no digit there): survive iff q >= max(q_peak_min,
            // qe(previous) + 1, qe(next)).
            const bool adj_ab = d_ab == 0u && tb < T;
            const uint32_t qpe_a = d_pa == 0u ? qp + 1u : 0u, qne_a = adj_ab ? qb : 0u;
            const uint32_t qpe_b = adj_ab ? qa + 1u : 0u, qne_b = (d_bn == 0u && tn < T) ? qn : 0u;
            const bool surv_a = own_a && qa >= max(max(qpe_a, qne_a), q_peak_min);
            const bool surv_b = own_b && qb >= max(max(qpe_b, qne_b), q_peak_min);
            const unsigned hma = __ballot_sync(0xffffffffu, head_a), hmb = __ballot_sync(0xffffffffu, head_b);
            const unsigned sma = __ballot_sync(0xffffffffu, surv_a), smb = __ballot_sync(0xffffffffu, surv_b);
            const uint32_t idx_a = nblk + (uint32_t)__popc(hma & le_mask) + (uint32_t)__popc(hmb & lt_mask);   // 1-based
            const uint32_t idx_b = idx_a + (head_b ? 1u : 0u);
            const uint32_t pos_a = nsurv + (uint32_t)__popc(sma & lt_mask) + (uint32_t)__popc(smb & lt_mask);
            const uint32_t pos_b = pos_a + (surv_a ? 1u : 0u);
            nblk += (uint32_t)__popc(hma) + (uint32_t)__popc(hmb);     // blocks opened so far (warp-uniform arithmetic)
            nsurv += (uint32_t)__popc(sma) + (uint32_t)__popc(smb);    // survivors so far
            if (nblk < pcap) {                              // (warp-uniform) every block so far is in the pool
                if (head_a) p_sts8(a_dir1 + (ta >> 3), idx_a);
                if (head_b) p_sts8(a_dir1 + (tb >> 3), idx_b);
                if (inb_a) p_sts16(a_pool + (idx_a << 4) + ((ta & 7u) << 1), qa);
                if (inb_b) p_sts16(a_pool + (idx_b << 4) + ((tb & 7u) << 1), qb);
            } else {
                if (head_a) p_sts8(a_dir1 + (ta >> 3), idx_a < pcap ? idx_a : 0xFFu);
                if (head_b) p_sts8(a_dir1 + (tb >> 3), idx_b < pcap ? idx_b : 0xFFu);
                if (inb_a && idx_a < pcap) p_sts16(a_pool + (idx_a << 4) + ((ta & 7u) << 1), qa);
                if (inb_b && idx_b < pcap) p_sts16(a_pool + (idx_b << 4) + ((tb & 7u) << 1), qb);
            }
            if (nsurv <= scap) {                            // (warp-uniform) the list holds every survivor so far
                if (surv_a) p_sts32(a_surv + (pos_a << 2), ya);
                if (surv_b) p_sts32(a_surv + (pos_b << 2), yb);
            } else {
                if (surv_a && pos_a < scap) p_sts32(a_surv + (pos_a << 2), ya);
                if (surv_b && pos_b < scap) p_sts32(a_surv + (pos_b << 2), yb);
            }
            if (MULTI && !last_pass) {
                // where the next pass starts in this line, and whether this pass has seen all it stores
                const bool tail = c == c_last;              // this iteration reaches the last digit of the line
                const uint32_t t31 = __shfl_sync(0xffffffffu, tb, 31);   // time of the iteration's last slot
                if (!found && (tail || t31 >= nlo)) {
                    unsigned ma = __ballot_sync(0xffffffffu, ta >= nlo);
                    unsigned mb = __ballot_sync(0xffffffffu, tb >= nlo);
                    if (c == 0u) { ma &= ~1u; mb &= ~odd; }     // leading sentinels
                    if (ma | mb) {
                        // first slot in order a0 b0 a1 b1 ...; line index of lane i's a is 64c + 2i - 1 - odd
                        const int fa = ma ? __ffs(ma) - 1 : 64, fb = mb ? __ffs(mb) - 1 : 64;
                        const uint32_t first = fa <= fb ? 2u * (uint32_t)fa : 2u * (uint32_t)fb + 1u;
                        next_pos = min(lbeg + 64u * c + first - 1u - odd, lend);    // (a trailing sentinel: lend)
                        found = true;
                    }
                }
                if (!tail && t31 >= whi) done = true;       // every later digit is beyond the window
            }
            if (c == c_last) done = true;
            ++c;
            }   // chunks of the piece
        }
        bad_order |= bad;
        // chunks that were issued for iterations this pass did not run (early exit): consume their barrier phases
        if (MULTI) {
            const uint32_t last = iters - 1u;               // last iteration run: chunk `last`, piece last >> 1
            // issued: pieces 0, 1 ahead of the loop, piece k + 1 in the first chunk of every piece k >= 1
            const uint32_t issued = min(np, 2u + (last >> 1)), waited = min(np, (last >> 1) + 1u);
            for (uint32_t k = waited; k < issued; ++k) {
                const uint32_t h = k & 1u;
                if (k == 1u && !head_split) continue;
                p_mbar_wait(bar0 + 8u * h, (phase >> (pbit + h)) & 1u);
                phase ^= 1u << (pbit + h);
            }
        }
        if (lane == 0) {
            p_sts32(slot, nsurv);
            p_sts32(slot + 8u, nblk);
            p_sts32(slot + 12u, nblk >= pcap ? 1u : 0u);
            if (MULTI && !last_pass) s_pos[p] = next_pos;
        }
        // R11: digits that are no cell with charge (time out of range, zero charge) are skipped and counted, by the pass
        // that owns their time (the last one for times >= n_time).  They are rare: found by the minimum above and by
        // the line's last digit, then counted from the digit array.
        if (p >= pa && p < pb) {                            // halo lines are counted by the unit that owns them
            const bool zero_q = __reduce_min_sync(0xffffffffu, ymin) < 0x10000u;
            const bool late_t = (!MULTI || last_pass) && (ylast & 0xffffu) >= T;
            if (zero_q || late_t) {
                uint32_t nbad = 0u;
                for (uint32_t j = lbeg + (uint32_t)lane; j < lend; j += 32u) {
                    const uint32_t y = __ldg(&digits[j].y), t = y & 0xffffu;
                    const bool own = MULTI ? (t - tlo) < own_span : t < T;
                    const bool considered = !MULTI ? true : (last_pass ? t >= tlo : own);
                    if (considered && !(own && y >= 0x10000u)) ++nbad;
                }
                nbad = __reduce_add_sync(0xffffffffu, nbad);
                if (nbad != 0u && lane == 0) atomicAdd(&cnt->n_bad, (unsigned long long)nbad);
            }
        }
    };

    // ---- K2 stage B + K4 stage C for line p (ring index vp), owned by this warp -------------------------------------
    auto process_line = [&](int p, int vp, const bool OVF) {
        const uint32_t gl = s_ls[p], lend = s_ls[p + 1];
        uint32_t sl[5];                                     // slots of lines p-2 .. p+2 (empty outside the plane, R2)
        {
            const uint32_t ring_end = sm0 + kPSlots * sg.slot_bytes;
            uint32_t a0 = sm0 + (uint32_t)pring_at(vp, -2) * sg.slot_bytes;
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
                for (int a = 0; a < 5; ++a) pwindow<2>(sl[a], MULTI ? dsub : 0u, sg, (int)t, c[a], digits, s_ls, p + a - 2, P, T, OVF);
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
                pwindow<1>(sl[1], MULTI ? dsub : 0u, sg, t, cm, digits, s_ls, p - 1, P, T, OVF);   // line p-1: earlier, strict (R1)
                pwindow<1>(sl[3], MULTI ? dsub : 0u, sg, t, cp, digits, s_ls, p + 1, P, T, OVF);   // line p+1: later, >=
                peak = q > (uint32_t)max(cm[0], max(cm[1], cm[2])) && q >= (uint32_t)max(cp[0], max(cp[1], cp[2]));
            }
            const unsigned pm = __ballot_sync(0xffffffffu, peak);
            if (pm == 0u) return;
            if (peak) p_sts32(pqa + ((pcount + (uint32_t)__popc(pm & lt_mask)) << 2), y);
            pcount += (uint32_t)__popc(pm);
            __syncwarp();
            if (pcount >= 32u) {
                pdone += moments(true, p_lds32(pqa + ((uint32_t)lane << 2)));
                const uint32_t mv = p_lds32(pqa + (((uint32_t)lane + 32u) << 2));
                __syncwarp();
                p_sts32(pqa + ((uint32_t)lane << 2), mv);
                pcount -= 32u;
                __syncwarp();
            }
        };

        const uint32_t ns = p_lds32(sl[2]);
        const uint32_t nst = min(ns, sg.scap);
        for (uint32_t i = 0; i < nst; i += 32u) {
            const bool act = i + (uint32_t)lane < nst;
            stage_b(act, act ? p_lds32(sl[2] + sg.surv_off + ((i + (uint32_t)lane) << 2)) : 0u);
        }
        if (ns > sg.scap) {
            // rare: more survivors than the slot's list holds.  Stage A again from the digit array, from where this
            // pass started in the line; survivors whose ordinal is >= scap were not listed and are tested here
            // (still in time order).
            const uint32_t lbeg = p_lds32(sl[2] + 4u), len = lend - lbeg;
            uint32_t seen = 0;
            for (uint32_t c0 = 0; c0 < len; c0 += 32u) {
                const uint32_t jl = c0 + (uint32_t)lane;
                const bool act = jl < len;
                const uint32_t y = act ? __ldg(&digits[lbeg + jl].y) : 0u;
                const uint32_t prevy = jl > 0u && act ? __ldg(&digits[lbeg + jl - 1u].y) : 0u;
                const uint32_t nexty = jl + 1u < len ? __ldg(&digits[lbeg + jl + 1u].y) : 0u;
                const bool surv = act && (MULTI ? ((y & 0xffffu) - tlo) < (thi - tlo) : (y & 0xffffu) < T) &&
                                  p_stage_a(y, prevy, jl > 0u, nexty, jl + 1u < len, T, q_peak_min);
                const unsigned smk = __ballot_sync(0xffffffffu, surv);
                const uint32_t ord = seen + (uint32_t)__popc(smk & lt_mask);
                seen += (uint32_t)__popc(smk);
                if (seen > sg.scap) stage_b(surv && ord >= sg.scap, y);
                if (seen >= ns) break;                      // all survivors of this pass have been seen
            }
        }
        if (pcount > 16u) {
            pdone += moments((uint32_t)lane < pcount, p_lds32(pqa + (((uint32_t)lane & 31u) << 2)));
        } else if (pcount > 0u) {
            // the usual case (a line has ~14 peaks): two lanes per peak, each gathers the rows on one side of the
            // peak plus the peak's row (3 windows instead of 5); the halves of the integer sums are added by shuffle
            const uint32_t i = (uint32_t)lane & 15u;
            const bool neg = lane >= 16;                        // this lane takes dp < 0 (lines p-2, p-1)
            const bool valid = i < pcount;
            ClusterSums h = {0, 0, 0, 0, 0};
            uint32_t y = 0u;
            if (valid) {
                y = p_lds32(pqa + (i << 2));
                const int t = (int)(y & 0xffffu);
                int o[5], m[5], z[5];
                pwindow<2>(neg ? sl[0] : sl[4], MULTI ? dsub : 0u, sg, t, o, digits, s_ls, neg ? p - 2 : p + 2, P, T, OVF);
                pwindow<2>(neg ? sl[1] : sl[3], MULTI ? dsub : 0u, sg, t, m, digits, s_ls, neg ? p - 1 : p + 1, P, T, OVF);
                pwindow<2>(sl[2], MULTI ? dsub : 0u, sg, t, z, digits, s_ls, p, P, T, OVF);
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
    auto process = [&](int p, int vp) {
        if (s_ls[p + 1] == s_ls[p]) return;                 // line_cnt stays 0 (cleared per run)
        // does any of the five lines keep blocks outside its pool?  (hdr word 3; warp-uniform)
        uint32_t ovf = 0u;
#pragma unroll
        for (int a = -2; a <= 2; ++a) ovf |= p_lds32(sm0 + (uint32_t)pring_at(vp, a) * sg.slot_bytes + 12u);
        process_line(p, vp, ovf != 0u);
    };

    // ---- main loop -------------------------------------------------------------------------------------------------
    // Warps 0..3 BUILD, warps 4..7 PROCESS, concurrently, one line per warp and step, ONE barrier per step of S = 4 lines:
    //   round -2, -1   builders fill the ring with lines pa-2 .. pa+S+1 (S + 4 = 8 lines); processors wait
    //   step l0 >= pa  processor i runs stages B + C on line l0 + i (lines l0-2 .. l0+S+1 are complete);
    //                  builder i rebuilds the slot of a line that left the ring (l0-S-2 .. l0-3) as line l0 + S + 2 + i
    // Ring index of line p is (p - (pa - 2)) mod kPSlots.  A builder issues the bulk copies of the head of its NEXT line
    // (other staging buffer) before it builds the current one, so a copy has a whole step to land.
    // The kernel is launched with 80 registers per thread (3 CTAs per SM) and each warp group re-sizes its share.
    // The time axis is covered in sg.n_pass passes over the unit's lines.
    const int n_rounds = 2 + (pb - pa + kPS - 1) / kPS;        // per pass
    if (builder) {
        asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegsBuild));
        // line of this builder in round r (r = step + 2); returns false if there is none
        auto line_of = [&](int r, int& p, int& v) -> bool {
            if (r < 2) {
                const int i = r * kPS + rw;                     // ring index = line - (pa - 2)
                p = pa - 2 + i; v = i;
                return i < kPS + 4;
            }
            const int l0 = pa + (r - 2) * kPS;
            p = l0 + kPS + 2 + rw;
            v = (p - (pa - 2)) % kPSlots;
            return l0 + kPS < pb;                               // lines l0+S+2 .. l0+2S+1 enter the ring in this step
        };
        uint32_t buf = 0u;
        for (uint32_t pass = 0; pass < (MULTI ? sg.n_pass : 1u); ++pass) {
            if (MULTI) {
                last_pass = pass + 1u == sg.n_pass;
                tlo = pass * sg.seg_len;
                thi = last_pass ? T : min(tlo + sg.seg_len, T);
                wlo = tlo >= 2u ? tlo - 2u : 0u;
                whi = min(thi + 2u, T);
                dsub = tlo >> 3;
            }
            // round r builds the line whose head round r - 1 issued (one call site each: the code is large)
            int p = 0, v = 0;
            bool cur = false;
            for (int r = -1; r < n_rounds; ++r) {
                int pn = 0, vn = 0;
                const bool nxt = r + 1 < n_rounds && line_of(r + 1, pn, vn);
                if (nxt) { set_buf(buf ^ 1u); stage_head(pn); }
                if (cur) { set_buf(buf); build_line(p, v); }
                buf ^= 1u;
                cur = nxt; p = pn; v = vn;
                if (r >= 1) __syncthreads();
            }
        }
    } else {
        asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegsProc));
        for (uint32_t pass = 0; pass < (MULTI ? sg.n_pass : 1u); ++pass) {
            if (MULTI) {
                last_pass = pass + 1u == sg.n_pass;
                tlo = pass * sg.seg_len;
                thi = last_pass ? T : min(tlo + sg.seg_len, T);
                dsub = tlo >> 3;
            }
            int vl0 = 2;                                        // ring index of line l0
            for (int r = 0; r < n_rounds; ++r) {
                if (r >= 2) {
                    const int l0 = pa + (r - 2) * kPS;
                    if (l0 + rw < pb) process(l0 + rw, pring_at(vl0, rw));
                    vl0 = pring_at(vl0, kPS);
                }
                if (r != 0) __syncthreads();
            }
        }
    }
    if (bad_order) s_unsorted = 1;
    __syncthreads();
    if (tid == 0 && s_unsorted) atomicOr(&cnt->unsorted, 1u);
}

cudaError_t fused_pairs_set_attributes()
{
    cudaError_t e = cudaSuccess;
    auto set = [&](const void* f, int bytes) {
        if (e == cudaSuccess) e = cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    };
    set((const void*)k_fused_pairs<false, false>, 112 * 1024); set((const void*)k_fused_pairs<true, false>, 112 * 1024);
    set((const void*)k_fused_pairs<false, true>, 112 * 1024);  set((const void*)k_fused_pairs<true, true>, 112 * 1024);
    return e;
}

// Launches k_fused_pairs after the line index is in ws.line_start.  Returns 1 (launched), 0 (not applicable: the
// mean line would not fit the block pool in <= 6 passes; the caller runs the bitmap kernel instead) or a negative
// tpc_cf error.  Launch shape: 3 CTAs of 4 + 4 warps per SM.  Lines too long
// for the 254-block pool are covered in several passes over the time axis (dir, pool and survivor list all scale with
// the segment length).
int launch_fused_pairs(const Geo& g, const Workspace& ws, const tpc_digit* digits, uint64_t n, uint64_t shape_n,
                       uint32_t q_peak_min, uint32_t q_gate, const Variant& var, const Tuning& tun, bool must,
                       cudaStream_t st, cudaEvent_t ev_k0, cudaEvent_t ev_k1)
{
    if (g.n_time >= kSentT0) return 0;        // the sentinel digits of the build loop need times above every real one
    uint64_t total_pads = 0;
    for (uint32_t r = 0; r < g.n_rows; ++r) total_pads += g.npads[r];
    total_pads *= g.n_sectors;
    // shape_n: digits of the whole frame when this run covers only some of its sectors (tpc_cf_run_host pipeline)
    const double mean_len = (double)(shape_n ? shape_n : n) / (double)(total_pads ? total_pads : 1);
    // measured on the synthetic frames: 0.38 blocks and 0.16 stage-A survivors per digit
    const double mean_blocks = 0.38 * mean_len, mean_surv = 0.16 * mean_len;

    const uint32_t fixed = kPBuild * kStgBytes + kPProc * kPqBytes;
    const uint32_t stat = 3584u;                                    // static shared memory of the kernel, rounded up
    const uint32_t budget = 227u * 1024u / 3u - 1024u - stat;      // 3 CTAs per SM: - 1 KB reserved each
    auto shape = [&](uint32_t n_pass, bool force, SlotGeo* out) -> bool {
        SlotGeo sg;
        sg.n_pass = n_pass;
        sg.seg_len = (((g.n_time + n_pass - 1u) / n_pass) + 7u) & ~7u;
        const uint32_t dir_bytes = ((sg.seg_len >> 3) + 2u + 15u) & ~15u;
        sg.pool_off = kHdrBytes + dir_bytes;
        const double mb = mean_blocks / n_pass + (n_pass > 1 ? 1.0 : 0.0), ms = mean_surv / n_pass;
        sg.scap = (((uint32_t)(ms * 1.5) + 12u) + 3u) & ~3u;
        uint32_t want = (uint32_t)(mb * 1.5) + 24u;                // blocks incl. the zero block
        if (want > 255u) want = 255u;
        const uint32_t per_slot_fixed = sg.pool_off + 4u * sg.scap;
        if (fixed + kPSlots * (per_slot_fixed + 16u * 8u) > budget) return false;
        const uint32_t fit = ((budget - fixed) / kPSlots - per_slot_fixed) / 16u;
        sg.pcap = want < fit ? want : fit;
        if (!force && (double)sg.pcap < mb * 1.2 + 8.0) return false;   // too many lines would overflow the pool
        *out = sg;
        return true;
    };
    // Passes: 1 when the mean line fits the pool, else the fewest that do (each pass costs a partly used chunk and a
    // partly filled survivor / peak batch per line, so fewer is better).
    SlotGeo sg;
    bool have = false;
    for (uint32_t np = 1; np <= 6 && !have; ++np) {
        if (tun.passes && (int)np != tun.passes) continue;
        if (np > 1 && g.n_time < 64u * np) break;
        have = shape(np, false, &sg);
    }
    if (!have) {
        if (!must) return 0;
        if (tun.passes >= 1 && tun.passes <= 8 && g.n_time >= 64u * (uint32_t)tun.passes) have = shape((uint32_t)tun.passes, true, &sg);
        for (uint32_t np = 1; np <= 8 && !have; ++np) have = (np == 1 || g.n_time >= 64u * np) && shape(np, true, &sg);
        if (!have) return 0;
    }
    if (tun.block_pool >= 2 && tun.block_pool <= 255 && (uint32_t)tun.block_pool <= sg.pcap) sg.pcap = (uint32_t)tun.block_pool;
    if (tun.surv_cap >= 4 && (uint32_t)tun.surv_cap <= sg.scap) sg.scap = (uint32_t)tun.surv_cap & ~3u;
    sg.surv_off = sg.pool_off + 16u * sg.pcap;
    sg.slot_bytes = sg.surv_off + 4u * sg.scap;
    const uint32_t smem = kPSlots * sg.slot_bytes + fixed;

    // Pads per CTA: a CTA builds its pad range plus a halo of 4 lines and pays a fixed prologue (~2 lines' worth), and
    // the grid runs in waves of 148 x (CTAs per SM) CTAs: take the range that minimises waves x (range + 6).  A full
    // frame gets whole planes; a single sector is cut so that the last wave is not nearly empty.
    const uint32_t whole = (g.max_pads + kPS - 1) / kPS * kPS;
    const uint32_t resident = 148u * (uint32_t)std::max(1, std::min(4, (int)(227u * 1024u / (smem + 1024u + stat))));
    uint32_t pads_per_unit = whole;
    {
        uint64_t best = ~0ull;
        for (uint32_t u = 3 * kPS; u <= whole; u += kPS) {
            const uint64_t units = (uint64_t)g.n_planes * ((g.max_pads + u - 1) / u);
            const uint64_t cost = ((units + resident - 1) / resident) * (u + 6);
            if (cost <= best) { best = cost; pads_per_unit = u; }     // ties: the larger range (less halo)
        }
    }
    if (tun.pads_per_unit >= kPS && tun.pads_per_unit <= 256) pads_per_unit = (uint32_t)(tun.pads_per_unit / kPS * kPS);
    const uint32_t upp = (g.max_pads + pads_per_unit - 1) / pads_per_unit;
    if (ev_k0) cudaEventRecord(ev_k0, st);
    g_last_kernel = "k_fused_pairs";
    const bool m = sg.n_pass > 1, v = var.active != 0u;
    auto kern = m ? (v ? k_fused_pairs<true, true> : k_fused_pairs<true, false>)
                  : (v ? k_fused_pairs<false, true> : k_fused_pairs<false, false>);
    kern<<<g.n_planes * upp, kPThreads, smem, st>>>((const uint2*)digits, (uint32_t)n, g, ws.line_start,
                                                    pads_per_unit, upp, sg, q_peak_min, q_gate, var,
                                                    ws.counters, ws.line_cnt, (uint4*)ws.stage);
    if (ev_k1) cudaEventRecord(ev_k1, st);
    return 1;
}

}  // namespace tpccf
