// tpc_ec.cu — entropy coder for the TPC cluster stream ("TPC-EC v1", include/tpc_ec.h; step named in PAPER.md:55, 57).
// Product code, sm_100a.  Shares nothing with oracle/tpc_ec_oracle.c: the format text in the header is the only link.
//
// Encoder, on the caller's stream:
//   k_ec_symbolize   (Q) one thread per cluster: 13 symbol bytes (SoA streams in the workspace), order / range checks;
//                    the cluster that opens a plane records where the plane starts
//   k_ec_hist        (N) counts: per-thread private byte counters in shared memory (no atomics: the streams are skewed,
//                    and a shared-memory atomic costs 2 cycles per lane), folded every 240 symbols per thread
//   k_ec_normalize   (N) one CTA per stream: 12-bit frequencies -> container table and the coding table
//                    (reciprocal | f, shift, bias: the coder divides by multiplying)
//   k_ec_code        (C) one warp per (stream, block), one rANS state per lane; bytes collected in a 64-bit register and
//                    stored 8 at a time into the lane's worst-case slot of a scratch area (L2-resident)
//   k_ec_layout      exclusive scan of the record sizes -> directory; plane counts, header, status; capacity check
//   k_ec_pack        one CTA per record: lane slots -> record image in shared memory -> coalesced word stores
// Decoder:
//   k_ec_dec_tables  header check, table sums, slot -> (symbol, f, slot - cum) table (16 KB per stream), plane starts
//   k_ec_decode      one warp per (stream, block): 32 lanes decode forwards into the symbol streams
//   k_ec_rebuild     inverse of (Q): one warp per plane, pads by a warp scan, times by a segmented warp scan
#include <new>
#include <string.h>

#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/tpc_ec.h"

namespace tpcec {

static constexpr uint32_t kStreams = 13;
static constexpr uint32_t kBlock = 16384;          // symbols per block
static constexpr uint32_t kLanes = 32;
static constexpr uint32_t kPerLane = kBlock / kLanes;
static constexpr uint32_t kProbBits = 12, kProbScale = 1u << kProbBits;
static constexpr uint32_t kL = 1u << 23;
static constexpr uint32_t kRecFixed = kLanes * 4 + kLanes * 2;   // states + byte counts
static constexpr uint32_t kMagic = 0x45435054u;
// a lane codes at most 512 symbols at <= 12 bits (+ 2^-11 relative) each: <= 768 bytes; stores are whole 8-byte words
static constexpr uint32_t kSlot = 776;
static constexpr uint32_t kHistPerThread = 240;    // symbols per thread between two folds of the byte counters (< 256)
static constexpr uint32_t kHistRound = 256 * kHistPerThread;

struct Layout {                // byte offsets inside the container (all host-computable from n and the geometry)
    uint64_t off_counts, off_freq, off_dir, off_records;
    uint32_t n_blocks, n_planes;
};

static inline Layout layout_of(uint32_t n_sectors, uint32_t n_rows, uint64_t n)
{
    Layout l;
    l.n_planes = n_sectors * n_rows;
    l.n_blocks = (uint32_t)((n + kBlock - 1) / kBlock);
    l.off_counts = 64;
    l.off_freq = l.off_counts + 4ull * l.n_planes;
    l.off_dir = (l.off_freq + 2ull * 256 * kStreams + 7) & ~7ull;
    l.off_records = l.off_dir + 8ull * ((uint64_t)kStreams * l.n_blocks + 1);
    return l;
}

struct Ws {
    uint8_t* sym;          // [13][stride]
    uint64_t stride;
    uint32_t* hist;        // [13][256]
    uint2* ctab;           // [13][256]  coding table: reciprocal, f | shift << 13 | bias << 18
    uint32_t* dtab;        // [13][4096] decoding table: symbol | (f - 1) << 8 | (slot - cum) << 20
    uint16_t* lane_nb;     // [13 * max_blocks * 32]
    uint32_t* lane_x;      // [13 * max_blocks * 32] final states
    uint8_t* slots;        // [13 * max_blocks * 32][kSlot] lane bytes before packing
    uint32_t* rec_size;    // [13 * max_blocks]
    uint32_t* plane_start; // [planes + 1]
    uint32_t* flags;       // [4]: error bits, payload-fits flag
};

// ---- (Q) ----------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t quant(float v)
{
    return (uint32_t)fminf(fmaxf(rintf(v), 0.0f), 255.0f);      // NaN -> 0
}

__global__ void __launch_bounds__(256)
k_ec_symbolize(const uint4* __restrict__ cl, uint32_t n, uint32_t n_sectors, uint32_t n_rows, Ws ws)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    uint32_t err = 0u;
    const uint4 lo = __ldg(cl + 2 * (size_t)i), hi = __ldg(cl + 2 * (size_t)i + 1);
    const uint32_t sector = lo.x & 0xffu, row = (lo.x >> 8) & 0xffu, pad = (lo.x >> 16) & 0xffu, fl = lo.x >> 24;
    const uint32_t time = lo.y & 0xffffu, qmax = lo.y >> 16, qtot = lo.z;
    bool same = false;
    uint32_t ppad = 0u, ptime = 0u;
    if (sector >= n_sectors || row >= n_rows) err |= TPC_EC_ERR_UNSORTED;
    // plane_start[q] = index of the first cluster of a plane >= q: written by the cluster that opens plane p for every
    // q in (plane of its predecessor, p]; the last cluster closes the planes behind its own
    const uint32_t n_planes = n_sectors * n_rows;
    const uint32_t plane = sector * n_rows + row;
    uint32_t q_lo = 0u, q_hi = plane;                          // planes [q_lo, q_hi] start at i
    if (i > 0u) {
        const uint2 p = __ldg((const uint2*)(cl + 2 * (size_t)(i - 1)));
        const uint32_t ps = p.x & 0xffu, pr = (p.x >> 8) & 0xffu;
        ppad = (p.x >> 16) & 0xffu; ptime = p.y & 0xffffu;
        const uint64_t kp = ((uint64_t)ps << 32) | ((uint64_t)pr << 24) | ((uint64_t)ppad << 16) | ptime;
        const uint64_t kc = ((uint64_t)sector << 32) | ((uint64_t)row << 24) | ((uint64_t)pad << 16) | time;
        if (kp >= kc) err |= TPC_EC_ERR_UNSORTED;
        same = ps == sector && pr == row;
        q_lo = ps * n_rows + pr + 1u;
    }
    if (err == 0u) {                                           // (an unsorted or out-of-range stream: content unspecified)
        for (uint32_t q = q_lo; q <= q_hi; ++q) ws.plane_start[q] = i;
        if (i == n - 1u) for (uint32_t q = plane + 1u; q <= n_planes; ++q) ws.plane_start[q] = n;
    }
    const uint32_t dpad = same ? ((pad - ppad) & 0xffu) : pad;
    const uint32_t v = (same && pad == ppad) ? ((time - ptime) & 0xffffu) : time;
    const uint32_t dq = (qtot - qmax) & 0xffffffu;
    if (qtot < qmax || qtot - qmax >= (1u << 24)) err |= TPC_EC_ERR_QTOT;
    uint32_t sym[kStreams];
    sym[0] = dpad; sym[1] = v & 255u; sym[2] = v >> 8; sym[3] = qmax & 255u; sym[4] = qmax >> 8;
    sym[5] = dq & 255u; sym[6] = (dq >> 8) & 255u; sym[7] = dq >> 16; sym[8] = fl;
    // fp32, one rounding per operation (explicit intrinsics: no contraction)
    sym[9] = quant(__fmul_rn(__fadd_rn(__fsub_rn(__uint_as_float(lo.w), (float)pad), 2.0f), 64.0f));
    sym[10] = quant(__fmul_rn(__fadd_rn(__fsub_rn(__uint_as_float(hi.x), (float)time), 2.0f), 64.0f));
    sym[11] = quant(__fmul_rn(__uint_as_float(hi.y), 128.0f));
    sym[12] = quant(__fmul_rn(__uint_as_float(hi.z), 128.0f));
#pragma unroll
    for (uint32_t s = 0; s < kStreams; ++s) ws.sym[s * ws.stride + i] = (uint8_t)sym[s];     // 32 bytes per warp and stream
    if (err) atomicOr(&ws.flags[0], err);
}

// (N) counts.  grid = (chunks, 13); a CTA walks `rounds` rounds of kHistRound symbols of one stream.  Thread t keeps a
// private byte counter per symbol value: word = value * 64 + (warp >> 2) * 32 + lane, byte = warp & 3, so the 32 lanes
// of an access hit 32 banks.  After at most 240 symbols per thread the counters are folded into the CTA's histogram.
__global__ void __launch_bounds__(256)
k_ec_hist(uint32_t n, uint32_t rounds, Ws ws)
{
    extern __shared__ __align__(16) uint8_t s_cnt[];           // 256 values x 256 threads
    __shared__ uint32_t s_hist[256];
    const uint32_t t = threadIdx.x, lane = t & 31u, warp = t >> 5;
    const uint32_t s = blockIdx.y;
    for (uint32_t k = t; k < 256u * 256u / 16u; k += 256u) ((uint4*)s_cnt)[k] = make_uint4(0u, 0u, 0u, 0u);
    s_hist[t] = 0u;
    __syncthreads();
    const uint8_t* src = ws.sym + s * ws.stride;               // 256-byte aligned
    uint8_t* mine = s_cnt + 4u * ((warp >> 2) * 32u + lane) + (warp & 3u);
    uint32_t* words = (uint32_t*)s_cnt;
    for (uint32_t r = 0; r < rounds; ++r) {
        const uint64_t base = ((uint64_t)blockIdx.x * rounds + r) * kHistRound;
        if (base >= n) break;
#pragma unroll 3
        for (uint32_t j = 0; j < kHistPerThread / 16u; ++j) {
            const uint64_t at = base + ((uint64_t)j * 256u + t) * 16u;
            if (at >= n) break;
            const uint4 v = *(const uint4*)(src + at);
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
            if (n - at >= 16u) {
                // two symbols at a time: both counters are read before either is written (two loads in flight); equal
                // symbols both write "old + 2"
#pragma unroll
                for (uint32_t k = 0; k < 16u; k += 2u) {
                    uint8_t* pa = mine + 256u * ((w[k >> 2] >> (8u * (k & 3u))) & 255u);
                    uint8_t* pb = mine + 256u * ((w[k >> 2] >> (8u * (k & 3u) + 8u)) & 255u);
                    const uint32_t ca = *pa, cb = *pb;
                    const uint32_t both = pa == pb ? 1u : 0u;
                    *pa = (uint8_t)(ca + 1u + both);
                    *pb = (uint8_t)(cb + 1u + both);
                }
            } else {
                const uint32_t left = (uint32_t)(n - at);
                for (uint32_t k = 0; k < left; ++k) ++mine[256u * src[at + k]];
            }
        }
        __syncthreads();
        // fold: thread t sums the 64 words of value t (rotated start: conflict-free) and clears them
        uint32_t sum = 0u;
#pragma unroll 8
        for (uint32_t j = 0; j < 64u; ++j) {
            const uint32_t w = t * 64u + ((j + lane) & 63u);
            sum = __dp4a(words[w], 0x01010101u, sum);
            words[w] = 0u;
        }
        s_hist[t] += sum;
        __syncthreads();
    }
    if (s_hist[t]) atomicAdd(&ws.hist[s * 256 + t], s_hist[t]);
}

// ---- (N) one warp per stream; lane l owns the symbols 8l .. 8l + 7 ---------------------------------------------------
// first lane-symbol (lowest symbol) at which `v` is largest over the warp's 256 values
__device__ __forceinline__ uint32_t warp_argmax(const uint32_t (&v)[8], uint32_t lane)
{
    uint32_t best = v[0], at = lane * 8u;
#pragma unroll
    for (uint32_t j = 1; j < 8u; ++j) if (v[j] > best) { best = v[j]; at = lane * 8u + j; }
    const uint32_t top = __reduce_max_sync(0xffffffffu, best);
    return __reduce_min_sync(0xffffffffu, best == top ? at : 0xffffffffu);
}

__global__ void __launch_bounds__(32)
k_ec_normalize(uint32_t n, Ws ws, uint16_t* __restrict__ freq_out)
{
    const uint32_t s = blockIdx.x, lane = threadIdx.x;
    uint32_t c[8], f[8];
    uint32_t sum = 0u;
#pragma unroll
    for (uint32_t j = 0; j < 8u; ++j) {
        c[j] = ws.hist[s * 256 + lane * 8u + j];
        uint32_t q = 0u;
        if (n != 0u && c[j] != 0u) {
            q = (uint32_t)(((uint64_t)c[j] * kProbScale) / n);
            if (q < 1u) q = 1u;
        }
        f[j] = q;
        sum += q;
    }
    sum = __reduce_add_sync(0xffffffffu, sum);
    if (n != 0u) {
        int D = (int)kProbScale - (int)sum;                    // |D| <= 256 + 4096
        if (D > 0) {                                           // surplus to the symbol with the largest count
            const uint32_t a = warp_argmax(c, lane);
#pragma unroll
            for (uint32_t j = 0; j < 8u; ++j) if (lane * 8u + j == a) f[j] += (uint32_t)D;
        }
        while (D < 0) {                                        // deficit from the symbol with the largest f, down to 1
            const uint32_t a = warp_argmax(f, lane);
            uint32_t fa = 0u;
#pragma unroll
            for (uint32_t j = 0; j < 8u; ++j) if (lane * 8u + j == a) fa = f[j];
            fa = __shfl_sync(0xffffffffu, fa, a >> 3);
            const int d = -D < (int)fa - 1 ? -D : (int)fa - 1;
#pragma unroll
            for (uint32_t j = 0; j < 8u; ++j) if (lane * 8u + j == a) f[j] -= (uint32_t)d;
            D += d;
        }
    }
    uint32_t mine = 0u;
#pragma unroll
    for (uint32_t j = 0; j < 8u; ++j) mine += f[j];
    uint32_t incl = mine;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t u = __shfl_up_sync(0xffffffffu, incl, d);
        if ((int)lane >= d) incl += u;
    }
    uint32_t cum = incl - mine;
#pragma unroll
    for (uint32_t j = 0; j < 8u; ++j) {
        const uint32_t a = lane * 8u + j;
        freq_out[s * 256 + a] = (uint16_t)f[j];
        // x / f for x < 2^31 as umulhi(x, rcp) >> sh with rcp = ceil(2^(31 + ceil(log2 f)) / f), sh = ceil(log2 f) - 1
        // (exact for every x < 2^31); f == 1: rcp = 2^32 - 1 gives x - 1, made up for by a bias of M - 1
        const uint32_t fa = f[j];
        uint32_t rcp = 0u, sh = 0u, bias = 0u;
        if (fa == 1u) { rcp = 0xffffffffu; sh = 0u; bias = cum + kProbScale - 1u; }
        else if (fa > 1u) {
            const uint32_t lg = 32u - (uint32_t)__clz(fa - 1u);
            rcp = (uint32_t)((((uint64_t)1 << (31u + lg)) + fa - 1u) / fa);
            sh = lg - 1u;
            bias = cum;
        }
        ws.ctab[s * 256 + a] = make_uint2(rcp, fa | (sh << 13) | (bias << 18));
        cum += fa;
    }
}

// ---- (C) encoder -------------------------------------------------------------------------------------------------
// One coding step.  tab.x = reciprocal, tab.y = f | shift << 13 | bias << 18.  Zero, one or two bytes leave the state
// per symbol (x < 2^31, x_max >= 2^19), without a branch: they enter a 96-bit shift register (r0 lowest) from the top;
// `bits` of it are valid.  As soon as 64 bits are there, the oldest eight bytes are stored as one word.
struct Emit { uint32_t r0, r1, r2, bits, words; };

__device__ __forceinline__ void code_step(uint32_t& x, Emit& em, uint2* slot, const uint2 tab)
{
    const uint32_t f = tab.y & 0x1fffu;
    const uint32_t x_max = f << 19;                            // (L >> 12 << 8) * f <= 2^31
    const uint32_t sh = (x >> 8) >= x_max ? 16u : (x >= x_max ? 8u : 0u);
    em.r0 = __funnelshift_r(em.r0, em.r1, sh);
    em.r1 = __funnelshift_r(em.r1, em.r2, sh);
    em.r2 = __funnelshift_r(em.r2, x, sh);
    x >>= sh;
    em.bits += sh;
    if (em.bits >= 64u) {                                      // 64 or 72 valid bits: the oldest 64 start at bit 96 - bits
        const uint32_t off = 96u - em.bits;
        slot[em.words++] = make_uint2(__funnelshift_rc(em.r0, em.r1, off), __funnelshift_rc(em.r1, em.r2, off));
        em.bits -= 64u;
    }
    const uint32_t q = __umulhi(x, tab.x) >> ((tab.y >> 13) & 31u);
    x = x + (tab.y >> 18) + q * (kProbScale - f);              // = (x / f) * M + x % f + cum
}

__global__ void __launch_bounds__(256)
k_ec_code(uint32_t n, uint32_t n_blocks, Ws ws)
{
    __shared__ uint2 s_tab[256];
    const uint32_t s = blockIdx.y;
    s_tab[threadIdx.x] = ws.ctab[s * 256 + threadIdx.x];
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t b = blockIdx.x * (blockDim.x >> 5) + warp;
    if (b >= n_blocks) return;
    const uint32_t e = s * n_blocks + b;
    const uint32_t first = b * kBlock + lane;
    uint32_t m = 0u;
    if (first < n) {
        m = (n - first + kLanes - 1) / kLanes;
        if (m > kPerLane) m = kPerLane;
    }
    const uint8_t* src = ws.sym + s * ws.stride + first;
    uint2* const slot = (uint2*)(ws.slots + ((size_t)e * kLanes + lane) * kSlot);
    Emit em = {0u, 0u, 0u, 0u, 0u};
    uint32_t x = kL;
    uint32_t k = m;
    while (k & 7u) { --k; code_step(x, em, slot, s_tab[src[(size_t)k * kLanes]]); }
    // groups of eight symbols; the next group's bytes are fetched before the current group's dependent chain
    uint32_t nxt[8];
    if (k) {
#pragma unroll
        for (int j = 0; j < 8; ++j) nxt[j] = src[(size_t)(k - 8u + j) * kLanes];
    }
    while (k) {
        uint2 tab[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) tab[j] = s_tab[nxt[j]];
        k -= 8u;
        if (k) {
#pragma unroll
            for (int j = 0; j < 8; ++j) nxt[j] = src[(size_t)(k - 8u + j) * kLanes];
        }
#pragma unroll
        for (int j = 7; j >= 0; --j) code_step(x, em, slot, tab[j]);
    }
    const uint32_t nbytes = em.words * 8u + (em.bits >> 3);
    if (em.bits) {                                             // the last bits / 8 < 8 bytes sit at the top of r2:r1
        const uint64_t v = (((uint64_t)em.r2 << 32) | em.r1) >> (64u - em.bits);
        slot[em.words] = make_uint2((uint32_t)v, (uint32_t)(v >> 32));
    }
    ws.lane_x[(size_t)e * kLanes + lane] = x;
    ws.lane_nb[(size_t)e * kLanes + lane] = (uint16_t)nbytes;
    const uint32_t total = __reduce_add_sync(0xffffffffu, nbytes);
    if (lane == 0) ws.rec_size[e] = (kRecFixed + total + 3u) & ~3u;
}

// Record e: states, byte counts, the lanes' bytes back to back, zero padding to 4 — assembled in shared memory, stored
// as whole words.
__global__ void __launch_bounds__(256)
k_ec_pack(Ws ws, uint8_t* __restrict__ out, const uint64_t* __restrict__ rec_off)
{
    __shared__ __align__(16) uint8_t s_rec[kRecFixed + kLanes * 768 + 8];
    __shared__ uint32_t s_off[kLanes + 1];
    if (ws.flags[1] == 0u) return;                             // the payload does not fit: nothing beyond the directory
    const uint32_t e = blockIdx.x;
    const uint32_t t = threadIdx.x, lane = t & 31u, warp = t >> 5;
    if (warp == 0) {
        const uint32_t nb = ws.lane_nb[(size_t)e * kLanes + lane];
        uint32_t incl = nb;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t u = __shfl_up_sync(0xffffffffu, incl, d);
            if ((int)lane >= d) incl += u;
        }
        s_off[lane] = incl - nb;
        if (lane == 31) s_off[32] = incl;
        ((uint32_t*)s_rec)[lane] = ws.lane_x[(size_t)e * kLanes + lane];
        ((uint16_t*)(s_rec + kLanes * 4))[lane] = (uint16_t)nb;
    }
    __syncthreads();
    const uint32_t total = s_off[32];
    if (t < 4u) s_rec[kRecFixed + total + t] = 0;               // padding (the bytes beyond it are not stored)
    for (uint32_t l = warp; l < kLanes; l += 8u) {
        const uint32_t off = kRecFixed + s_off[l], nb = s_off[l + 1] - s_off[l];
        const uint32_t* from = (const uint32_t*)(ws.slots + ((size_t)e * kLanes + l) * kSlot);
        for (uint32_t j = lane; 4u * j < nb; j += 32u) {
            const uint32_t v = from[j];
#pragma unroll
            for (uint32_t k = 0; k < 4u; ++k)
                if (4u * j + k < nb) s_rec[off + 4u * j + k] = (uint8_t)(v >> (8u * k));
        }
    }
    __syncthreads();
    const uint32_t words = (kRecFixed + total + 3u) >> 2;
    uint32_t* to = (uint32_t*)(out + rec_off[e]);
    for (uint32_t j = t; j < words; j += 256u) to[j] = ((const uint32_t*)s_rec)[j];
}

// exclusive scan of the record sizes (one CTA; at most a few 10^4 entries) -> directory, header, status
__global__ void __launch_bounds__(1024)
k_ec_layout(uint32_t n, uint32_t n_sectors, uint32_t n_rows, Layout lay, Ws ws, uint8_t* __restrict__ out,
            uint64_t capacity, tpc_ec_status* __restrict__ status)
{
    __shared__ unsigned long long s_warp[32];
    __shared__ unsigned long long s_base;
    const uint32_t entries = kStreams * lay.n_blocks;
    uint64_t* dir = (uint64_t*)(out + lay.off_dir);
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_base = lay.off_records;
    __syncthreads();
    for (uint32_t c0 = 0; c0 < entries; c0 += 1024u) {
        const uint32_t i = c0 + threadIdx.x;
        const unsigned long long v = i < entries ? ws.rec_size[i] : 0ull;
        unsigned long long incl = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned long long t = __shfl_up_sync(0xffffffffu, incl, d);
            if ((int)lane >= d) incl += t;
        }
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            unsigned long long w = s_warp[lane], wi = w;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const unsigned long long t = __shfl_up_sync(0xffffffffu, wi, d);
                if ((int)lane >= d) wi += t;
            }
            s_warp[lane] = wi - w;                              // exclusive over warps
        }
        __syncthreads();
        const unsigned long long base = s_base;
        if (i < entries) dir[i] = base + s_warp[warp] + (incl - v);
        __syncthreads();
        if (threadIdx.x == 1023) s_base = base + s_warp[31] + incl;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const unsigned long long total = s_base;
        dir[entries] = total;
        uint32_t* h = (uint32_t*)out;
        h[0] = kMagic; h[1] = 1u; h[2] = n; h[3] = 0u; h[4] = n_sectors; h[5] = n_rows; h[6] = kStreams; h[7] = kBlock;
        h[8] = lay.n_blocks; h[9] = 0u; h[10] = (uint32_t)total; h[11] = (uint32_t)(total >> 32);
        h[12] = h[13] = h[14] = h[15] = 0u;
        const bool fits = total <= capacity;
        ws.flags[1] = fits ? 1u : 0u;
        status->n_clusters = n;
        status->bytes = total;
        status->error = ws.flags[0] | (fits ? 0u : TPC_EC_ERR_CAPACITY);
        status->rsv = 0u;
    }
    uint32_t* counts = (uint32_t*)(out + lay.off_counts);
    for (uint32_t p = threadIdx.x; p < lay.n_planes; p += 1024u)
        counts[p] = n ? ws.plane_start[p + 1] - ws.plane_start[p] : 0u;
    // zero padding between the tables and the directory
    for (uint64_t a = lay.off_freq + 2ull * 256 * kStreams + threadIdx.x; a < lay.off_dir; a += 1024u) out[a] = 0;
}

// ---- decoder -----------------------------------------------------------------------------------------------------
// grid = 13 + 1: CTA s < 13 checks table s and builds its slot -> symbol table; the last CTA checks the header and
// scans the plane counts.
__global__ void __launch_bounds__(256)
k_ec_dec_tables(const uint8_t* __restrict__ in, uint64_t in_bytes, uint32_t n, uint32_t n_sectors, uint32_t n_rows,
                Layout lay, Ws ws)
{
    __shared__ uint32_t s_f[256], s_c[257];
    __shared__ unsigned long long s_sum;
    if (blockIdx.x < kStreams) {
        const uint32_t s = blockIdx.x;
        const uint16_t* freq = (const uint16_t*)(in + lay.off_freq) + s * 256;
        s_f[threadIdx.x] = freq[threadIdx.x];
        __syncthreads();
        if (threadIdx.x < 32u) {                               // exclusive prefix sums: lane l owns 8 symbols
            const uint32_t lane = threadIdx.x;
            uint32_t mine = 0u;
#pragma unroll
            for (uint32_t j = 0; j < 8u; ++j) mine += s_f[lane * 8u + j];
            uint32_t incl = mine;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) {
                const uint32_t u = __shfl_up_sync(0xffffffffu, incl, d);
                if ((int)lane >= d) incl += u;
            }
            uint32_t cum = incl - mine;
#pragma unroll
            for (uint32_t j = 0; j < 8u; ++j) { s_c[lane * 8u + j] = cum; cum += s_f[lane * 8u + j]; }
            if (lane == 31u) {
                s_c[256] = cum;
                if (n != 0u && cum != kProbScale) atomicOr(&ws.flags[0], TPC_EC_ERR_CONTAINER);
            }
        }
        __syncthreads();
        const bool ok = s_c[256] == kProbScale;
        // slot -> symbol | (f - 1) << 8 | (slot - cum) << 20, the symbol found by bisection on the prefix sums; a table
        // that does not sum to 4096 decodes as "symbol 0, f = 1" everywhere (harmless: the error bit is already set)
        for (uint32_t slot = threadIdx.x; slot < kProbScale; slot += 256u) {
            uint32_t v = 0u;
            if (ok) {
                uint32_t a = 0u;                               // largest a with s_c[a] <= slot and f[a] > 0: the last one
#pragma unroll
                for (uint32_t step = 128u; step > 0u; step >>= 1) if (s_c[a + step] <= slot) a += step;
                v = a | ((s_f[a] - 1u) << 8) | ((slot - s_c[a]) << 20);
            }
            ws.dtab[s * kProbScale + slot] = v;
        }
        return;
    }
    // header
    if (threadIdx.x == 0) {
        const uint32_t* h = (const uint32_t*)in;
        const unsigned long long total = (unsigned long long)h[10] | ((unsigned long long)h[11] << 32);
        const bool ok = h[0] == kMagic && h[1] == 1u && h[2] == n && h[3] == 0u && h[4] == n_sectors && h[5] == n_rows &&
                        h[6] == kStreams && h[7] == kBlock && h[8] == lay.n_blocks && total == in_bytes;
        if (!ok) atomicOr(&ws.flags[0], TPC_EC_ERR_CONTAINER);
        s_sum = 0ull;
    }
    __syncthreads();
    // plane starts: exclusive scan of the plane counts, clamped to n so that no later write can leave the output
    const uint32_t* counts = (const uint32_t*)(in + lay.off_counts);
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    __shared__ unsigned long long s_w[8];
    for (uint32_t c0 = 0; c0 < lay.n_planes; c0 += 256u) {
        const uint32_t p = c0 + threadIdx.x;
        const unsigned long long v = p < lay.n_planes ? counts[p] : 0ull;
        unsigned long long incl = v;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const unsigned long long t = __shfl_up_sync(0xffffffffu, incl, d);
            if ((int)lane >= d) incl += t;
        }
        if (lane == 31) s_w[warp] = incl;
        __syncthreads();
        unsigned long long wbase = 0ull;
        for (uint32_t w = 0; w < warp; ++w) wbase += s_w[w];
        const unsigned long long base = s_sum;
        const unsigned long long excl = base + wbase + incl - v;
        if (p < lay.n_planes) ws.plane_start[p] = (uint32_t)(excl < n ? excl : n);
        __syncthreads();
        if (threadIdx.x == 255) s_sum = base + wbase + incl;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        ws.plane_start[lay.n_planes] = (uint32_t)(s_sum < n ? s_sum : n);
        if (s_sum != n) atomicOr(&ws.flags[0], TPC_EC_ERR_CONTAINER);
    }
}

__global__ void __launch_bounds__(256)
k_ec_decode(const uint8_t* __restrict__ in, uint64_t in_bytes, uint32_t n, Layout lay, Ws ws)
{
    __shared__ __align__(16) uint32_t s_tab[kProbScale];
    const uint32_t s = blockIdx.y;
    for (uint32_t k = threadIdx.x; k < kProbScale / 4; k += blockDim.x)
        ((uint4*)s_tab)[k] = ((const uint4*)(ws.dtab + s * kProbScale))[k];
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t b = blockIdx.x * (blockDim.x >> 5) + warp;
    if (b >= lay.n_blocks) return;
    const uint32_t e = s * lay.n_blocks + b;
    const uint64_t* dir = (const uint64_t*)(in + lay.off_dir);
    const uint64_t r0 = dir[e], r1 = dir[e + 1];
    bool bad = r0 < lay.off_records || r0 > r1 || r1 > in_bytes || r1 - r0 < kRecFixed || (r0 & 3u) != 0u;
    bad = __any_sync(0xffffffffu, bad);
    if (bad) { if (lane == 0) atomicOr(&ws.flags[0], TPC_EC_ERR_CONTAINER); return; }
    const uint8_t* rec = in + r0;
    uint32_t x = ((const uint32_t*)rec)[lane];
    const uint32_t nb = ((const uint16_t*)(rec + kLanes * 4))[lane];
    uint32_t incl = nb;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
        if ((int)lane >= d) incl += t;
    }
    const uint32_t total = __shfl_sync(0xffffffffu, incl, 31);
    if ((uint64_t)kRecFixed + total > r1 - r0) { if (lane == 0) atomicOr(&ws.flags[0], TPC_EC_ERR_CONTAINER); return; }
    // The lane's bytes are consumed from the last one down, through a 64-bit register that keeps the next bytes at its
    // top (`have` of them).  They are fetched as aligned 32-bit words, one word ahead of their use (in is 16-byte
    // aligned and in_bytes a multiple of 4, so a word never leaves the buffer; at most 2 bytes per symbol are consumed,
    // so even a malformed lane stays within 1 KB below its end, inside the fixed part).  A well-formed lane consumes
    // exactly its nb bytes — whatever lies below them in the register is never used — and ends at x == L.
    const uint64_t end = r0 + kRecFixed + incl;                 // offset one past the lane's last byte
    const uint32_t* wp = (const uint32_t*)(in + ((end - 1u) & ~(uint64_t)3));      // word holding that byte
    const uint32_t valid = (uint32_t)(end - ((end - 1u) & ~(uint64_t)3));           // its bytes below `end`: 1..4
    uint32_t b_hi = __ldg(wp) << (8u * (4u - valid));
    uint32_t b_lo = 0u;
    uint32_t have = valid;
    uint32_t ahead = __ldg(--wp);
    const uint32_t first = b * kBlock + lane;
    uint32_t m = 0u;
    if (first < n) {
        m = (n - first + kLanes - 1) / kLanes;
        if (m > kPerLane) m = kPerLane;
    }
    uint8_t* dst = ws.sym + s * ws.stride + first;
    uint32_t used = 0u;
    for (uint32_t k = 0; k < m; ++k) {
        if (have <= 4u) {                                       // room for a word: it goes right below the valid bytes
            const uint64_t w = (uint64_t)ahead << (32u - 8u * have);
            b_hi |= (uint32_t)(w >> 32);
            b_lo = (uint32_t)w;
            have += 4u;
            ahead = __ldg(--wp);
        }
        const uint32_t slot = x & (kProbScale - 1u);
        const uint32_t tab = s_tab[slot];
        dst[(size_t)k * kLanes] = (uint8_t)tab;
        x = (((tab >> 8) & 0xfffu) + 1u) * (x >> kProbBits) + (tab >> 20);
        const uint32_t sh = x < (kL >> 8) ? 16u : (x < kL ? 8u : 0u);          // bytes needed to reach x >= L
        x = __funnelshift_l(b_hi, x, sh);                       // (x << sh) | top sh bits of the register
        b_hi = __funnelshift_l(b_lo, b_hi, sh);
        b_lo <<= sh;
        have -= sh >> 3;
        used += sh >> 3;
    }
    if (x != kL || used != nb) atomicOr(&ws.flags[0], TPC_EC_ERR_CONTAINER);
}

// inverse of (Q): one warp per plane
__global__ void __launch_bounds__(256)
k_ec_rebuild(uint32_t n, uint32_t n_rows, uint32_t n_planes, uint64_t capacity, Ws ws, uint4* __restrict__ out)
{
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t plane = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (plane >= n_planes) return;
    const uint32_t beg = ws.plane_start[plane], end = ws.plane_start[plane + 1];
    const uint32_t w0 = (plane / n_rows) | ((plane % n_rows) << 8);
    uint32_t carry_pad = 0u, carry_time = 0u;
    for (uint32_t c0 = beg; c0 < end; c0 += 32u) {
        const uint32_t i = c0 + lane;
        const bool act = i < end;
        uint32_t sy[kStreams];
#pragma unroll
        for (uint32_t s = 0; s < kStreams; ++s) sy[s] = act ? ws.sym[s * ws.stride + i] : 0u;
        uint32_t pad = sy[0];
        uint32_t tv = sy[1] | (sy[2] << 8);
        bool head = act && (sy[0] != 0u || i == beg);          // starts a pad line: its time is absolute
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) {
            const uint32_t pu = __shfl_up_sync(0xffffffffu, pad, d);
            const uint32_t tu = __shfl_up_sync(0xffffffffu, tv, d);
            const bool hu = __shfl_up_sync(0xffffffffu, head, d);
            if ((int)lane >= d) {
                pad += pu;
                if (!head) { tv += tu; head = hu; }
            }
        }
        pad += carry_pad;
        if (!head) tv += carry_time;                            // no line start at or before this lane in the chunk
        carry_pad = __shfl_sync(0xffffffffu, pad, 31);
        carry_time = __shfl_sync(0xffffffffu, tv, 31);          // inactive tail lanes add 0 and start nothing
        if (act && i < capacity) {
            const uint32_t qmax = sy[3] | (sy[4] << 8);
            const uint32_t dq = sy[5] | (sy[6] << 8) | (sy[7] << 16);
            pad &= 0xffu; tv &= 0xffffu;
            uint4 lo, hi;
            lo.x = w0 | (pad << 16) | (sy[8] << 24);
            lo.y = tv | (qmax << 16);
            lo.z = qmax + dq;
            lo.w = __float_as_uint(__fadd_rn((float)pad, __fmul_rn((float)sy[9] - 128.0f, 0.015625f)));
            hi.x = __float_as_uint(__fadd_rn((float)tv, __fmul_rn((float)sy[10] - 128.0f, 0.015625f)));
            hi.y = __float_as_uint(__fmul_rn((float)sy[11], 0.0078125f));
            hi.z = __float_as_uint(__fmul_rn((float)sy[12], 0.0078125f));
            hi.w = 0u;
            out[2 * (size_t)i] = lo;
            out[2 * (size_t)i + 1] = hi;
        }
    }
}

__global__ void k_ec_dec_status(uint32_t n, uint64_t in_bytes, uint64_t capacity, Ws ws, tpc_ec_status* status)
{
    status->n_clusters = n;
    status->bytes = in_bytes;
    status->error = ws.flags[0] | (n > capacity ? TPC_EC_ERR_CAPACITY : 0u);
    status->rsv = 0u;
}

}  // namespace tpcec

using namespace tpcec;

struct tpc_ec {
    uint32_t n_sectors, n_rows;
    uint64_t max_clusters;
    Ws ws;
    uint32_t hist_ctas;    // CTAs of k_ec_hist that are resident at once
    int last_launches;
};

static inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

static size_t carve(uint32_t n_sectors, uint32_t n_rows, uint64_t max_clusters, char* base, Ws* ws)
{
    size_t off = 0;
    auto take = [&](size_t bytes) { char* p = base ? base + off : nullptr; off += align256(bytes ? bytes : 1); return p; };
    const uint64_t max_blocks = (max_clusters + kBlock - 1) / kBlock;
    Ws w;
    w.stride = align256(max_clusters ? max_clusters : 1);
    w.sym = (uint8_t*)take((size_t)kStreams * w.stride);
    w.hist = (uint32_t*)take(kStreams * 256 * 4);
    w.ctab = (uint2*)take(kStreams * 256 * 8);
    w.dtab = (uint32_t*)take((size_t)kStreams * kProbScale * 4);
    w.lane_nb = (uint16_t*)take((size_t)kStreams * max_blocks * kLanes * 2);
    w.lane_x = (uint32_t*)take((size_t)kStreams * max_blocks * kLanes * 4);
    w.slots = (uint8_t*)take((size_t)kStreams * max_blocks * kLanes * kSlot);
    w.rec_size = (uint32_t*)take((size_t)kStreams * max_blocks * 4);
    w.plane_start = (uint32_t*)take(((size_t)n_sectors * n_rows + 1) * 4);
    w.flags = (uint32_t*)take(16);
    if (ws) *ws = w;
    return off;
}

static bool geometry_ok(uint32_t n_sectors, uint32_t n_rows, uint64_t max_clusters)
{
    return n_sectors >= 1 && n_sectors <= 256 && n_rows >= 1 && n_rows <= 256 && max_clusters < (1ull << 32);
}

extern "C" size_t tpc_ec_workspace_bytes(uint32_t n_sectors, uint32_t n_rows, uint64_t max_clusters)
{
    if (!geometry_ok(n_sectors, n_rows, max_clusters)) return 0;
    return carve(n_sectors, n_rows, max_clusters, nullptr, nullptr);
}

extern "C" uint64_t tpc_ec_max_encoded_bytes(uint32_t n_sectors, uint32_t n_rows, uint64_t n)
{
    if (!geometry_ok(n_sectors, n_rows, n)) return 0;
    const Layout l = layout_of(n_sectors, n_rows, n);
    // per record: fixed part, < 4 bytes of padding, and per lane at most 12 bits per symbol plus 2 bytes of slack
    return l.off_records + (uint64_t)kStreams * l.n_blocks * (kRecFixed + 4 + 2 * kLanes) + kStreams * ((3 * n + 1) / 2);
}

extern "C" int tpc_ec_create(tpc_ec** h, uint32_t n_sectors, uint32_t n_rows, uint64_t max_clusters,
                             void* workspace, size_t workspace_bytes)
{
    if (!h || !workspace) return TPC_CF_E_NULL;
    if (n_sectors == 0 || n_sectors > 256 || n_rows == 0 || n_rows > 256) return TPC_CF_E_GEOMETRY;
    if (max_clusters >= (1ull << 32)) return TPC_CF_E_CAPACITY;
    if (((uintptr_t)workspace & 255u) != 0 || workspace_bytes < carve(n_sectors, n_rows, max_clusters, nullptr, nullptr))
        return TPC_CF_E_WORKSPACE;
    tpc_ec* e = new (std::nothrow) tpc_ec;
    if (!e) return TPC_CF_E_NOMEM;
    e->n_sectors = n_sectors; e->n_rows = n_rows; e->max_clusters = max_clusters; e->last_launches = 0;
    carve(n_sectors, n_rows, max_clusters, (char*)workspace, &e->ws);
    // k_ec_hist needs 64 KB of dynamic shared memory; without a device (host-only tests) the call fails harmlessly
    e->hist_ctas = 3 * 148;
    if (cudaFuncSetAttribute(k_ec_hist, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536) == cudaSuccess) {
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) == cudaSuccess &&
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
            e->hist_ctas = 3u * (uint32_t)sms;
    } else {
        cudaGetLastError();
    }
    *h = e;
    return TPC_CF_OK;
}

extern "C" int tpc_ec_encode(tpc_ec* h, const tpc_cluster* clusters, uint64_t n, uint8_t* out, uint64_t out_capacity,
                             tpc_ec_status* status, void* stream)
{
    if (!h || !out || !status || (n && !clusters)) return TPC_CF_E_NULL;
    if (n > h->max_clusters) return TPC_CF_E_CAPACITY;
    if (((uintptr_t)out & 15u) != 0 || ((uintptr_t)clusters & 15u) != 0) return TPC_CF_E_WORKSPACE;
    const Layout lay = layout_of(h->n_sectors, h->n_rows, n);
    if (out_capacity < lay.off_records) return TPC_CF_E_CAPACITY;
    cudaStream_t st = (cudaStream_t)stream;
    const Ws& ws = h->ws;
    const uint32_t n32 = (uint32_t)n;
    int launches = 0;
    cudaMemsetAsync(ws.hist, 0, kStreams * 256 * 4, st);
    cudaMemsetAsync(ws.flags, 0, 16, st);
    if (n32) {
        k_ec_symbolize<<<(n32 + 255) / 256, 256, 0, st>>>((const uint4*)clusters, n32, h->n_sectors, h->n_rows, ws);
        // rounds of kHistRound symbols, shared out so that the grid is about one wave of 3 CTAs per SM
        const uint32_t total_rounds = (n32 + kHistRound - 1) / kHistRound;
        const uint32_t per = (kStreams * total_rounds + h->hist_ctas - 1) / h->hist_ctas;
        const dim3 hgrid((total_rounds + per - 1) / per, kStreams);
        k_ec_hist<<<hgrid, 256, 65536, st>>>(n32, per, ws);
        launches += 2;
    }
    k_ec_normalize<<<kStreams, 32, 0, st>>>(n32, ws, (uint16_t*)(out + lay.off_freq));
    ++launches;
    if (lay.n_blocks) {
        k_ec_code<<<dim3((lay.n_blocks + 7) / 8, kStreams), 256, 0, st>>>(n32, lay.n_blocks, ws);
        ++launches;
    }
    k_ec_layout<<<1, 1024, 0, st>>>(n32, h->n_sectors, h->n_rows, lay, ws, out, out_capacity, status);
    ++launches;
    if (lay.n_blocks) {
        k_ec_pack<<<kStreams * lay.n_blocks, 256, 0, st>>>(ws, out, (const uint64_t*)(out + lay.off_dir));
        ++launches;
    }
    h->last_launches = launches;
    return cudaGetLastError() == cudaSuccess ? TPC_CF_OK : TPC_CF_E_CUDA;
}

extern "C" int tpc_ec_decode(tpc_ec* h, const uint8_t* in, uint64_t in_bytes, uint64_t n, tpc_cluster* clusters,
                             uint64_t capacity, tpc_ec_status* status, void* stream)
{
    if (!h || !in || !status || (n && !clusters)) return TPC_CF_E_NULL;
    if (n > h->max_clusters) return TPC_CF_E_CAPACITY;
    if (((uintptr_t)in & 15u) != 0 || ((uintptr_t)clusters & 15u) != 0) return TPC_CF_E_WORKSPACE;
    const Layout lay = layout_of(h->n_sectors, h->n_rows, n);
    if (in_bytes < lay.off_records || (in_bytes & 3u) != 0) return TPC_CF_E_CAPACITY;   // not even the fixed part / not whole words
    cudaStream_t st = (cudaStream_t)stream;
    const Ws& ws = h->ws;
    const uint32_t n32 = (uint32_t)n;
    int launches = 0;
    cudaMemsetAsync(ws.flags, 0, 16, st);
    k_ec_dec_tables<<<kStreams + 1, 256, 0, st>>>(in, in_bytes, n32, h->n_sectors, h->n_rows, lay, ws);
    ++launches;
    if (lay.n_blocks) {
        k_ec_decode<<<dim3((lay.n_blocks + 7) / 8, kStreams), 256, 0, st>>>(in, in_bytes, n32, lay, ws);
        k_ec_rebuild<<<(lay.n_planes + 7) / 8, 256, 0, st>>>(n32, h->n_rows, lay.n_planes, capacity, ws, (uint4*)clusters);
        launches += 2;
    }
    k_ec_dec_status<<<1, 1, 0, st>>>(n32, in_bytes, capacity, ws, status);
    ++launches;
    h->last_launches = launches;
    return cudaGetLastError() == cudaSuccess ? TPC_CF_OK : TPC_CF_E_CUDA;
}

extern "C" int tpc_ec_last_launch_count(const tpc_ec* h) { return h ? h->last_launches : TPC_CF_E_NULL; }

extern "C" int tpc_ec_destroy(tpc_ec* h)
{
    if (!h) return TPC_CF_E_NULL;
    delete h;
    return TPC_CF_OK;
}
