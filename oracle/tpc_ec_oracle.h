/*
 * tpc_ec_oracle.h — CPU ORACLE of the entropy coder for the TPC cluster stream.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.  It shares no
 * code, header, table or constant generator with the CUDA path (paper_2402_01205_b200/csrc/tpc_ec.cu); record and
 * container layouts are restated here on purpose.
 *
 * What it computes.  The paper: "Data compression for all detectors uses a custom rANS
 * library for entropy encoding"; the TPC chain ends in "common ANS compression" after the lossy steps
 * (PAPER.md:57); Tables 1/2 list "TPC rANS Encoding / Decoding".  The paper gives no format, alphabet
 * or table layout, and the step before it in the paper (track-model residuals) needs tracking, which is out of scope.
 * So the format below ("TPC-EC v1") is this repository's definition; the coder itself is the published range-variant
 * ANS (rANS: 32-bit state, 12-bit probabilities, byte-wise renormalisation), restated step by step.
 *
 * TPC-EC v1
 * ---------
 * Input: n clusters (32-byte tpc_cluster records) strictly ascending in (sector,row,pad,time), n_sectors, n_rows.
 * plane = sector * n_rows + row.  "same" below means: i > 0 and cluster i-1 lies in the same plane.
 *
 * (Q) Symbol streams.  13 streams of n bytes; symbol of cluster i:
 *    0 DPAD   same ? pad_i - pad_{i-1} : pad_i
 *    1 T_LO, 2 T_HI   low / high byte of v = (same and pad_i == pad_{i-1}) ? time_i - time_{i-1} : time_i
 *    3 QMAX_LO, 4 QMAX_HI
 *    5,6,7 DQ0..DQ2   bytes 0..2 of (qtot - qmax) mod 2^24   [qtot < qmax or a difference >= 2^24: error bit 8]
 *    8 FLAGS
 *    9 PM     clamp(rintf((pad_mean  - (float)pad  + 2.0f) * 64.0f), 0, 255)       fp32 arithmetic, round-half-even
 *   10 TM     clamp(rintf((time_mean - (float)time + 2.0f) * 64.0f), 0, 255)
 *   11 SP     clamp(rintf(sigma_pad  * 128.0f), 0, 255)
 *   12 ST     clamp(rintf(sigma_time * 128.0f), 0, 255)
 *   (clamp(v) = fminf(fmaxf(v, 0), 255), so NaN -> 0.)  This step is lossy for the four floats only.
 *   Inverse: pad_mean' = (float)pad + ((float)PM - 128.0f) / 64.0f, same for time; sigma' = (float)SP / 128.0f (all exact).
 *
 * (N) Statistics.  Per stream: hist[256] over all n symbols, normalised to freq[256] with sum 4096:
 *    f[s] = c[s] == 0 ? 0 : max(1, floor(c[s] * 4096 / n));  D = 4096 - sum f
 *    D > 0: f[a] += D, a = the symbol with the largest count (lowest symbol on ties)
 *    while D < 0: b = the symbol with the largest f (lowest on ties); d = min(-D, f[b] - 1); f[b] -= d; D += d
 *    cum[s] = sum_{j<s} f[j].     (n == 0: all zero.)
 *
 * (C) Coding.  A stream is cut into blocks of 16384 symbols; lane l (0..31) of block b owns the symbols at positions
 *    b*16384 + l + 32k (k = 0..511) that are < n: m of them.  Lane encoder (rANS, L = 2^23, M = 2^12):
 *       x = L;  for k = m-1 down to 0:  (f, c) = (freq, cum) of the symbol
 *           while x >= (L >> 12 << 8) * f:  emit byte x & 255;  x >>= 8
 *           x = (x / f) * 4096 + (x % f) + c
 *    Lane record = final x and the emitted bytes in emission order.  Lane decoder: x = final; ptr = nbytes;
 *       for k = 0..m-1:  slot = x & 4095; s = the symbol with cum[s] <= slot < cum[s] + f[s]; output s
 *           x = f * (x >> 12) + slot - c;  while x < L: x = (x << 8) | bytes[--ptr]
 *    and at the end x == L and ptr == 0.
 *
 * (F) Container (little-endian; every offset from the start of the buffer):
 *    0    u32 magic 0x45435054 ("TPCE"), u32 version 1, u64 n, u32 n_sectors, u32 n_rows, u32 n_streams 13,
 *         u32 block_syms 16384, u32 n_blocks = ceil(n / 16384), u32 0, u64 total_bytes, 16 zero bytes      (64 bytes)
 *    64   u32 plane_count[n_sectors * n_rows]            clusters per plane (sector and row are not coded per cluster)
 *    ..   u16 freq[13][256]
 *    ..   zero padding to a multiple of 8
 *    D    u64 rec_off[13 * n_blocks + 1]                 record (stream s, block b) is entry s * n_blocks + b; last = total_bytes
 *    ..   records in entry order: u32 state[32], u16 nbytes[32], lane 0 bytes, lane 1 bytes, ..., zero padding to a multiple of 4
 */
#ifndef TPC_EC_ORACLE_H
#define TPC_EC_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* restated 32-byte cluster record (same bytes as the product's tpc_cluster) */
typedef struct {
    uint8_t  sector, row, pad, flags;
    uint16_t time, qmax;
    uint32_t qtot;
    float    pad_mean, time_mean, sigma_pad, sigma_time;
    uint32_t rsv;
} tpc_ec_oracle_cluster;

enum {
    TPC_EC_ORACLE_ERR_UNSORTED = 1,   /* keys not strictly ascending, or sector / row outside the geometry */
    TPC_EC_ORACLE_ERR_CAPACITY = 2,   /* output buffer too small */
    TPC_EC_ORACLE_ERR_CONTAINER = 4,  /* decode: malformed container */
    TPC_EC_ORACLE_ERR_QTOT = 8        /* a cluster with qtot < qmax or qtot - qmax >= 2^24 (coded modulo 2^24) */
};

/* (Q): streams[s * n + i].  Returns error bits. */
uint32_t tpc_ec_oracle_symbolize(const tpc_ec_oracle_cluster* cl, uint64_t n, uint32_t n_sectors, uint32_t n_rows,
                                 uint8_t* streams);
/* (N) */
void tpc_ec_oracle_normalize(const uint64_t hist[256], uint16_t freq[256]);
/* (C) one lane: symbols sym[k * stride], k = 0..m-1.  bytes must hold 3 * m / 2 + 4.  Returns the final state. */
uint32_t tpc_ec_oracle_lane_encode(const uint8_t* sym, uint64_t m, uint64_t stride, const uint16_t freq[256],
                                   uint8_t* bytes, uint32_t* nbytes);
/* returns 0, or TPC_EC_ORACLE_ERR_CONTAINER if the lane does not end at x == L, ptr == 0 */
uint32_t tpc_ec_oracle_lane_decode(uint32_t state, const uint8_t* bytes, uint32_t nbytes, const uint16_t freq[256],
                                   uint8_t* sym, uint64_t m, uint64_t stride);

/* upper bound of the container size for n clusters */
uint64_t tpc_ec_oracle_max_bytes(uint32_t n_sectors, uint32_t n_rows, uint64_t n);
/* whole encoder: returns the container size (written only if <= capacity); *err receives error bits */
uint64_t tpc_ec_oracle_encode(const tpc_ec_oracle_cluster* cl, uint64_t n, uint32_t n_sectors, uint32_t n_rows,
                              uint8_t* out, uint64_t capacity, uint32_t* err);
/* whole decoder: returns error bits; *n receives the cluster count of the container */
uint32_t tpc_ec_oracle_decode(const uint8_t* in, uint64_t bytes, tpc_ec_oracle_cluster* out, uint64_t capacity,
                              uint64_t* n);

#ifdef __cplusplus
}
#endif
#endif
