/*
 * tpc_ec.h — C ABI of the B200-native entropy coder for the TPC cluster stream (product boundary; SURVEY.md §8(f)
 * NEXT #2).
 *
 * Operation: the last step of the paper's TPC compression chain, "common ANS compression", done there
 * with "a custom rANS library for entropy encoding" (Tables 1/2 list TPC rANS encoding / decoding,
 * PAPER.md:76, 89).  The paper gives no format, alphabet or table layout, and its step in between (track-model
 * residuals) needs tracking, which is out of scope — so the coded stream here is the cluster finder's own output and
 * the format, "TPC-EC v1", is this library's definition:
 *
 *   (Q) 13 byte streams, one symbol per cluster each ("same" = the previous cluster lies in the same (sector,row)):
 *        0 DPAD  same ? pad - prev.pad : pad          1,2 T_LO,T_HI  v = (same && pad == prev.pad) ? time - prev.time : time
 *        3,4 QMAX_LO,QMAX_HI     5..7 DQ0..2  (qtot - qmax) mod 2^24      8 FLAGS
 *        9 PM  clamp(rintf((pad_mean - (float)pad + 2.0f) * 64.0f), 0, 255)    10 TM  the same with time
 *        11 SP clamp(rintf(sigma_pad * 128.0f), 0, 255)                        12 ST  the same with sigma_time
 *       fp32, round-half-even, NaN -> 0.  Lossy for the four floats only; the decoder returns
 *       pad + (PM - 128) / 64, time + (TM - 128) / 64, SP / 128, ST / 128 (exact in fp32).
 *   (N) per stream a histogram over all n symbols, normalised to 12-bit frequencies (sum 4096):
 *       f = max(1, floor(c * 4096 / n)) for c > 0; a surplus goes to the symbol with the largest count (lowest on
 *       ties); a deficit is taken from the symbol with the largest f (lowest on ties), down to 1, repeatedly.
 *   (C) blocks of 16384 symbols, 32 lanes per block; lane l codes the symbols at block positions l, l + 32, ... with
 *       its own rANS state (32-bit, L = 2^23, byte-wise renormalisation), backwards; the lane record is the final
 *       state and the emitted bytes; the decoder runs forwards and must end at x == L with every byte consumed.
 *   (F) container: 64-byte header (magic "TPCE", version 1, n, n_sectors, n_rows, 13, 16384, n_blocks, total bytes),
 *       u32 clusters per plane, u16 freq[13][256], padding to 8, u64 record offsets[13 * n_blocks + 1], then the
 *       records (stream-major): u32 state[32], u16 nbytes[32], lane bytes, zero padding to 4.
 *
 * The encoder's output is bit-identical to the oracle's (oracle/tpc_ec_oracle.c, written from the same text and
 * sharing no code with this library); decode(encode(c)) returns c with the floats quantised as stated.
 *
 * All pointers are DEVICE pointers unless marked HOST; the caller owns every buffer; nothing synchronises the host.
 */
#ifndef TPC_EC_H
#define TPC_EC_H

#include <stddef.h>
#include <stdint.h>

#include "tpc_cf.h"   /* tpc_cluster, TPC_CF_E_* error codes */

#ifdef __cplusplus
extern "C" {
#endif

enum {
    TPC_EC_ERR_UNSORTED = 1u,   /* encode: keys not strictly ascending, or a sector / row outside the geometry;
                                   the container content is then unspecified */
    TPC_EC_ERR_CAPACITY = 2u,   /* encode: container larger than out_capacity (status.bytes holds the size needed, only
                                   header, tables and directory are written); decode: n > capacity */
    TPC_EC_ERR_CONTAINER = 4u,  /* decode: malformed container (header, table sums, offsets, a lane that does not end
                                   at x == L with all bytes consumed, plane counts) */
    TPC_EC_ERR_QTOT = 8u        /* encode: a cluster with qtot < qmax or qtot - qmax >= 2^24 (coded modulo 2^24) */
};

/* Written last on the stream, by the device. */
typedef struct {
    uint64_t n_clusters;   /* clusters coded / decoded */
    uint64_t bytes;        /* encode: container size; decode: bytes consumed (= the header's total) */
    uint32_t error;        /* TPC_EC_ERR_* bits, 0 = success */
    uint32_t rsv;
} tpc_ec_status;

typedef struct tpc_ec tpc_ec;   /* opaque handle: host state only */

/* Bytes of DEVICE workspace for up to max_clusters clusters: 13 symbol streams, histograms, coding tables, lane byte
 * counts and record sizes, decoding tables, plane starts.  0 on invalid arguments. */
size_t tpc_ec_workspace_bytes(uint32_t n_sectors, uint32_t n_rows, uint64_t max_clusters);

/* Upper bound of the container size for n clusters (12 bits per symbol plus the fixed parts). */
uint64_t tpc_ec_max_encoded_bytes(uint32_t n_sectors, uint32_t n_rows, uint64_t n);

/* workspace: DEVICE, 256-byte aligned, >= tpc_ec_workspace_bytes.  n_sectors, n_rows <= 256, max_clusters < 2^32.
 * Returns TPC_CF_OK or a negative TPC_CF_E_* code (E_NULL, E_GEOMETRY, E_CAPACITY, E_WORKSPACE, E_NOMEM). */
int tpc_ec_create(tpc_ec** h, uint32_t n_sectors, uint32_t n_rows, uint64_t max_clusters,
                  void* workspace, size_t workspace_bytes);

/* Enqueues the encoder on `stream` (cudaStream_t): clusters (32-byte records, strictly ascending keys, e.g. the output
 * of tpc_cf_run) -> container in `out` (16-byte aligned).  out_capacity must hold at least the fixed part (header,
 * plane counts, tables, directory; TPC_CF_E_CAPACITY otherwise); the payload is checked on the device.
 * status is written last.  Synchronous errors: negative return, nothing enqueued. */
int tpc_ec_encode(tpc_ec* h, const tpc_cluster* clusters, uint64_t n, uint8_t* out, uint64_t out_capacity,
                  tpc_ec_status* status, void* stream);

/* Enqueues the decoder: container `in` (16-byte aligned, in_bytes long) holding n clusters (the caller knows n from
 * the encoder's status; it is checked against the header on the device) -> clusters[0..n).  Every read is bounded
 * by in_bytes and every write by capacity; a malformed container sets TPC_EC_ERR_CONTAINER and leaves the output
 * unspecified. */
int tpc_ec_decode(tpc_ec* h, const uint8_t* in, uint64_t in_bytes, uint64_t n, tpc_cluster* clusters,
                  uint64_t capacity, tpc_ec_status* status, void* stream);

/* Kernel launches enqueued by the last encode / decode call (bench.py's gpu_launches). */
int tpc_ec_last_launch_count(const tpc_ec* h);

int tpc_ec_destroy(tpc_ec* h);

#ifdef __cplusplus
}
#endif
#endif /* TPC_EC_H */
