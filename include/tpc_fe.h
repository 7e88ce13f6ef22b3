/*
 * tpc_fe.h — C ABI of the B200-native TPC front-end filter (product boundary).
 *
 * Operation: the step in front of the cluster finder in the paper's TPC chain, "zero-suppression after common-mode
 * correction and ion tail cancellation in the FPGAs in the FLPs" — restated as a CUDA pre-pass whose
 * output is exactly the cluster finder's input (sorted tpc_digit records, include/tpc_cf.h).  The paper gives no
 * algorithm, coefficient or number format for it, so the filter, "TPC-FE v1", is this library's definition.  It is
 * all-integer (fixed point, shifts instead of multipliers, as a front-end FPGA would do it), so that the result is
 * defined bit for bit:
 *
 *   Input, per (sector,row) plane pl = sector * n_rows + row, P = npads[row], T = n_time, W = tpc_fe_pad_stride():
 *     raw [pl][t][w]  uint16  ADC samples, TIME-MAJOR (all pads of one time bin are contiguous, as the samples
 *                             leave the detector link); entries w >= P are ignored
 *     ped4[pl][w]     uint16  pedestal of pad w in quarter ADC counts
 *   For t = 0 .. T-1 in this order, with one int32 state S[p] per pad (S = 0 before t = 0):
 *     (P)   x[p] = 4 * raw[t][p] - ped4[p]                                      quarter ADC, signed
 *     (CM)  quiet pads Q = { p < P : |x[p]| <= cm_quiet4 };  n = |Q|,  s = sum of x over Q;
 *           cm = (n >= cm_min_pads) ? floor((2 s + n) / (2 n)) : 0              mean over the quiet pads, half up
 *     (IT)  z = x[p] - cm + (S[p] >> 12)                                         the tail state is >= 0
 *     (ZS)  q = min(floor((z + 2) / 4), 65535);  the sample is kept iff q >= zs_threshold  (ADC, half up)
 *           S[p] <- S[p] - (S[p] >> it_decay_shift) + (kept and it_kappa_shift != 0 ? q << (14 - it_kappa_shift) : 0)
 *   Output: one tpc_digit (sector,row,pad,time,charge = q, rsv = 0) per kept sample, ascending (sector,row,pad,time).
 *
 *   The decay per bin is 1 - 2^-it_decay_shift, the tail amplitude 2^-it_kappa_shift of the kept charge; the
 *   restriction it_decay_shift <= it_kappa_shift keeps S < 2^30.  Only kept samples feed the tail.
 *
 * The result is bit-identical to the oracle's (oracle/tpc_fe_oracle.c, written from this text, sharing no code).
 * All pointers are DEVICE pointers unless marked HOST; the caller owns every buffer; nothing synchronises the host.
 */
#ifndef TPC_FE_H
#define TPC_FE_H

#include <stddef.h>
#include <stdint.h>

#include "tpc_cf.h"   /* tpc_digit, tpc_cf_geometry, TPC_CF_E_* error codes */

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    uint16_t zs_threshold;    /* ADC, >= 1; default 2 (BASELINE.json:configs "zero-suppressed <2 ADC") */
    uint16_t cm_quiet4;       /* quarter ADC, <= 4095; default 12 */
    uint16_t cm_min_pads;     /* >= 1; more than the row's pads switches the correction off for that row; default 8 */
    uint8_t  it_decay_shift;  /* 1..15; default 6 */
    uint8_t  it_kappa_shift;  /* it_decay_shift..14, or 0 = no ion-tail cancellation; default 8 */
} tpc_fe_params;

enum {
    TPC_FE_OVF_PLANE = 1u,    /* a plane's staging area overflowed: output incomplete.  The area of max_digits_per_plane
                                 records is cut into chunks of 32 records, shared evenly by the plane's groups of 32 pads
                                 (ceil(W / 32) of them); a pad line occupies whole chunks.  Size it for the densest
                                 group: 2x the expected digits per plane + 64 per pad is plenty; n_time + 32 per pad
                                 (pads rounded up to 32) can never overflow */
    TPC_FE_OVF_OUTPUT = 2u    /* more digits than `capacity`: only records below `capacity` are written */
};

/* Written last on the stream, by the device. */
typedef struct {
    uint64_t n_digits;        /* true number of kept samples, whatever the capacities */
    uint32_t overflow;        /* TPC_FE_OVF_* bits, 0 = the output is complete */
    uint32_t rsv;
} tpc_fe_status;

typedef struct tpc_fe tpc_fe;   /* opaque handle: host state only */

/* Row pitch of raw and ped4 in samples: max_pads rounded up to a multiple of 8 (16-byte rows). */
uint32_t tpc_fe_pad_stride(uint32_t max_pads);

/* Bytes of DEVICE workspace: per plane a staging area of max_digits_per_plane 4-byte records in chunks of 32 with a
 * 4-byte directory entry per chunk, per pad line a count, per plane 2 x 8 group counts and an offset.  0 on invalid
 * arguments. */
size_t tpc_fe_workspace_bytes(const tpc_cf_geometry* g, uint64_t max_digits_per_plane);

/* workspace: DEVICE, 256-byte aligned, >= tpc_fe_workspace_bytes.  Geometry limits as in tpc_cf.h.
 * Returns TPC_CF_OK or a negative TPC_CF_E_* code (E_NULL, E_GEOMETRY, E_CAPACITY, E_WORKSPACE, E_NOMEM). */
int tpc_fe_create(tpc_fe** h, const tpc_cf_geometry* g, uint64_t max_digits_per_plane,
                  void* workspace, size_t workspace_bytes);

/* Enqueues the filter on `stream` (cudaStream_t): raw, ped4 (16-byte aligned, layouts above) -> out[0 .. n_digits).
 * status is written last.  Synchronous errors (negative return, nothing enqueued): E_NULL, E_PARAMS (a parameter
 * outside the ranges above), E_CUDA. */
int tpc_fe_run(tpc_fe* h, const uint16_t* raw, const uint16_t* ped4, const tpc_fe_params* params,
               tpc_digit* out, uint64_t capacity, tpc_fe_status* status, void* stream);

/* Kernel launches enqueued by the last run (bench.py's gpu_launches). */
int tpc_fe_last_launch_count(const tpc_fe* h);

/* Profiling for bench.py's roofline: with on != 0 every run records two events around its dominant kernel
 * (k_fe_filter) on the run's stream.  tpc_fe_profile_ms waits for the last run's pair and returns the elapsed
 * milliseconds (a negative value if there is none). */
int tpc_fe_set_profiling(tpc_fe* h, int on);
float tpc_fe_profile_ms(tpc_fe* h);

int tpc_fe_destroy(tpc_fe* h);

#ifdef __cplusplus
}
#endif
#endif /* TPC_FE_H */
