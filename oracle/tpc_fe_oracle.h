/*
 * tpc_fe_oracle.h — CPU ORACLE of the TPC front-end filter.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.  It shares no
 * code, header, table or constant generator with the CUDA path (paper_2402_01205_b200/csrc/tpc_fe.cu); record and
 * array layouts are restated here on purpose.
 *
 * What it computes.  The paper: "The TPC chain for data compression consists of
 * zero-suppression after common-mode correction and ion tail cancellation in the FPGAs in the FLPs and cluster finding
 * in the GPUs".  The paper gives no algorithm, coefficient or number format for these three steps, so the
 * filter below ("TPC-FE v1") is this repository's definition: integer fixed point, executed literally.
 *
 * TPC-FE v1
 * ---------
 * Geometry: n_sectors, n_rows, max_pads, n_time, npads[row] (NULL: every row has max_pads pads).  W = max_pads rounded
 * up to a multiple of 8.  plane = sector * n_rows + row;  P = npads[row];  T = n_time.
 * Inputs: raw[plane][t][w] (uint16, time-major: index (plane * T + t) * W + w; entries w >= P are ignored) and
 * ped4[plane][w] (uint16, pedestal in quarter ADC counts).
 * Parameters: zs_threshold >= 1 (ADC), cm_quiet4 <= 4095 (quarter ADC), cm_min_pads >= 1, it_decay_shift k in 1..15,
 * it_kappa_shift j in k..14 or 0 (no ion-tail cancellation).
 *
 * Per plane, one state S[p] per pad, S = 0 before the first time bin.  For t = 0, 1, .. T-1:
 *   (P)  x[p] = 4 raw[t][p] - ped4[p]                                   (p < P)
 *   (CM) Q = { p < P : |x[p]| <= cm_quiet4 },  n = |Q|,  s = sum_{p in Q} x[p]
 *        cm = n >= cm_min_pads ? floor((2 s + n) / (2 n)) : 0            (the mean over Q, rounded half up)
 *   for every p < P:
 *   (IT) z = x[p] - cm + floor(S[p] / 4096)
 *   (ZS) q = min(floor((z + 2) / 4), 65535);  kept iff q >= zs_threshold
 *        S[p] = S[p] - floor(S[p] / 2^k) + (kept and j != 0 ? q * 2^(14 - j) : 0)
 * Output: a tpc_digit {sector,row,pad,rsv=0,time,charge=q} per kept sample, ascending (sector,row,pad,time).
 * (S stays in [0, 2^30): S >= 0 since only q >= 1 is ever added, and S < 65535 * 2^(14-j) * 2^k + 2^k <= 2^30.)
 *
 * Pins (tests/test_fe_oracle_pins.py): hand-evaluated example (tests/golden/fe_examples.txt), identity on generated
 * digits (raw = pedestal + charge + a common shift per time bin  =>  the digits come back), the library special case
 * without CM and IT (one numpy expression), the exact geometric decay of an isolated impulse, an independent Python
 * implementation (tests/fe_brute.py) on random small inputs, and invariants.
 */
#ifndef TPC_FE_ORACLE_H
#define TPC_FE_ORACLE_H

#include <stdint.h>

typedef struct { uint8_t sector, row, pad, rsv; uint16_t time, charge; } tpc_fe_oracle_digit;   /* 8 bytes */

typedef struct {
    uint32_t n_sectors, n_rows, max_pads, n_time;
    const uint16_t* npads;      /* n_rows entries or NULL */
} tpc_fe_oracle_geometry;

typedef struct {
    uint16_t zs_threshold, cm_quiet4, cm_min_pads;
    uint8_t it_decay_shift, it_kappa_shift;
} tpc_fe_oracle_params;

typedef struct { uint64_t n_digits; uint32_t overflow, rsv; } tpc_fe_oracle_status;

/* Planes [plane_begin, plane_end) of raw / ped4 (both indexed from plane 0 of the arrays passed in) -> out, at most
 * capacity records (status->n_digits is the true count, overflow = 2 if it exceeds capacity).  Returns 0, or -1 on a
 * NULL pointer, -2 on a bad geometry, -5 on a parameter outside its range, -7 if memory runs out. */
int tpc_fe_oracle_run(const uint16_t* raw, const uint16_t* ped4, const tpc_fe_oracle_geometry* g,
                      const tpc_fe_oracle_params* prm, uint32_t plane_begin, uint32_t plane_end,
                      tpc_fe_oracle_digit* out, uint64_t capacity, tpc_fe_oracle_status* status);

#endif
