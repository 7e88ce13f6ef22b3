/*
 * tpc_cf_oracle.h — CPU ORACLE of the TPC cluster finder.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, link, import or call anything in oracle/.  The product path (paper_2402_01205_b200/)
 * shares no code, header, table or helper with this directory: the record layouts below are
 * restated here on purpose (same bytes as include/tpc_cf.h, independent text).
 *
 * What it computes: the step the paper names "cluster finding in the GPUs on the EPNs"
 * (§5), on one 2.8 ms time frame.  The paper gives no algorithm;
 * the definition is BASELINE.json:north_star as made unambiguous in SURVEY.md §8(c)
 * (readings R1..R19, restated in DESIGN.md §3).  The oracle is that definition executed
 * literally, one (sector,row) plane at a time, single-threaded, sums in int64, moments in double.
 *
 * Parity pins (tests/test_oracle_*.py): hand-evaluated grids under tests/golden/ (worked_examples.txt E1..E15,
 * variant_examples.txt V1..V10, sharing_examples.txt S1..S7), brute-force sparse-dict checker (tests/brute.py),
 * numpy argmax / box-filter special cases, closed-form moments, invariants.
 * No function in this file is "parity unpinned".
 */
#ifndef TPC_CF_ORACLE_H
#define TPC_CF_ORACLE_H

#include <stdint.h>
#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* 8-byte input record: one zero-suppressed ADC sample (BASELINE.json:north_star "digits
 * (sector, pad row, pad, time bin, charge)").  Little-endian, naturally aligned. */
typedef struct {
    uint8_t  sector, row, pad, rsv;
    uint16_t time, charge;
} orc_digit;

/* 32-byte output record: one cluster (north_star: "qTot, qMax, pad and time centroids and sigmas").
 * (sector,row,pad,time) is the peak cell; flags: V1 below (0 unless requested); rsv is 0. */
typedef struct {
    uint8_t  sector, row, pad, flags;
    uint16_t time, qmax;
    uint32_t qtot;
    float    pad_mean, time_mean, sigma_pad, sigma_time;
    uint32_t rsv;
} orc_cluster;

typedef struct {
    uint32_t n_sectors, n_rows, max_pads, n_time;
    const uint16_t* npads;      /* host, n_rows entries; NULL => every row has max_pads pads */
} orc_geometry;

/* Cluster-finder variants ("different cuts" in PAPER.md:21 — the paper names none,
 * the definitions are this repository's, DESIGN.md §3 V1..V4).  Peaks are found exactly as before; then
 *   V1 flags (written iff ORC_CLUSTER_FLAGS, else 0), from the peak cell and the sums of the accepted cells:
 *        1 EDGE_PAD     pad < 2 or pad + 2 >= npads[row]      (the 5x5 window is clipped by the plane in pad)
 *        2 EDGE_TIME    time < 2 or time + 2 >= n_time
 *        4 SINGLE_PAD   no charge outside the peak's pad line entered qTot   (sum c*dp*dp == 0)
 *        8 SINGLE_TIME  no charge outside the peak's time bin entered qTot   (sum c*dt*dt == 0)
 *       16 SATURATED    q_saturation != 0 and qMax >= q_saturation
 *   V2 cuts: a peak whose cluster has qTot < q_tot_min, or is SINGLE_PAD / SINGLE_TIME while the matching
 *        ORC_CUT_* bit is set, yields no cluster and is not counted in n_clusters.
 *   V3 a cut never changes which cells are peaks.
 *   V4 charge sharing between overlapping clusters (ORC_SHARE_CHARGE), in place of the double counting of R5.  The
 *        clusters of the run are found, cut and flagged exactly as above, on the unshared sums.  Let A(x) = qMax of
 *        the cluster whose peak is cell x (0 if x is no cluster's peak) and D(x) = sum of A over the 5x5 cells around
 *        x in the same plane = the summed peak charges of the clusters whose window contains x.  For the cluster with
 *        peak z, every cell x that enters its sums (R3 / R4 unchanged, decided on the raw charges) enters with
 *            c'(x) = floor(64 * Q(x) * A(z) / D(x))
 *        in place of Q(x): its charge in units of 1/64 ADC count, split among the windows that contain it in proportion
 *        to their peak charges (a window that contains x but gates it out keeps its share: that part is dropped).
 *        From the sums S' over c': qtot = floor((S0' + 32) / 64); centroids and sigmas by the same formulas on S'
 *        (S0' = 0, possible only if every share rounds to 0: the peak's position, sigmas 0).  sector..time, qmax and
 *        flags 1..16 are those of the unshared cluster; flag 32 SHARED iff D(x) != A(z) for some cell x with charge
 *        that entered.  A cluster no other window touches comes out bit-identical to the unshared run. */
enum { ORC_CLUSTER_FLAGS = 4u, ORC_CUT_SINGLE_PAD = 8u, ORC_CUT_SINGLE_TIME = 16u, ORC_SHARE_CHARGE = 32u };
enum { ORC_F_EDGE_PAD = 1, ORC_F_EDGE_TIME = 2, ORC_F_SINGLE_PAD = 4, ORC_F_SINGLE_TIME = 8, ORC_F_SATURATED = 16,
       ORC_F_SHARED = 32 };

typedef struct {
    uint16_t q_peak_min;        /* R6: peak threshold, default 4 */
    uint16_t q_inner_gate;      /* R4: gate threshold on the inner cell, default 2 */
    uint32_t flags;             /* ORC_* bits above; every other bit is ignored by the oracle */
    uint32_t q_tot_min;         /* V2: minimum qTot, 0 = no cut */
    uint16_t q_saturation;      /* V1: saturation threshold for the SATURATED flag, 0 = never */
    uint16_t rsv;
} orc_params;

typedef struct {
    uint64_t n_clusters;        /* true number of clusters (peaks that pass the cuts), even if > capacity */
    uint64_t n_digits_used;
    uint64_t n_bad_digits;      /* R11: out-of-range or zero-charge digits, skipped */
    uint32_t overflow;          /* 1 if n_clusters > capacity */
    uint32_t rsv;
} orc_status;

/* Runs the definition over all digits (any order).  All pointers are HOST pointers.
 * Writes at most `capacity` clusters, ascending (sector,row,pad,time); returns 0, or
 * -1 on a NULL/invalid argument, -2 on allocation failure, -3 if a moment sum reaches 2^24
 * (cannot happen for uint16 charges; asserted per SURVEY.md §8(c)-P5). */
int tpc_cf_oracle_run(const orc_digit* digits, uint64_t n,
                      const orc_geometry* geom, const orc_params* params,
                      orc_cluster* out, uint64_t capacity, orc_status* status);

/* Same, restricted to planes [plane_begin, plane_end) with plane = sector*n_rows + row.
 * Used by bench.py's cpu_baseline to time a bounded sample of a large frame. */
int tpc_cf_oracle_run_planes(const orc_digit* digits, uint64_t n,
                             const orc_geometry* geom, const orc_params* params,
                             uint32_t plane_begin, uint32_t plane_end,
                             orc_cluster* out, uint64_t capacity, orc_status* status);

/* Fills dense[npads*n_time] (pad-major, time-minor) with the charge map of one plane, the
 * way step "Q[d.pad][d.time] = d.charge" of the definition builds it.  For map-parity tests. */
int tpc_cf_oracle_dense_plane(const orc_digit* digits, uint64_t n,
                              const orc_geometry* geom, uint32_t sector, uint32_t row,
                              uint16_t* dense);

#ifdef __cplusplus
}
#endif
#endif
