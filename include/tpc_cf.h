/*
 * tpc_cf.h — C ABI of the B200-native TPC cluster finder (product boundary).
 *
 * Operation: the step the paper names "cluster finding in the GPUs on the EPNs" (§5), run on one
 * 2.8 ms time frame: zero-suppressed ADC digits (sector, pad row, pad, time bin, charge) ->
 * clusters (qTot, qMax, pad/time centroids and sigmas).  The paper gives no algorithm; the definition is
 * BASELINE.json:north_star, made unambiguous by the readings R1..R19 of SURVEY.md §8(c) (restated in DESIGN.md §3):
 *   peak      : q >= q_peak_min (4) and 3x3 (pad x time) local maximum, strict '>' against the 4 neighbours that
 *               are lexicographically earlier in (pad,time), '>=' against the 4 later ones               (R1, R6)
 *   qTot      : inner 3x3 always + each outer 5x5-ring cell (dp,dt) whose gate cell (dp-sgn dp, dt-sgn dt)
 *               holds >= q_inner_gate (2) ADC                                                            (R3, R4)
 *   moments   : charge-weighted mean / population sigma over exactly those cells, offsets taken relative to
 *               the peak (so the fp32 sums are exact integers < 2^24), zero border outside the plane   (R2, R7, R8)
 *   order     : one cluster per peak, ascending (sector,row,pad,time) of the peak cell                   (R10)
 *
 * All structs are POD, little-endian, naturally aligned.  No C++ or torch type crosses this boundary.
 * Pointers are marked HOST or DEVICE.  The library never allocates device memory: the caller (PyTorch in the
 * Python binding) owns digits, clusters, status and workspace.
 */
#ifndef TPC_CF_H
#define TPC_CF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* 8-byte input record (north_star: "digits (sector, pad row, pad, time bin, charge)"). */
typedef struct {
    uint8_t  sector, row, pad, rsv;   /* rsv is ignored */
    uint16_t time, charge;
} tpc_digit;

/* 32-byte output record (north_star: "clusters (qTot, qMax, pad and time centroids and sigmas)").
 * (sector,row,pad,time) is the peak cell; flags: TPC_CF_F_* bits if TPC_CF_CLUSTER_FLAGS was set, else 0; rsv = 0. */
typedef struct {
    uint8_t  sector, row, pad, flags;
    uint16_t time, qmax;
    uint32_t qtot;
    float    pad_mean, time_mean, sigma_pad, sigma_time;
    uint32_t rsv;
} tpc_cluster;

/* Detector geometry.  Limits (8/16-bit record fields): n_sectors <= 256, n_rows <= 256, max_pads <= 255,
 * n_time <= 65535.  npads: HOST pointer to n_rows entries (1..max_pads), or NULL => every row has max_pads
 * pads (R15, R19).  It is copied at create; it need not outlive the call. */
typedef struct {
    uint32_t n_sectors, n_rows, max_pads, n_time;
    const uint16_t* npads;
} tpc_cf_geometry;

enum {
    TPC_CF_DIGITS_SORTED = 1u,  /* promise: digits ascend in (sector,row,pad,time).  Selects the fused shared-memory
                                   path ("T3") and skips the key sort.  The promise is verified on the device for
                                   free; if it is false nothing is output and status.path = 0, n_clusters = 0
                                   (rerun without the flag; tpc_cf_run_host does that by itself).  A wrong result
                                   is never returned silently. */
    TPC_CF_FORCE_GENERAL = 2u,  /* always run the general (map in HBM, "T1") path, whatever the order.  Without this flag
                                   and without the promise above, the digits are sorted on the device into a workspace
                                   buffer and the fused path runs on the sorted copy (status.path = 2): same result
                                   array (R12), several times faster on unordered input */
    /* Cluster-finder variants.  The paper only says that "different cuts" are used in the
     * synchronous phase and names none; these definitions are this library's (DESIGN.md §3 V1..V4).
     * Peaks are always found by the same rule (R1): a cut never changes which cells are peaks (V3). */
    TPC_CF_CLUSTER_FLAGS = 4u,    /* V1: fill tpc_cluster.flags with the TPC_CF_F_* bits below (else the byte is 0) */
    TPC_CF_CUT_SINGLE_PAD = 8u,   /* V2: a SINGLE_PAD cluster is not output and not counted */
    TPC_CF_CUT_SINGLE_TIME = 16u, /* V2: same for SINGLE_TIME */
    TPC_CF_SHARE_CHARGE = 32u     /* V4: charge sharing between overlapping clusters in place of the double counting of R5.
                                     The clusters of the run are found, cut and flagged exactly as without this bit, on the
                                     unshared sums.  Let A(x) = qMax of the cluster whose peak is cell x (0 if none) and
                                     D(x) = sum of A over the 5x5 cells around x in the same plane (the summed peak charges
                                     of the clusters whose window holds x).  For the cluster with peak z every cell x that
                                     enters its sums (R3 / R4 unchanged, on raw charges) enters with
                                         c'(x) = floor(64 * Q(x) * A(z) / D(x))
                                     in place of Q(x): its charge in 1/64 ADC counts, split among the windows that hold it
                                     in proportion to their peak charges.  From the sums S' over c':
                                     qtot = floor((S0' + 32) / 64), centroids and sigmas by the same formulas (S0' = 0: the
                                     peak's position, sigmas 0).  sector..time, qmax and flags 1..16 stay those of the
                                     unshared cluster; a cluster no other window touches comes out bit-identical.
                                     Runs as a post-pass (K6) over the ordered output of whichever path produced it.
                                     With status.overflow = 1 the clusters written near the cut may miss neighbours that
                                     were not written: their shared values are unspecified. */
};

/* V1: bits of tpc_cluster.flags, from the peak cell and the cells that entered qTot. */
enum {
    TPC_CF_F_EDGE_PAD = 1u,     /* pad < 2 or pad + 2 >= npads[row]: the 5x5 window is clipped by the plane in pad */
    TPC_CF_F_EDGE_TIME = 2u,    /* time < 2 or time + 2 >= n_time */
    TPC_CF_F_SINGLE_PAD = 4u,   /* no charge outside the peak's pad line entered qTot (sigma_pad == 0) */
    TPC_CF_F_SINGLE_TIME = 8u,  /* no charge outside the peak's time bin entered qTot (sigma_time == 0) */
    TPC_CF_F_SATURATED = 16u,   /* q_saturation != 0 and qMax >= q_saturation */
    TPC_CF_F_SHARED = 32u       /* V4 only: some cell with charge that entered this cluster lies in another cluster's window
                                   too (its charge was split) */
};

typedef struct {
    uint16_t q_peak_min;    /* R6, default 4; 0 is rejected */
    uint16_t q_inner_gate;  /* R4, default 2 */
    uint32_t flags;         /* TPC_CF_* bits */
    uint32_t q_tot_min;     /* V2: clusters with qTot < q_tot_min are not output and not counted; 0 = no cut */
    uint16_t q_saturation;  /* V1: threshold of the SATURATED flag; 0 = never */
    uint16_t rsv;           /* 0 */
} tpc_cf_params;

/* Written last on the stream, by the device. */
typedef struct {
    uint64_t n_clusters;     /* true number of clusters (peaks that pass the cuts), even if > capacity */
    uint64_t n_digits_used;  /* valid digits */
    uint64_t n_bad_digits;   /* R11: out-of-range or zero-charge digits: skipped and counted */
    uint32_t overflow;       /* 1 if n_clusters > capacity: the first `capacity` clusters in output order are written.
                                Unsorted input is ordered by a key sort that holds at most the max_clusters given to
                                create: with more peaks than that, overflow = 1 too, and what is written are the first
                                max_clusters peaks in DIGIT order, sorted (A2) */
    uint32_t path;           /* 1 = general path (T1) produced the output, 3 = fused sorted path (T3), 2 = the digits were
                                sorted on the device and the fused path ran on the sorted copy (input without the
                                DIGITS_SORTED promise), 0 = no output: DIGITS_SORTED was promised but the digits are not
                                sorted, or (path 2) two digits address the same cell */
} tpc_cf_status;

typedef struct {
    tpc_cluster*   clusters;  /* DEVICE, caller-owned, `capacity` entries, 32-byte aligned */
    uint64_t       capacity;
    tpc_cf_status* status;    /* DEVICE, caller-owned, 8-byte aligned; valid after the stream is synchronised */
    void*          stream;    /* cudaStream_t (0 = legacy default stream) */
} tpc_cf_out;

typedef struct tpc_cf tpc_cf;   /* opaque handle: host state only */

enum {
    TPC_CF_OK = 0,
    TPC_CF_E_NULL = -1,       /* a required pointer is NULL */
    TPC_CF_E_GEOMETRY = -2,   /* zero or out-of-limit dimension, bad npads entry, or differs from create */
    TPC_CF_E_CAPACITY = -3,   /* n > max_digits */
    TPC_CF_E_WORKSPACE = -4,  /* workspace too small or not 256-byte aligned */
    TPC_CF_E_PARAMS = -5,     /* q_peak_min == 0 or unknown flag bits */
    TPC_CF_E_CUDA = -6,       /* a CUDA call failed; text via tpc_cf_strerror */
    TPC_CF_E_NOMEM = -7       /* host allocation failed */
};

/* Bytes of DEVICE workspace `create` needs for this geometry and these capacities (0 on invalid geometry).
 * Layout: dense uint16 charge map with a 2-cell zero border per plane (general path: 22.3 GB for the
 * full 36-sector geometry), peak mask, line index and counts, cluster staging (32 B per max_DIGITS: the cluster of a
 * peak is staged at its line's digit range, only peak slots are ever touched), and 56 B per max_clusters of
 * compaction + sort scratch for unsorted input. */
size_t tpc_cf_workspace_bytes(const tpc_cf_geometry* geom, uint64_t max_digits, uint64_t max_clusters);

/* Workspace variants.  TPC_CF_WS_SORTED_ONLY: the caller will only ever run with TPC_CF_DIGITS_SORTED (and without
 * TPC_CF_FORCE_GENERAL): the workspace then holds no charge map, no peak mask and no sort scratch — line index,
 * counts and staging only.  A run that would need the general path returns TPC_CF_E_PARAMS on such a handle, and
 * tpc_cf_run_host does not fall back on a false promise (the status then says path 0). */
enum { TPC_CF_WS_SORTED_ONLY = 1u };
size_t tpc_cf_workspace_bytes_ex(const tpc_cf_geometry* geom, uint64_t max_digits, uint64_t max_clusters, uint32_t ws_flags);
int tpc_cf_create_ex(tpc_cf** h, const tpc_cf_geometry* geom, uint64_t max_digits, uint64_t max_clusters,
                     uint32_t ws_flags, void* workspace, size_t workspace_bytes, void* stream);

/* Creates a handle bound to a caller-owned DEVICE workspace (256-byte aligned, >= tpc_cf_workspace_bytes).
 * Enqueues on `stream` the one-time zeroing of the charge map; every run leaves the map zero again (K0 is an
 * "un-scatter").  Returns TPC_CF_OK or a negative error; *h is set only on success. */
int tpc_cf_create(tpc_cf** h, const tpc_cf_geometry* geom, uint64_t max_digits, uint64_t max_clusters,
                  void* workspace, size_t workspace_bytes, void* stream);

/* Enqueues the whole hot path for `n` digits on out->stream and returns without
 * synchronising.  digits: DEVICE pointer, 8-byte aligned, any order, at most one digit per cell (R11), must
 * stay alive until the stream has passed the run.  geom must equal the geometry given to create.
 * Synchronous errors (nothing enqueued): negative return.  Asynchronous conditions are in out->status.
 * One handle serves one stream at a time.  The call only enqueues kernels, memsets and device-to-device copies on that
 * stream (no allocation, no synchronisation, no host read), so it may be captured in a CUDA graph (with profiling off)
 * and replayed on the same buffers; launch-bound small frames gain from that. */
int tpc_cf_run(tpc_cf* h, const tpc_digit* digits, uint64_t n,
               const tpc_cf_geometry* geom, const tpc_cf_params* params, tpc_cf_out* out);

/* End-to-end convenience used by bench.py's `e2e` leg: HOST digits in (pinned or pageable), HOST clusters and
 * status out; copies host->device, runs, copies the status and the clusters back, synchronises the stream.
 * dev_digits / dev_clusters / dev_status are caller-owned DEVICE staging buffers (max_digits / capacity / 1).
 * A frame of >= 4 Mi digits in >= 2 sectors that carries TPC_CF_DIGITS_SORTED is pipelined over groups of whole
 * sectors (sectors are independent, R2): the copy-in of the next group, the run of the current one and the copy-out of
 * the previous one overlap on three streams (two of them internal to the handle); with pinned host buffers the call
 * then costs about the host->device copy alone.  The result is the same array.  A false promise, or a group that
 * needs more than its share of `capacity`, falls back to the single-shot route by itself. */
int tpc_cf_run_host(tpc_cf* h, const tpc_digit* host_digits, uint64_t n,
                    const tpc_cf_geometry* geom, const tpc_cf_params* params,
                    tpc_digit* dev_digits, tpc_cluster* dev_clusters, tpc_cf_status* dev_status,
                    tpc_cluster* host_clusters, uint64_t capacity, tpc_cf_status* host_status, void* stream);

/* Test hook for the K1 map-parity check: scatters the digits, copies the dense plane
 * (sector,row) into `dense` (DEVICE, npads(row) x n_time uint16, pad-major), and un-scatters again. */
int tpc_cf_debug_dense_plane(tpc_cf* h, const tpc_digit* digits, uint64_t n,
                             uint32_t sector, uint32_t row, uint16_t* dense, void* stream);

/* Launch-shape hint for runs that cover only part of a frame (one frame cut over several GPUs, paper_2402_01205_b200/
 * shard.py; PAPER.md:100 has whole frames per GPU instead).  The fused path sizes its shared-memory line slots from
 * the mean digits per pad line = n / (pads of the WHOLE geometry); a run on a slice of the planes would take them N
 * times too small and fall back to its (exact, slower) overflow paths.  frame_digits = digits of the whole frame the
 * following runs are slices of; 0 = every run is a whole frame (default).  Never changes the result. */
int tpc_cf_set_frame_digits(tpc_cf* h, uint64_t frame_digits);

/* Test / tuning overrides of one handle (the tests force every kernel and every slow path with them; profiling uses
 * them to compare launch shapes).  They select among exact implementations and never change the result.  value 0
 * restores the library's own choice.  Returns TPC_CF_OK, TPC_CF_E_NULL or TPC_CF_E_PARAMS (unknown key, value < 0). */
enum {
    TPC_CF_DEBUG_FUSED_KERNEL = 1,  /* 1 k_fused_pairs, 2 k_fused_blocks (first generation), 3 k_fused_lines (bitmap slots) */
    TPC_CF_DEBUG_PASSES = 2,        /* passes over the time axis of the block-sparse kernels */
    TPC_CF_DEBUG_BLOCK_POOL = 3,    /* pool blocks per line slot (a small pool forces the cell-from-digit-array path) */
    TPC_CF_DEBUG_SURV_CAP = 4,      /* stage-A survivor entries per line slot (a small list forces its overflow path) */
    TPC_CF_DEBUG_PADS_PER_UNIT = 5, /* pads per CTA (multiple of 8) */
    TPC_CF_DEBUG_CTAS_PER_SM = 6    /* 2: never use the 3-CTAs-per-SM instantiation */
};
int tpc_cf_debug_set(tpc_cf* h, int key, int value);

/* Number of kernel launches the last run enqueued (for bench.py's gpu_launches). */
int tpc_cf_last_launch_count(const tpc_cf* h);

/* Name of the dominant kernel the last run enqueued: "k_fused_pairs" ("k_fused_blocks" / "k_fused_lines" where the
 * mean line length or tpc_cf_debug_set asks for them) on the fused sorted path, "k_peaks_map" on the general path.
 * Static string, never NULL for a valid handle ("" before the first run). */
const char* tpc_cf_last_kernel(const tpc_cf* h);

/* Profiling (bench.py's roofline leg).  After tpc_cf_set_profiling(h, 1) every run records CUDA events on its
 * stream around the whole run and around its dominant kernel (the fused kernel on the sorted path, the
 * peak+moment kernel on the general path); the last 64 runs are kept.  tpc_cf_profile_ms(h, run, which) returns
 * the device time in ms of run number `run` (0 = first run after profiling was switched on): which = 0 whole
 * run, 1 dominant kernel.  It synchronises on that run's events.  Negative on error / unknown run. */
int   tpc_cf_set_profiling(tpc_cf* h, int on);
float tpc_cf_profile_ms(tpc_cf* h, uint32_t run, int which);

/* Exclusive prefix sum of n uint32 (in -> out, DEVICE pointers, may alias; *total, optional DEVICE pointer, receives
 * the sum as 64-bit) WITHOUT any allocation and without a handle: the scan of K3 (compaction) for callers that cannot
 * allocate — code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc.  The kernels are the ones
 * tpc_cf_run uses; their scratch (one partial sum per 1024 elements) lives in a file-scope device array of the
 * library: 257 KB that every GPU which loads the library holds until exit.  Limit: n <= tpc_cf_scan_static_max_n() =
 * 2^26 elements per call; beyond it the call enqueues nothing and returns TPC_CF_E_CAPACITY.  Calls no cudaMalloc /
 * cudaFree / allocating routine; enqueues on `stream` and returns.  All calls on a device share the scratch: each
 * overwrites what it reads, so back-to-back calls on one stream are independent, but calls that OVERLAP on the GPU
 * (several streams, concurrent graph replays) race.  The array's device address is resolved once per device by
 * tpc_cf_scan_static_setup() (cudaGetSymbolAddress with that device current); the scan calls it on first use — call it
 * yourself before capturing a graph. */
uint64_t tpc_cf_scan_static_max_n(void);
int tpc_cf_scan_static_setup(void);
int tpc_cf_scan_u32_static(const uint32_t* in, uint32_t* out, uint64_t n, unsigned long long* total, void* stream);

/* Test hook: the same scan with its scratch taken from the handle's caller-owned workspace (the path tpc_cf_run
 * takes); n is limited by the workspace.  tests/test_zz_no_alloc.py compares the two. */
int tpc_cf_debug_scan_u32(tpc_cf* h, const uint32_t* in, uint32_t* out, uint64_t n, unsigned long long* total, void* stream);

int tpc_cf_destroy(tpc_cf* h);

const char* tpc_cf_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* TPC_CF_H */
