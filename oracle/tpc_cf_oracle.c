/*
 * tpc_cf_oracle.c — CPU ORACLE of the TPC cluster finder.  TEST INFRASTRUCTURE, NOT PRODUCT.
 * See tpc_cf_oracle.h for who may use it.  Plain C99, single thread, no blocking / fusion /
 * reordering beyond the definition: SURVEY.md §8(c) "Algorithm (oracle, step by step)",
 * which restates BASELINE.json:north_star for the step named in PAPER.md:57.
 *
 * Notation follows the definition: Q = zero-bordered charge map of one (sector,row) plane,
 * p = pad, t = time bin, (dp,dt) = offset from the peak, S0/S1p/S1t/S2p/S2t = moment sums.
 */
#include "tpc_cf_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#define BORDER 2            /* 5x5 window => reads reach +-2 outside the plane (R2: they return 0) */
#define ABORDER 4           /* V4: D(x) reads the peak-charge map +-2 around a cell that is +-2 from the peak */

static int sgn(int x) { return (x > 0) - (x < 0); }

static uint32_t pads_of_row(const orc_geometry* g, uint32_t r)
{
    return g->npads ? (uint32_t)g->npads[r] : g->max_pads;
}

/* R11: a digit is valid iff it addresses an existing cell and carries charge. */
static int digit_valid(const orc_geometry* g, const orc_digit* d)
{
    if (d->sector >= g->n_sectors) return 0;
    if (d->row >= g->n_rows) return 0;
    if (d->pad >= pads_of_row(g, d->row)) return 0;
    if (d->time >= g->n_time) return 0;
    if (d->charge == 0) return 0;
    return 1;
}

static int geometry_ok(const orc_geometry* g)
{
    if (!g) return 0;
    if (g->n_sectors == 0 || g->n_rows == 0 || g->max_pads == 0 || g->n_time == 0) return 0;
    if (g->n_sectors > 256 || g->n_rows > 256 || g->max_pads > 256 || g->n_time > 65536) return 0;
    if (g->npads)
        for (uint32_t r = 0; r < g->n_rows; ++r)
            if (g->npads[r] == 0 || g->npads[r] > g->max_pads) return 0;
    return 1;
}

typedef struct { int64_t S0, S1p, S1t, S2p, S2t; } orc_sums;

#define QAT(pp, tt) Q[(size_t)((pp) + BORDER) * W + (size_t)((tt) + BORDER)]
#define AAT(pp, tt) A[(size_t)((pp) + ABORDER) * WA + (size_t)((tt) + ABORDER)]

/* R1 / R6: is cell (p,t) a peak? */
static int is_peak(const uint16_t* Q, size_t W, int p, int t, const orc_params* prm)
{
    const uint16_t q = QAT(p, t);
    if (q < prm->q_peak_min) return 0;                       /* R6 */
    for (int dp = -1; dp <= 1; ++dp)
        for (int dt = -1; dt <= 1; ++dt) {
            if (dp == 0 && dt == 0) continue;
            const uint16_t nb = QAT(p + dp, t + dt);
            if (dp < 0 || (dp == 0 && dt < 0)) { if (!(q > nb)) return 0; }    /* earlier: strict (R1) */
            else                               { if (!(q >= nb)) return 0; }   /* later: non-strict   */
        }
    return 1;
}

/* R3 / R4: sums over the cells that enter the cluster at peak (p,t).
 * A == NULL: every cell enters with its charge Q(x).
 * A != NULL (V4): A is the peak-charge map of the plane's clusters (qMax at a cluster's peak cell, else 0); a cell
 * enters with c'(x) = floor(64 * Q(x) * A(peak) / D(x)), D(x) = sum of A over the 5x5 cells around x;
 * *shared is set iff D(x) != A(peak) for some cell x with charge that entered. */
static orc_sums window_sums(const uint16_t* Q, size_t W, const uint16_t* A, size_t WA,
                            int p, int t, const orc_params* prm, int* shared)
{
    orc_sums m = {0, 0, 0, 0, 0};
    if (shared) *shared = 0;
    for (int dp = -2; dp <= 2; ++dp)
        for (int dt = -2; dt <= 2; ++dt) {
            const int ring = (abs(dp) == 2 || abs(dt) == 2);
            if (ring) {                                       /* outer ring: gated (R3, R4) */
                const int ip = dp - sgn(dp), it = dt - sgn(dt);
                if (QAT(p + ip, t + it) < prm->q_inner_gate) continue;
            }
            int64_t c = QAT(p + dp, t + dt);                  /* inner 3x3 always counted */
            if (A) {
                int64_t D = 0;
                for (int a = -2; a <= 2; ++a)
                    for (int b = -2; b <= 2; ++b) D += AAT(p + dp + a, t + dt + b);
                const int64_t Az = AAT(p, t);
                if (c > 0 && D != Az) *shared = 1;
                c = (64 * c * Az) / D;                        /* D >= Az > 0: the cluster's own window contains x */
            }
            m.S0 += c; m.S1p += c * dp; m.S1t += c * dt; m.S2p += c * dp * dp; m.S2t += c * dt * dt;
        }
    return m;
}

/* V1 / V2 on the UNSHARED sums: flags of the cluster at peak (p,t); returns 0 if a cut drops it. */
static int flags_and_cuts(const orc_sums* m, uint16_t q, int p, int t, uint32_t P, uint32_t T,
                          const orc_params* prm, unsigned* flags)
{
    unsigned fl = 0;
    if (p < 2 || p + 2 >= (int)P) fl |= ORC_F_EDGE_PAD;
    if (t < 2 || t + 2 >= (int)T) fl |= ORC_F_EDGE_TIME;
    if (m->S2p == 0) fl |= ORC_F_SINGLE_PAD;
    if (m->S2t == 0) fl |= ORC_F_SINGLE_TIME;
    if (prm->q_saturation != 0 && q >= prm->q_saturation) fl |= ORC_F_SATURATED;
    *flags = fl;
    if (m->S0 < (int64_t)prm->q_tot_min) return 0;
    if ((prm->flags & ORC_CUT_SINGLE_PAD) && (fl & ORC_F_SINGLE_PAD)) return 0;
    if ((prm->flags & ORC_CUT_SINGLE_TIME) && (fl & ORC_F_SINGLE_TIME)) return 0;
    return 1;
}

/* One plane: Q is (P+4) x (T+4), row stride W = T+4, already filled; A is scratch of (P+8) x (T+8) for V4.
 * Emits clusters in (pad,time) loop order.  Returns the number of clusters found (all counted, only those
 * that fit are written), or -3 if an exactness assertion fails (P5). */
static int64_t scan_plane(const uint16_t* Q, uint16_t* A, uint32_t P, uint32_t T,
                          uint32_t s, uint32_t r, const orc_params* prm,
                          orc_cluster* out, uint64_t room)
{
    const size_t W = (size_t)T + 2 * BORDER, WA = (size_t)T + 2 * ABORDER;
    const int share = (prm->flags & ORC_SHARE_CHARGE) != 0;
    int64_t n_found = 0;

    if (share) {
        /* V4, first the set of clusters of the plane: A(x) = qMax of the cluster whose peak is x, else 0 */
        memset(A, 0, ((size_t)P + 2 * ABORDER) * WA * sizeof(uint16_t));
        for (int p = 0; p < (int)P; ++p)
            for (int t = 0; t < (int)T; ++t) {
                if (QAT(p, t) < prm->q_peak_min) continue;    /* R6 (most cells are empty) */
                if (!is_peak(Q, W, p, t, prm)) continue;
                const orc_sums m = window_sums(Q, W, NULL, 0, p, t, prm, NULL);
                unsigned fl;
                if (flags_and_cuts(&m, QAT(p, t), p, t, P, T, prm, &fl)) AAT(p, t) = QAT(p, t);
            }
    }

    for (int p = 0; p < (int)P; ++p) {                       /* pad-major, time-minor (R10) */
        for (int t = 0; t < (int)T; ++t) {
            const uint16_t q = QAT(p, t);
            if (q < prm->q_peak_min) continue;                /* R6 (most cells are empty) */
            if (!is_peak(Q, W, p, t, prm)) continue;
            orc_sums m = window_sums(Q, W, NULL, 0, p, t, prm, NULL);
            /* P5 / R8: every sum is an integer below 2^24, so fp32 accumulation is exact. */
            if (m.S0 >= (1 << 24) || llabs(m.S1p) >= (1 << 24) || llabs(m.S1t) >= (1 << 24) ||
                m.S2p >= (1 << 24) || m.S2t >= (1 << 24)) return -3;

            /* V1 / V2: flags from the peak cell and the sums, then the cuts */
            unsigned fl;
            if (!flags_and_cuts(&m, q, p, t, P, T, prm, &fl)) continue;

            uint32_t qtot = (uint32_t)m.S0;
            if (share) {                                      /* V4: the same cells, with their shared charges */
                int shared;
                m = window_sums(Q, W, A, WA, p, t, prm, &shared);
                if (shared) fl |= ORC_F_SHARED;
                qtot = (uint32_t)((m.S0 + 32) / 64);
            }

            if ((uint64_t)n_found < room) {
                double mp = 0, mt = 0, vp = 0, vt = 0;
                if (m.S0 > 0) {                               /* (S0 = 0: only under V4, every share rounded to 0) */
                    mp = (double)m.S1p / (double)m.S0;
                    mt = (double)m.S1t / (double)m.S0;
                    vp = (double)m.S2p / (double)m.S0 - mp * mp;
                    vt = (double)m.S2t / (double)m.S0 - mt * mt;
                }
                if (vp < 0) vp = 0;
                if (vt < 0) vt = 0;
                orc_cluster c;
                memset(&c, 0, sizeof c);
                c.sector = (uint8_t)s; c.row = (uint8_t)r; c.pad = (uint8_t)p;
                c.flags = (prm->flags & ORC_CLUSTER_FLAGS) ? (uint8_t)fl : 0;
                c.time = (uint16_t)t; c.qmax = q; c.qtot = qtot;
                c.pad_mean = (float)((double)p + mp);         /* R7 */
                c.time_mean = (float)((double)t + mt);
                c.sigma_pad = (float)sqrt(vp);
                c.sigma_time = (float)sqrt(vt);
                c.rsv = 0;
                out[n_found] = c;
            }
            ++n_found;
        }
    }
    return n_found;
}
#undef QAT
#undef AAT

int tpc_cf_oracle_run_planes(const orc_digit* digits, uint64_t n,
                             const orc_geometry* g, const orc_params* prm,
                             uint32_t plane_begin, uint32_t plane_end,
                             orc_cluster* out, uint64_t capacity, orc_status* st)
{
    if (!g || !prm || !st || (n && !digits) || (capacity && !out)) return -1;
    if (!geometry_ok(g) || prm->q_peak_min == 0) return -1;
    const uint32_t n_planes = g->n_sectors * g->n_rows;
    if (plane_end > n_planes) plane_end = n_planes;
    if (plane_begin > plane_end) return -1;
    memset(st, 0, sizeof *st);

    /* bucket digits by plane (counting sort on sector*n_rows+row; input order is free, R12) */
    uint64_t* first = (uint64_t*)calloc((size_t)n_planes + 1, sizeof(uint64_t));
    uint64_t* order = (uint64_t*)malloc((size_t)(n ? n : 1) * sizeof(uint64_t));
    uint64_t* fill  = (uint64_t*)malloc((size_t)(n_planes + 1) * sizeof(uint64_t));
    const size_t W = (size_t)g->n_time + 2 * BORDER;
    uint16_t* Q = (uint16_t*)malloc(((size_t)g->max_pads + 2 * BORDER) * W * sizeof(uint16_t));
    uint16_t* A = (uint16_t*)malloc(((size_t)g->max_pads + 2 * ABORDER) * ((size_t)g->n_time + 2 * ABORDER) * sizeof(uint16_t));
    if (!first || !order || !fill || !Q || !A) { free(first); free(order); free(fill); free(Q); free(A); return -2; }

    uint64_t n_bad = 0, n_used = 0;
    for (uint64_t i = 0; i < n; ++i) {
        if (!digit_valid(g, &digits[i])) {
            /* count a bad digit once, and only if the full frame is being processed or it
             * cannot be attributed to a plane outside the requested range */
            const uint32_t pl = (digits[i].sector < g->n_sectors && digits[i].row < g->n_rows)
                                ? digits[i].sector * g->n_rows + digits[i].row : plane_begin;
            if (pl >= plane_begin && pl < plane_end) ++n_bad;
            continue;
        }
        ++first[(uint32_t)digits[i].sector * g->n_rows + digits[i].row + 1];
    }
    for (uint32_t k = 0; k < n_planes; ++k) first[k + 1] += first[k];
    memcpy(fill, first, (size_t)(n_planes + 1) * sizeof(uint64_t));
    for (uint64_t i = 0; i < n; ++i)
        if (digit_valid(g, &digits[i]))
            order[fill[(uint32_t)digits[i].sector * g->n_rows + digits[i].row]++] = i;

    uint64_t n_clusters = 0;
    int rc = 0;
    for (uint32_t pl = plane_begin; pl < plane_end; ++pl) {
        const uint32_t s = pl / g->n_rows, r = pl % g->n_rows;
        const uint32_t P = pads_of_row(g, r), T = g->n_time;
        memset(Q, 0, ((size_t)P + 2 * BORDER) * W * sizeof(uint16_t));          /* Q = 0, zero border */
        for (uint64_t k = first[pl]; k < first[pl + 1]; ++k) {
            const orc_digit* d = &digits[order[k]];
            Q[(size_t)(d->pad + BORDER) * W + (size_t)(d->time + BORDER)] = d->charge;
            ++n_used;
        }
        const uint64_t room = capacity > n_clusters ? capacity - n_clusters : 0;
        const int64_t found = scan_plane(Q, A, P, T, s, r, prm, out ? out + n_clusters : NULL, room);
        if (found < 0) { rc = (int)found; break; }
        n_clusters += (uint64_t)found;
    }
    st->n_clusters = n_clusters;
    st->n_digits_used = n_used;
    st->n_bad_digits = n_bad;
    st->overflow = n_clusters > capacity ? 1u : 0u;
    free(first); free(order); free(fill); free(Q); free(A);
    return rc;
}

int tpc_cf_oracle_run(const orc_digit* digits, uint64_t n,
                      const orc_geometry* g, const orc_params* prm,
                      orc_cluster* out, uint64_t capacity, orc_status* st)
{
    if (!g) return -1;
    return tpc_cf_oracle_run_planes(digits, n, g, prm, 0, g->n_sectors * g->n_rows, out, capacity, st);
}

int tpc_cf_oracle_dense_plane(const orc_digit* digits, uint64_t n,
                              const orc_geometry* g, uint32_t sector, uint32_t row,
                              uint16_t* dense)
{
    if (!g || !dense || (n && !digits) || !geometry_ok(g)) return -1;
    if (sector >= g->n_sectors || row >= g->n_rows) return -1;
    const uint32_t P = pads_of_row(g, row), T = g->n_time;
    memset(dense, 0, (size_t)P * T * sizeof(uint16_t));
    for (uint64_t i = 0; i < n; ++i) {
        const orc_digit* d = &digits[i];
        if (!digit_valid(g, d) || d->sector != sector || d->row != row) continue;
        dense[(size_t)d->pad * T + d->time] = d->charge;
    }
    return 0;
}
