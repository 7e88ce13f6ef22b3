/* tpc_fe_oracle.c — CPU ORACLE of the TPC front-end filter "TPC-FE v1" (tpc_fe_oracle.h; step named in PAPER.md:57).
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Plain C99, single thread, int64 arithmetic, the definition executed literally in
 * the order of the text: no blocking, no fusion. */
#include <stdlib.h>
#include <string.h>

#include "tpc_fe_oracle.h"

/* floor(a / b) for b > 0 */
static int64_t floor_div(int64_t a, int64_t b)
{
    int64_t q = a / b;
    if (a % b != 0 && a < 0) q -= 1;
    return q;
}

int tpc_fe_oracle_run(const uint16_t* raw, const uint16_t* ped4, const tpc_fe_oracle_geometry* g,
                      const tpc_fe_oracle_params* prm, uint32_t plane_begin, uint32_t plane_end,
                      tpc_fe_oracle_digit* out, uint64_t capacity, tpc_fe_oracle_status* status)
{
    if (!raw || !ped4 || !g || !prm || !status || (!out && capacity)) return -1;
    if (g->n_sectors == 0 || g->n_sectors > 256 || g->n_rows == 0 || g->n_rows > 256 || g->max_pads == 0 ||
        g->max_pads > 255 || g->n_time == 0 || g->n_time > 65535) return -2;
    if (g->npads)
        for (uint32_t r = 0; r < g->n_rows; r++)
            if (g->npads[r] == 0 || g->npads[r] > g->max_pads) return -2;
    if (plane_begin > plane_end || plane_end > g->n_sectors * g->n_rows) return -2;
    const int k = prm->it_decay_shift, j = prm->it_kappa_shift;
    if (prm->zs_threshold < 1 || prm->cm_quiet4 > 4095 || prm->cm_min_pads < 1 || k < 1 || k > 15 ||
        (j != 0 && (j < k || j > 14))) return -5;

    const uint32_t W = (g->max_pads + 7u) / 8u * 8u, T = g->n_time;
    int64_t* S = (int64_t*)malloc(sizeof(int64_t) * W);
    int64_t* x = (int64_t*)malloc(sizeof(int64_t) * W);
    int32_t* kept = (int32_t*)malloc(sizeof(int32_t) * (size_t)W * T);     /* q of a kept sample, else -1 */
    if (!S || !x || !kept) { free(S); free(x); free(kept); return -7; }

    uint64_t n_out = 0;
    for (uint32_t plane = plane_begin; plane < plane_end; plane++) {
        const uint32_t sector = plane / g->n_rows, row = plane % g->n_rows;
        const uint32_t P = g->npads ? g->npads[row] : g->max_pads;
        const uint16_t* ped = ped4 + (size_t)plane * W;
        for (uint32_t p = 0; p < P; p++) S[p] = 0;
        for (uint32_t t = 0; t < T; t++) {
            const uint16_t* r = raw + ((size_t)plane * T + t) * W;
            /* (P) */
            for (uint32_t p = 0; p < P; p++) x[p] = 4 * (int64_t)r[p] - (int64_t)ped[p];
            /* (CM) */
            int64_t n = 0, s = 0;
            for (uint32_t p = 0; p < P; p++) {
                int64_t a = x[p] < 0 ? -x[p] : x[p];
                if (a <= (int64_t)prm->cm_quiet4) { n += 1; s += x[p]; }
            }
            int64_t cm = 0;
            if (n >= (int64_t)prm->cm_min_pads) cm = floor_div(2 * s + n, 2 * n);
            for (uint32_t p = 0; p < P; p++) {
                /* (IT) */
                int64_t z = x[p] - cm + floor_div(S[p], 4096);
                /* (ZS) */
                int64_t q = floor_div(z + 2, 4);
                if (q > 65535) q = 65535;
                int is_kept = q >= (int64_t)prm->zs_threshold;
                kept[(size_t)p * T + t] = is_kept ? (int32_t)q : -1;
                int64_t add = 0;
                if (is_kept && j != 0) add = q * ((int64_t)1 << (14 - j));
                S[p] = S[p] - floor_div(S[p], (int64_t)1 << k) + add;
            }
        }
        for (uint32_t p = 0; p < P; p++)
            for (uint32_t t = 0; t < T; t++) {
                int32_t q = kept[(size_t)p * T + t];
                if (q < 0) continue;
                if (n_out < capacity) {
                    tpc_fe_oracle_digit d;
                    d.sector = (uint8_t)sector; d.row = (uint8_t)row; d.pad = (uint8_t)p; d.rsv = 0;
                    d.time = (uint16_t)t; d.charge = (uint16_t)q;
                    out[n_out] = d;
                }
                n_out++;
            }
    }
    free(S); free(x); free(kept);
    status->n_digits = n_out;
    status->overflow = n_out > capacity ? 2u : 0u;
    status->rsv = 0;
    return 0;
}
