/* tpc_fe_gen.c — seeded synthetic RAW TPC samples (inputs only) for the front-end filter.
 *
 * Stands in for the detector's raw ADC stream in front of "zero-suppression after common-mode correction and ion tail
 * cancellation", which is not available.  It is a forward model of the effects the filter removes, laid
 * over the digits of the cluster generator (tpc_gen.c); it holds none of the filter's arithmetic (floating point here,
 * integer fixed point there) and serves the oracle tests and the CUDA path alike.
 *
 *   ped4[pl][p]  = 240 + (hash mod 161)                     pedestal 60 .. 100 ADC in quarter counts
 *   sig[t][p]    = charge of the digit at (pl, p, t), else 0
 *   cm[t]        = -cm_frac * sum_p sig[t][p] / P            common-mode dip, shared by all pads of the row
 *   tail[t][p]   : u = 0;  per t:  tail = u;  u = lambda * u + kappa * sig[t][p]       undershoot after a signal
 *   raw[t][p]    = clamp(rint(ped4/4 + sig + cm - tail + sigma * g), 0, 4095),  g ~ approximately N(0,1): the sum of
 *                  four 16-bit uniforms of one SplitMix64 hash of (seed, plane, t, p), centred and scaled
 *   Entries p >= P (up to the row pitch W) are filled with 0xFFFF so that a reader that uses them is caught.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct { uint8_t sector, row, pad, rsv; uint16_t time, charge; } digit_t;

typedef struct {
    uint64_t seed;
    uint32_t n_sectors, n_rows, max_pads, n_time;
    const uint16_t* npads;
    double noise_sigma, cm_frac, tail_lambda, tail_kappa;
    uint32_t plane_begin, plane_end;     /* planes to fill; raw / ped4 are indexed from plane_begin */
} fe_cfg_t;

static uint64_t mix(uint64_t z)
{
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

static size_t lower_bound(const digit_t* d, size_t n, uint32_t sector, uint32_t row)
{
    size_t lo = 0, hi = n;
    uint32_t key = sector * 256u + row;
    while (lo < hi) {
        size_t mid = (lo + hi) / 2;
        if ((uint32_t)d[mid].sector * 256u + d[mid].row < key) lo = mid + 1; else hi = mid;
    }
    return lo;
}

int tpc_fe_gen_raw(const fe_cfg_t* c, const digit_t* digits, uint64_t n, uint16_t* raw, uint16_t* ped4)
{
    const uint32_t W = (c->max_pads + 7u) / 8u * 8u, T = c->n_time;
    int err = 0;
#pragma omp parallel
    {
        uint16_t* sig = (uint16_t*)malloc(sizeof(uint16_t) * (size_t)W * T);
        double* u = (double*)malloc(sizeof(double) * W);
        if (!sig || !u) {
#pragma omp atomic write
            err = 1;
        }
#pragma omp for schedule(dynamic, 1)
        for (uint32_t plane = c->plane_begin; plane < c->plane_end; plane++) {
            if (err) continue;
            const uint32_t sector = plane / c->n_rows, row = plane % c->n_rows;
            const uint32_t P = c->npads ? c->npads[row] : c->max_pads;
            uint16_t* r = raw + (size_t)(plane - c->plane_begin) * T * W;
            uint16_t* ped = ped4 + (size_t)(plane - c->plane_begin) * W;
            const uint64_t base = mix(c->seed * 0x100000001B3ull + plane);
            for (uint32_t p = 0; p < W; p++) ped[p] = p < P ? (uint16_t)(240 + mix(base ^ (0xA5A5ull + p)) % 161) : 0xFFFFu;
            memset(sig, 0, sizeof(uint16_t) * (size_t)W * T);
            size_t lo = lower_bound(digits, n, sector, row), hi = lower_bound(digits, n, sector, row + 1);
            for (size_t i = lo; i < hi; i++)
                if (digits[i].pad < P && digits[i].time < T) sig[(size_t)digits[i].time * W + digits[i].pad] = digits[i].charge;
            for (uint32_t p = 0; p < W; p++) u[p] = 0.0;
            for (uint32_t t = 0; t < T; t++) {
                const uint16_t* s = sig + (size_t)t * W;
                uint16_t* o = r + (size_t)t * W;
                double sum = 0.0;
                for (uint32_t p = 0; p < P; p++) sum += s[p];
                const double cm = -c->cm_frac * sum / (double)P;
                const uint64_t hb = mix(base + ((uint64_t)t << 20));
                for (uint32_t p = 0; p < P; p++) {
                    uint64_t h = mix(hb + p);
                    double g = (double)((h & 0xFFFF) + ((h >> 16) & 0xFFFF) + ((h >> 32) & 0xFFFF) + (h >> 48)) - 131070.0;
                    g *= 1.0 / 37837.2;    /* sd of the sum of four uniform 16-bit integers */
                    double v = 0.25 * ped[p] + s[p] + cm - u[p] + c->noise_sigma * g;
                    u[p] = c->tail_lambda * u[p] + c->tail_kappa * s[p];
                    double rv = rint(v);
                    o[p] = (uint16_t)(rv < 0.0 ? 0.0 : rv > 4095.0 ? 4095.0 : rv);
                }
                for (uint32_t p = P; p < W; p++) o[p] = 0xFFFFu;
            }
        }
        free(sig);
        free(u);
    }
    return err;
}
