/*
 * tpc_gen.c — seeded synthetic TPC time-frame generator (INPUTS ONLY; holds none of the cluster finder's
 * arithmetic).  Serves both the oracle tests and the CUDA path; neither of those shares anything else.
 *
 * Stands in for the paper's workload (2.8 ms Pb-Pb / pp time frames from ALICE MC and 2022 data, PAPER.md:21,
 * 115, 129), which is not available here.  Recipe: BASELINE.json:configs as made concrete in SURVEY.md §8(d)
 * "Synthetic inputs" and restated in DESIGN.md §6:
 *   per (frame, sector, row) plane, an independent substream (SplitMix64 -> xoshiro256**):
 *   1. n ~ Poisson(rho * npads[row] * n_time) clusters (count of unit-rate exponential arrivals before lambda)
 *   2. centre uniform on [-1/2, P-1/2) x [-1/2, T-1/2); sigma_pad ~ U(0.6,1.0); sigma_time ~ U(0.8,1.5);
 *      Q = exp(N(ln 120, 0.6))
 *   3. (pair_prob > 0) each base cluster spawns a partner at (c_p + U(-2,2), c_t + U(-3,3)) with that probability
 *   4. signal = pixel-integrated 2-D Gaussian on the 7 x 11 window around the rounded centre, summed in float
 *   5. ADC = clamp(rint(signal + N(0,1)), 0, 65535) for cells inside at least one window; others stay 0
 *   6. zero suppression: ADC < 2 dropped
 *   7. (plateau_rate > 0) Poisson(plateau_rate * rho * cells) flat-top rectangles k_p in {1,2,3} x k_t in {2..5},
 *      value max(U{30..300}, 1 + max ADC over the rectangle and its 1-cell border)
 *   8. one 8-byte digit per non-zero cell, ascending (sector,row,pad,time)
 * Output is bit-identical for any thread count (planes are independent and concatenated in plane order).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    uint8_t  sector, row, pad, rsv;
    uint16_t time, charge;
} gen_digit;

typedef struct {
    uint64_t seed;
    uint32_t n_sectors, n_rows, max_pads, n_time;
    const uint16_t* npads;     /* n_rows entries or NULL */
    double rho;                /* generated clusters per cell */
    double pair_prob;          /* config 4: 3/17 */
    double plateau_rate;       /* config 4: 0.01 */
    uint32_t n_threads;        /* 0 = all */
    uint32_t sector_begin, sector_end;   /* generate sectors [begin,end) only (end = 0 => n_sectors) */
} gen_config;

typedef struct { uint64_t s[4]; double spare; int has_spare; } rng_t;

static uint64_t splitmix64(uint64_t* x)
{
    uint64_t z = (*x += 0x9E3779B97F4A7C15ull);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
static inline uint64_t rotl(uint64_t x, int k) { return (x << k) | (x >> (64 - k)); }
static uint64_t rng_next(rng_t* r)
{
    uint64_t* s = r->s;
    const uint64_t result = rotl(s[1] * 5, 7) * 9;
    const uint64_t t = s[1] << 17;
    s[2] ^= s[0]; s[3] ^= s[1]; s[1] ^= s[2]; s[0] ^= s[3]; s[2] ^= t; s[3] = rotl(s[3], 45);
    return result;
}
static void rng_seed(rng_t* r, uint64_t seed, uint32_t frame, uint32_t sector, uint32_t row)
{
    uint64_t x = seed * 0xD1342543DE82EF95ull + 0x2545F4914F6CDD1Dull;
    x ^= (uint64_t)frame << 42; splitmix64(&x);
    x ^= (uint64_t)sector << 21; splitmix64(&x);
    x ^= (uint64_t)row; splitmix64(&x);
    for (int i = 0; i < 4; ++i) r->s[i] = splitmix64(&x);
    r->has_spare = 0;
}
static double rng_uniform(rng_t* r) { return (double)(rng_next(r) >> 11) * (1.0 / 9007199254740992.0); }
static double rng_range(rng_t* r, double a, double b) { return a + (b - a) * rng_uniform(r); }
static double rng_normal(rng_t* r)
{
    if (r->has_spare) { r->has_spare = 0; return r->spare; }
    const double u1 = 1.0 - rng_uniform(r), u2 = rng_uniform(r);
    const double m = sqrt(-2.0 * log(u1)), a = 6.283185307179586476925 * u2;
    r->spare = m * sin(a); r->has_spare = 1;
    return m * cos(a);
}
static uint32_t rng_poisson(rng_t* r, double lambda)
{
    uint32_t k = 0; double acc = 0.0;
    for (;;) { acc += -log(1.0 - rng_uniform(r)); if (acc >= lambda) return k; ++k; }
}
static uint32_t rng_int(rng_t* r, uint32_t lo, uint32_t hi) /* inclusive */
{
    uint32_t v = lo + (uint32_t)(rng_uniform(r) * (double)(hi - lo + 1));
    return v > hi ? hi : v;
}

typedef struct { int p0, p1, t0, t1; } rect_t;   /* inclusive, clipped */
typedef struct { gen_digit* d; uint64_t n, cap; } dvec_t;
typedef struct { float* sig; uint8_t* mask; uint16_t* adc; rect_t* rects; size_t nrect, caprect; } scratch_t;

static int push_digit(dvec_t* v, gen_digit d)
{
    if (v->n == v->cap) {
        uint64_t nc = v->cap ? v->cap * 2 : 4096;
        gen_digit* nd = (gen_digit*)realloc(v->d, nc * sizeof(gen_digit));
        if (!nd) return -1;
        v->d = nd; v->cap = nc;
    }
    v->d[v->n++] = d;
    return 0;
}
static int push_rect(scratch_t* s, rect_t r)
{
    if (s->nrect == s->caprect) {
        size_t nc = s->caprect ? s->caprect * 2 : 1024;
        rect_t* nr = (rect_t*)realloc(s->rects, nc * sizeof(rect_t));
        if (!nr) return -1;
        s->rects = nr; s->caprect = nc;
    }
    s->rects[s->nrect++] = r;
    return 0;
}
static double Phi(double x) { return 0.5 * (1.0 + erf(x * 0.70710678118654752440)); }

static int add_cluster(scratch_t* s, int P, int T, double cp, double ct, double sp, double st, double Q)
{
    const int rp = (int)lrint(cp), rt = (int)lrint(ct);
    double fp[7], ft[11];
    for (int i = 0; i < 7; ++i) { const double p = rp - 3 + i; fp[i] = Phi((p + 0.5 - cp) / sp) - Phi((p - 0.5 - cp) / sp); }
    for (int j = 0; j < 11; ++j) { const double t = rt - 5 + j; ft[j] = Phi((t + 0.5 - ct) / st) - Phi((t - 0.5 - ct) / st); }
    rect_t r = { rp - 3, rp + 3, rt - 5, rt + 5 };
    if (r.p0 < 0) r.p0 = 0; if (r.p1 > P - 1) r.p1 = P - 1;
    if (r.t0 < 0) r.t0 = 0; if (r.t1 > T - 1) r.t1 = T - 1;
    if (r.p0 > r.p1 || r.t0 > r.t1) return 0;
    for (int p = r.p0; p <= r.p1; ++p)
        for (int t = r.t0; t <= r.t1; ++t) {
            const size_t c = (size_t)p * T + t;
            s->sig[c] += (float)(Q * fp[p - (rp - 3)] * ft[t - (rt - 5)]);
            s->mask[c] = 1;
        }
    return push_rect(s, r);
}

static int gen_plane(const gen_config* cfg, uint32_t frame, uint32_t sector, uint32_t row, scratch_t* s, dvec_t* out)
{
    const int P = cfg->npads ? cfg->npads[row] : (int)cfg->max_pads, T = (int)cfg->n_time;
    rng_t rng; rng_seed(&rng, cfg->seed, frame, sector, row);
    s->nrect = 0;
    const uint32_t n = rng_poisson(&rng, cfg->rho * (double)P * (double)T);
    for (uint32_t k = 0; k < n; ++k) {
        const double cp = rng_range(&rng, -0.5, P - 0.5), ct = rng_range(&rng, -0.5, T - 0.5);
        const double sp = rng_range(&rng, 0.6, 1.0), st = rng_range(&rng, 0.8, 1.5);
        const double Q = exp(log(120.0) + 0.6 * rng_normal(&rng));
        if (add_cluster(s, P, T, cp, ct, sp, st, Q)) return -1;
        if (cfg->pair_prob > 0.0 && rng_uniform(&rng) < cfg->pair_prob) {
            const double cp2 = cp + rng_range(&rng, -2.0, 2.0), ct2 = ct + rng_range(&rng, -3.0, 3.0);
            const double sp2 = rng_range(&rng, 0.6, 1.0), st2 = rng_range(&rng, 0.8, 1.5);
            const double Q2 = exp(log(120.0) + 0.6 * rng_normal(&rng));
            if (cp2 > -3.5 && cp2 < P + 2.5 && ct2 > -5.5 && ct2 < T + 4.5)
                if (add_cluster(s, P, T, cp2, ct2, sp2, st2, Q2)) return -1;
        }
    }
    /* noise + digitisation + zero suppression, cells in (pad,time) order */
    const size_t cells = (size_t)P * T;
    for (size_t c = 0; c < cells; ++c) {
        if ((c & 7) == 0 && c + 8 <= cells) { uint64_t w; memcpy(&w, s->mask + c, 8); if (!w) { c += 7; continue; } }
        if (!s->mask[c]) continue;
        double v = rint((double)s->sig[c] + rng_normal(&rng));
        if (v < 0) v = 0; if (v > 65535) v = 65535;
        s->adc[c] = v < 2 ? 0 : (uint16_t)v;
    }
    if (cfg->plateau_rate > 0.0) {
        const uint32_t npl = rng_poisson(&rng, cfg->plateau_rate * cfg->rho * (double)cells);
        for (uint32_t k = 0; k < npl; ++k) {
            const int kp = (int)rng_int(&rng, 1, 3), kt = (int)rng_int(&rng, 2, 5);
            if (kp > P || kt > T) continue;
            const int p0 = (int)rng_int(&rng, 0, (uint32_t)(P - kp)), t0 = (int)rng_int(&rng, 0, (uint32_t)(T - kt));
            uint32_t v = rng_int(&rng, 30, 300), mx = 0;
            for (int p = p0 - 1; p <= p0 + kp; ++p)
                for (int t = t0 - 1; t <= t0 + kt; ++t)
                    if (p >= 0 && p < P && t >= 0 && t < T) { const uint32_t a = s->adc[(size_t)p * T + t]; if (a > mx) mx = a; }
            if (mx + 1 > v) v = mx + 1;
            if (v > 65535) v = 65535;
            for (int p = p0; p < p0 + kp; ++p)
                for (int t = t0; t < t0 + kt; ++t) { s->adc[(size_t)p * T + t] = (uint16_t)v; s->mask[(size_t)p * T + t] = 1; }
            rect_t r = { p0, p0 + kp - 1, t0, t0 + kt - 1 };
            if (push_rect(s, r)) return -1;
        }
    }
    for (size_t c = 0; c < cells; ++c) {
        if ((c & 7) == 0 && c + 8 <= cells) { uint64_t w; memcpy(&w, s->mask + c, 8); if (!w) { c += 7; continue; } }
        if (!s->mask[c] || !s->adc[c]) continue;
        gen_digit d = { (uint8_t)sector, (uint8_t)row, (uint8_t)(c / T), 0, (uint16_t)(c % T), s->adc[c] };
        if (push_digit(out, d)) return -1;
    }
    for (size_t k = 0; k < s->nrect; ++k) {   /* restore the scratch to all-zero */
        const rect_t r = s->rects[k];
        for (int p = r.p0; p <= r.p1; ++p) {
            const size_t c = (size_t)p * T + r.t0; const size_t w = (size_t)(r.t1 - r.t0 + 1);
            memset(s->sig + c, 0, w * sizeof(float)); memset(s->mask + c, 0, w); memset(s->adc + c, 0, w * 2);
        }
    }
    return 0;
}

/* Generates frame `frame`.  *out is malloc'ed (free with tpc_gen_free); returns 0, or -1 on failure. */
int tpc_gen_frame(const gen_config* cfg, uint32_t frame, gen_digit** out, uint64_t* n_out)
{
    if (!cfg || !out || !n_out || !cfg->n_sectors || !cfg->n_rows || !cfg->max_pads || !cfg->n_time) return -1;
    const uint32_t s0 = cfg->sector_begin, s1 = cfg->sector_end ? cfg->sector_end : cfg->n_sectors;
    if (s0 > s1 || s1 > cfg->n_sectors) return -1;
    const uint32_t n_planes = (s1 - s0) * cfg->n_rows;
    dvec_t* planes = (dvec_t*)calloc(n_planes ? n_planes : 1, sizeof(dvec_t));
    if (!planes) return -1;
    int fail = 0;
#ifdef _OPENMP
    if (cfg->n_threads) omp_set_num_threads((int)cfg->n_threads);
#endif
#pragma omp parallel
    {
        scratch_t s; memset(&s, 0, sizeof s);
        const size_t cells = (size_t)cfg->max_pads * cfg->n_time;
        s.sig = (float*)calloc(cells, sizeof(float));
        s.mask = (uint8_t*)calloc(cells + 8, 1);
        s.adc = (uint16_t*)calloc(cells, sizeof(uint16_t));
        if (!s.sig || !s.mask || !s.adc) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp barrier
        if (!fail) {
#pragma omp for schedule(dynamic, 1)
            for (long pl = 0; pl < (long)n_planes; ++pl) {
                const uint32_t sector = s0 + (uint32_t)pl / cfg->n_rows, row = (uint32_t)pl % cfg->n_rows;
                if (gen_plane(cfg, frame, sector, row, &s, &planes[pl])) {
#pragma omp atomic write
                    fail = 1;
                }
            }
        }
        free(s.sig); free(s.mask); free(s.adc); free(s.rects);
    }
    uint64_t total = 0;
    for (uint32_t pl = 0; pl < n_planes; ++pl) total += planes[pl].n;
    gen_digit* all = fail ? NULL : (gen_digit*)malloc((total ? total : 1) * sizeof(gen_digit));
    if (!all) fail = 1;
    uint64_t off = 0;
    for (uint32_t pl = 0; pl < n_planes; ++pl) {
        if (!fail && planes[pl].n) memcpy(all + off, planes[pl].d, planes[pl].n * sizeof(gen_digit));
        off += planes[pl].n;
        free(planes[pl].d);
    }
    free(planes);
    if (fail) { free(all); return -1; }
    *out = all; *n_out = total;
    return 0;
}

void tpc_gen_free(gen_digit* p) { free(p); }

/* FNV-1a-64 over the record bytes: dataset checksum printed in every report. */
uint64_t tpc_gen_checksum(const gen_digit* d, uint64_t n)
{
    const uint8_t* b = (const uint8_t*)d; uint64_t h = 0xcbf29ce484222325ull;
    for (uint64_t i = 0; i < n * sizeof(gen_digit); ++i) { h ^= b[i]; h *= 0x100000001b3ull; }
    return h;
}
