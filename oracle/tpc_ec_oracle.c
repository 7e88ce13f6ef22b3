/*
 * tpc_ec_oracle.c — CPU ORACLE of the TPC-EC v1 entropy coder.  TEST INFRASTRUCTURE, NOT PRODUCT (see tpc_ec_oracle.h
 * for the definition it follows, letter by letter: (Q) symbol streams, (N) statistics, (C) lane coder, (F) container;
 * step named in PAPER.md:55, 57).  Plain C, single thread, no blocking or reordering beyond what the definition states.
 * Pins: tests/test_ec_oracle_pins.py (hand-evaluated coder steps and symbol bytes in tests/golden/ec_examples.txt, an
 * independent decoder and container parser in another language, the information-content identity of rANS, closed-form
 * normalisations, degenerate streams, round trips).  No function here is "parity unpinned".
 */
#include "tpc_ec_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#define N_STREAMS 13u
#define BLOCK_SYMS 16384u
#define LANES 32u
#define PROB_BITS 12u
#define PROB_SCALE 4096u
#define RANS_L (1u << 23)

static float clamp255(float v) { return fminf(fmaxf(v, 0.0f), 255.0f); }

/* (Q) */
uint32_t tpc_ec_oracle_symbolize(const tpc_ec_oracle_cluster* cl, uint64_t n, uint32_t n_sectors, uint32_t n_rows,
                                 uint8_t* streams)
{
    uint32_t err = 0;
    for (uint64_t i = 0; i < n; ++i) {
        const tpc_ec_oracle_cluster* c = &cl[i];
        int same = 0;
        if (c->sector >= n_sectors || c->row >= n_rows) err |= TPC_EC_ORACLE_ERR_UNSORTED;
        if (i > 0) {
            const tpc_ec_oracle_cluster* p = &cl[i - 1];
            const uint64_t kp = ((uint64_t)p->sector << 32) | ((uint64_t)p->row << 24) | ((uint64_t)p->pad << 16) | p->time;
            const uint64_t kc = ((uint64_t)c->sector << 32) | ((uint64_t)c->row << 24) | ((uint64_t)c->pad << 16) | c->time;
            if (kp >= kc) err |= TPC_EC_ORACLE_ERR_UNSORTED;
            same = p->sector == c->sector && p->row == c->row;
        }
        const uint32_t dpad = same ? (uint32_t)(uint8_t)(c->pad - cl[i - 1].pad) : c->pad;
        const uint32_t v = (same && c->pad == cl[i - 1].pad) ? (uint32_t)(uint16_t)(c->time - cl[i - 1].time) : c->time;
        const uint32_t dq = (c->qtot - (uint32_t)c->qmax) & 0xffffffu;
        if (c->qtot < c->qmax || c->qtot - (uint32_t)c->qmax >= (1u << 24)) err |= TPC_EC_ORACLE_ERR_QTOT;
        streams[0 * n + i] = (uint8_t)dpad;
        streams[1 * n + i] = (uint8_t)(v & 255u);
        streams[2 * n + i] = (uint8_t)(v >> 8);
        streams[3 * n + i] = (uint8_t)(c->qmax & 255u);
        streams[4 * n + i] = (uint8_t)(c->qmax >> 8);
        streams[5 * n + i] = (uint8_t)(dq & 255u);
        streams[6 * n + i] = (uint8_t)((dq >> 8) & 255u);
        streams[7 * n + i] = (uint8_t)(dq >> 16);
        streams[8 * n + i] = c->flags;
        {   /* fp32, one rounding per operation (no contraction: there is no multiply-add pattern here) */
            volatile float a = c->pad_mean - (float)c->pad;
            volatile float b = a + 2.0f;
            volatile float d = b * 64.0f;
            streams[9 * n + i] = (uint8_t)clamp255(rintf(d));
            a = c->time_mean - (float)c->time;
            b = a + 2.0f;
            d = b * 64.0f;
            streams[10 * n + i] = (uint8_t)clamp255(rintf(d));
            d = c->sigma_pad * 128.0f;
            streams[11 * n + i] = (uint8_t)clamp255(rintf(d));
            d = c->sigma_time * 128.0f;
            streams[12 * n + i] = (uint8_t)clamp255(rintf(d));
        }
    }
    return err;
}

/* (N) */
void tpc_ec_oracle_normalize(const uint64_t hist[256], uint16_t freq[256])
{
    uint64_t n = 0;
    uint32_t f[256];
    for (int s = 0; s < 256; ++s) n += hist[s];
    if (n == 0) { memset(freq, 0, 256 * sizeof(uint16_t)); return; }
    long long D = PROB_SCALE;
    for (int s = 0; s < 256; ++s) {
        if (hist[s] == 0) f[s] = 0;
        else {
            /* hist[s] * 4096 / n without overflow: hist < 2^52 in any use; split to be safe */
            const uint64_t q = (hist[s] / n) * PROB_SCALE + ((hist[s] % n) * PROB_SCALE) / n;
            f[s] = q < 1 ? 1u : (uint32_t)q;
        }
        D -= f[s];
    }
    if (D > 0) {
        int a = 0;
        for (int s = 1; s < 256; ++s) if (hist[s] > hist[a]) a = s;   /* strict: lowest symbol on ties */
        f[a] += (uint32_t)D;
    }
    while (D < 0) {
        int b = 0;
        for (int s = 1; s < 256; ++s) if (f[s] > f[b]) b = s;
        long long d = -D < (long long)f[b] - 1 ? -D : (long long)f[b] - 1;
        f[b] -= (uint32_t)d;
        D += d;
    }
    for (int s = 0; s < 256; ++s) freq[s] = (uint16_t)f[s];
}

static void cumulate(const uint16_t freq[256], uint32_t cum[257])
{
    cum[0] = 0;
    for (int s = 0; s < 256; ++s) cum[s + 1] = cum[s] + freq[s];
}

/* (C) encoder */
uint32_t tpc_ec_oracle_lane_encode(const uint8_t* sym, uint64_t m, uint64_t stride, const uint16_t freq[256],
                                   uint8_t* bytes, uint32_t* nbytes)
{
    uint32_t cum[257];
    cumulate(freq, cum);
    uint32_t x = RANS_L, nb = 0;
    for (uint64_t k = m; k-- > 0;) {
        const uint32_t s = sym[k * stride];
        const uint32_t f = freq[s], c = cum[s];
        const uint64_t x_max = (uint64_t)((RANS_L >> PROB_BITS) << 8) * f;   /* 2^19 * f, up to 2^31 */
        while ((uint64_t)x >= x_max) {
            bytes[nb++] = (uint8_t)(x & 255u);
            x >>= 8;
        }
        x = (x / f) * PROB_SCALE + (x % f) + c;
    }
    *nbytes = nb;
    return x;
}

/* (C) decoder */
uint32_t tpc_ec_oracle_lane_decode(uint32_t state, const uint8_t* bytes, uint32_t nbytes, const uint16_t freq[256],
                                   uint8_t* sym, uint64_t m, uint64_t stride)
{
    uint32_t cum[257];
    cumulate(freq, cum);
    uint32_t x = state, ptr = nbytes;
    for (uint64_t k = 0; k < m; ++k) {
        const uint32_t slot = x & (PROB_SCALE - 1u);
        uint32_t s = 0;
        while (s < 255u && !(cum[s] <= slot && slot < cum[s + 1])) ++s;
        if (!(cum[s] <= slot && slot < cum[s + 1])) return TPC_EC_ORACLE_ERR_CONTAINER;
        sym[k * stride] = (uint8_t)s;
        x = freq[s] * (x >> PROB_BITS) + slot - cum[s];
        while (x < RANS_L) {
            if (ptr == 0) return TPC_EC_ORACLE_ERR_CONTAINER;
            x = (x << 8) | bytes[--ptr];
        }
    }
    return (x == RANS_L && ptr == 0) ? 0u : TPC_EC_ORACLE_ERR_CONTAINER;
}

/* number of symbols lane l of block b owns in a stream of n symbols */
static uint64_t lane_count(uint64_t n, uint64_t b, uint32_t l)
{
    const uint64_t first = b * BLOCK_SYMS + l;
    if (first >= n) return 0;
    uint64_t m = (n - first + LANES - 1) / LANES;
    return m > BLOCK_SYMS / LANES ? BLOCK_SYMS / LANES : m;
}

static uint64_t align_up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }

uint64_t tpc_ec_oracle_max_bytes(uint32_t n_sectors, uint32_t n_rows, uint64_t n)
{
    const uint64_t planes = (uint64_t)n_sectors * n_rows, nb = (n + BLOCK_SYMS - 1) / BLOCK_SYMS;
    /* 12 bits per symbol at most (f >= 1), plus less than one extra byte per lane from the state's slack */
    return align_up(64 + 4 * planes + 2 * 256 * N_STREAMS, 8) + 8 * (N_STREAMS * nb + 1) +
           N_STREAMS * nb * (LANES * 6 + LANES * 2 + 4) + N_STREAMS * ((n * 3 + 1) / 2);
}

static void put32(uint8_t* p, uint32_t v) { p[0] = (uint8_t)v; p[1] = (uint8_t)(v >> 8); p[2] = (uint8_t)(v >> 16); p[3] = (uint8_t)(v >> 24); }
static void put64(uint8_t* p, uint64_t v) { put32(p, (uint32_t)v); put32(p + 4, (uint32_t)(v >> 32)); }
static void put16(uint8_t* p, uint32_t v) { p[0] = (uint8_t)v; p[1] = (uint8_t)(v >> 8); }
static uint32_t get32(const uint8_t* p) { return (uint32_t)p[0] | ((uint32_t)p[1] << 8) | ((uint32_t)p[2] << 16) | ((uint32_t)p[3] << 24); }
static uint64_t get64(const uint8_t* p) { return (uint64_t)get32(p) | ((uint64_t)get32(p + 4) << 32); }
static uint32_t get16(const uint8_t* p) { return (uint32_t)p[0] | ((uint32_t)p[1] << 8); }

/* (F) encoder */
uint64_t tpc_ec_oracle_encode(const tpc_ec_oracle_cluster* cl, uint64_t n, uint32_t n_sectors, uint32_t n_rows,
                              uint8_t* out, uint64_t capacity, uint32_t* err)
{
    const uint64_t planes = (uint64_t)n_sectors * n_rows, nb = (n + BLOCK_SYMS - 1) / BLOCK_SYMS;
    const uint64_t worst = tpc_ec_oracle_max_bytes(n_sectors, n_rows, n);
    uint8_t* streams = (uint8_t*)malloc(N_STREAMS * (n ? n : 1));
    uint8_t* buf = (uint8_t*)calloc(worst, 1);           /* built in a worst-case buffer, copied out if it fits */
    uint8_t* lane_bytes = (uint8_t*)malloc(3 * (BLOCK_SYMS / LANES) / 2 + 8);
    *err = 0;
    if (!streams || !buf || !lane_bytes) { free(streams); free(buf); free(lane_bytes); *err = TPC_EC_ORACLE_ERR_CAPACITY; return 0; }

    *err |= tpc_ec_oracle_symbolize(cl, n, n_sectors, n_rows, streams);

    const uint64_t off_counts = 64, off_freq = off_counts + 4 * planes;
    const uint64_t off_dir = align_up(off_freq + 2 * 256 * N_STREAMS, 8);
    uint64_t pos = off_dir + 8 * (N_STREAMS * nb + 1);

    /* plane counts */
    for (uint64_t i = 0; i < n; ++i) {
        if (cl[i].sector >= n_sectors || cl[i].row >= n_rows) continue;   /* flagged by symbolize */
        uint8_t* p = buf + off_counts + 4 * ((uint64_t)cl[i].sector * n_rows + cl[i].row);
        put32(p, get32(p) + 1);
    }
    /* statistics, then the records stream by stream, block by block */
    for (uint32_t s = 0; s < N_STREAMS; ++s) {
        uint64_t hist[256] = {0};
        uint16_t freq[256];
        const uint8_t* st = streams + (uint64_t)s * n;
        for (uint64_t i = 0; i < n; ++i) hist[st[i]]++;
        tpc_ec_oracle_normalize(hist, freq);
        for (int a = 0; a < 256; ++a) put16(buf + off_freq + 2 * (256 * (uint64_t)s + a), freq[a]);
        for (uint64_t b = 0; b < nb; ++b) {
            put64(buf + off_dir + 8 * (s * nb + b), pos);
            uint8_t* rec = buf + pos;
            uint64_t at = LANES * 4 + LANES * 2;
            for (uint32_t l = 0; l < LANES; ++l) {
                uint32_t nbytes = 0;
                const uint64_t m = lane_count(n, b, l);
                const uint32_t x = tpc_ec_oracle_lane_encode(st + b * BLOCK_SYMS + l, m, LANES, freq, lane_bytes, &nbytes);
                put32(rec + 4 * l, x);
                put16(rec + LANES * 4 + 2 * l, nbytes);
                memcpy(rec + at, lane_bytes, nbytes);
                at += nbytes;
            }
            pos += align_up(at, 4);
        }
    }
    put64(buf + off_dir + 8 * (N_STREAMS * nb), pos);
    put32(buf + 0, 0x45435054u); put32(buf + 4, 1u); put64(buf + 8, n);
    put32(buf + 16, n_sectors); put32(buf + 20, n_rows); put32(buf + 24, N_STREAMS); put32(buf + 28, BLOCK_SYMS);
    put32(buf + 32, (uint32_t)nb); put32(buf + 36, 0); put64(buf + 40, pos);
    if (pos <= capacity) memcpy(out, buf, pos); else *err |= TPC_EC_ORACLE_ERR_CAPACITY;
    free(streams); free(buf); free(lane_bytes);
    return pos;
}

/* (F) decoder, then the inverse of (Q) */
uint32_t tpc_ec_oracle_decode(const uint8_t* in, uint64_t bytes, tpc_ec_oracle_cluster* out, uint64_t capacity,
                              uint64_t* n_out)
{
    *n_out = 0;
    if (bytes < 64 || get32(in) != 0x45435054u || get32(in + 4) != 1u) return TPC_EC_ORACLE_ERR_CONTAINER;
    const uint64_t n = get64(in + 8);
    const uint32_t n_sectors = get32(in + 16), n_rows = get32(in + 20);
    const uint64_t planes = (uint64_t)n_sectors * n_rows, nb = (n + BLOCK_SYMS - 1) / BLOCK_SYMS;
    if (get32(in + 24) != N_STREAMS || get32(in + 28) != BLOCK_SYMS || get32(in + 32) != nb || get64(in + 40) != bytes)
        return TPC_EC_ORACLE_ERR_CONTAINER;
    const uint64_t off_counts = 64, off_freq = off_counts + 4 * planes;
    const uint64_t off_dir = align_up(off_freq + 2 * 256 * N_STREAMS, 8);
    if (off_dir + 8 * (N_STREAMS * nb + 1) > bytes) return TPC_EC_ORACLE_ERR_CONTAINER;
    *n_out = n;
    if (n > capacity) return TPC_EC_ORACLE_ERR_CAPACITY;

    uint8_t* streams = (uint8_t*)malloc(N_STREAMS * (n ? n : 1));
    if (!streams) return TPC_EC_ORACLE_ERR_CAPACITY;
    uint32_t err = 0;
    for (uint32_t s = 0; s < N_STREAMS && !err; ++s) {
        uint16_t freq[256];
        uint32_t total = 0;
        for (int a = 0; a < 256; ++a) { freq[a] = (uint16_t)get16(in + off_freq + 2 * (256 * (uint64_t)s + a)); total += freq[a]; }
        if (n > 0 && total != PROB_SCALE) { err = TPC_EC_ORACLE_ERR_CONTAINER; break; }
        for (uint64_t b = 0; b < nb && !err; ++b) {
            const uint64_t r0 = get64(in + off_dir + 8 * (s * nb + b)), r1 = get64(in + off_dir + 8 * (s * nb + b + 1));
            if (r0 > r1 || r1 > bytes || r1 - r0 < LANES * 6) { err = TPC_EC_ORACLE_ERR_CONTAINER; break; }
            const uint8_t* rec = in + r0;
            uint64_t at = LANES * 6;
            for (uint32_t l = 0; l < LANES; ++l) {
                const uint32_t x = get32(rec + 4 * l), nbytes = get16(rec + LANES * 4 + 2 * l);
                if (at + nbytes > r1 - r0) { err = TPC_EC_ORACLE_ERR_CONTAINER; break; }
                err |= tpc_ec_oracle_lane_decode(x, rec + at, nbytes, freq, streams + (uint64_t)s * n + b * BLOCK_SYMS + l,
                                                 lane_count(n, b, l), LANES);
                at += nbytes;
            }
        }
    }
    /* inverse of (Q): walk the planes in order; plane_count gives sector and row */
    if (!err) {
        uint64_t i = 0;
        for (uint64_t pl = 0; pl < planes && !err; ++pl) {
            const uint32_t cnt = get32(in + off_counts + 4 * pl);
            if (i + cnt > n) { err = TPC_EC_ORACLE_ERR_CONTAINER; break; }
            uint32_t pad = 0, time = 0;
            for (uint32_t j = 0; j < cnt; ++j, ++i) {
                const uint32_t dpad = streams[0 * n + i];
                const uint32_t v = streams[1 * n + i] | ((uint32_t)streams[2 * n + i] << 8);
                if (j == 0) { pad = dpad; time = v; }
                else if (dpad != 0) { pad += dpad; time = v; }
                else time += v;
                tpc_ec_oracle_cluster* c = &out[i];
                const uint32_t qmax = streams[3 * n + i] | ((uint32_t)streams[4 * n + i] << 8);
                const uint32_t dq = streams[5 * n + i] | ((uint32_t)streams[6 * n + i] << 8) | ((uint32_t)streams[7 * n + i] << 16);
                c->sector = (uint8_t)(pl / n_rows); c->row = (uint8_t)(pl % n_rows);
                c->pad = (uint8_t)pad; c->flags = streams[8 * n + i];
                c->time = (uint16_t)time; c->qmax = (uint16_t)qmax; c->qtot = qmax + dq;
                c->pad_mean = (float)(uint8_t)pad + ((float)streams[9 * n + i] - 128.0f) / 64.0f;
                c->time_mean = (float)(uint16_t)time + ((float)streams[10 * n + i] - 128.0f) / 64.0f;
                c->sigma_pad = (float)streams[11 * n + i] / 128.0f;
                c->sigma_time = (float)streams[12 * n + i] / 128.0f;
                c->rsv = 0;
            }
        }
        if (!err && i != n) err = TPC_EC_ORACLE_ERR_CONTAINER;
    }
    free(streams);
    return err;
}
