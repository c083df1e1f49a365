/*
 * oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.  See oracle.h for scope and citations.
 *
 * Per-spin checkerboard Metropolis for the square-lattice Ising and Blume-Capel models,
 * one int8 per site, no packing, no bit tricks, no blocking: every step is the literal
 * definition so that it can be checked against the paper (and DESIGN.md's readings) by eye.
 * The only parallelism is "rows of one colour are independent" (OpenMP over rows), which
 * is exactly what the checkerboard decomposition states.
 */
#include "oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------------------------ */
/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), from the definition:               */
/* one round maps (c0,c1,c2,c3),(k0,k1) to                                              */
/*   (hi(M1*c2) ^ c1 ^ k0,  lo(M1*c2),  hi(M0*c0) ^ c3 ^ k1,  lo(M0*c0))                  */
/* with M0 = 0xD2511F53, M1 = 0xCD9E8D57; the key is bumped by the Weyl constants        */
/* (0x9E3779B9, 0xBB67AE85) between rounds; ten rounds.                                  */
/* ------------------------------------------------------------------------------------ */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* ------------------------------------------------------------------------------------ */
/* RNG keying (BASELINE.json: keyed by (seed, sweep, colour,      */
/* site)).  key = (seed lo, seed hi); counter = (unit lo, unit hi, t, c | tag<<8 | k<<16). */
/* ------------------------------------------------------------------------------------ */
enum {
    TAG_INIT_PLANE = 0,  /* Ising start:      unit = P>>7, lane = P&127                       */
    TAG_INIT_QUAD  = 1,  /* Blume-Capel start: unit = P>>2, word = P&3                         */
    TAG_ACC_QUAD   = 2,  /* scheme 0:         unit = P>>2, u32 = word P&3                      */
    TAG_ACC_PLANE  = 3,  /* scheme 1:         unit = P>>7, plane k = 0..7, lane = P&127         */
    TAG_ACC_TAIL   = 4,  /* scheme 1:         unit = P,    tail = word 0                       */
    TAG_PROP_PLANE = 5   /* BC proposal bit:  unit = P>>7, lane = P&127                        */
};

static void keyed_block(uint64_t seed, uint64_t unit, uint32_t t, int colour, int tag, int k,
                        uint32_t out[4])
{
    uint32_t key[2] = { (uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { (uint32_t)(unit & 0xffffffffu), (uint32_t)(unit >> 32), t,
                        (uint32_t)colour | ((uint32_t)tag << 8) | ((uint32_t)k << 16) };
    oracle_philox4x32_10(ctr, key, out);
}

/* bit of lane l = P & 127 in a 128-bit block: bit (l & 31) of word (l >> 5) */
static int lane_bit(const uint32_t blk[4], uint64_t P)
{
    unsigned l = (unsigned)(P & 127u);
    return (int)((blk[l >> 5] >> (l & 31u)) & 1u);
}

uint32_t oracle_u32(uint64_t seed, int scheme, uint32_t t, int colour, uint64_t P)
{
    uint32_t blk[4];
    if (scheme == 0) {
        keyed_block(seed, P >> 2, t, colour, TAG_ACC_QUAD, 0, blk);
        return blk[P & 3u];
    }
    /* scheme 1: top 8 bits from 8 bit-planes shared by 128 sites (MSB first),
     * low 24 bits from a per-site tail block */
    uint32_t u = 0;
    for (int k = 0; k < 8; ++k) {
        keyed_block(seed, P >> 7, t, colour, TAG_ACC_PLANE, k, blk);
        u |= (uint32_t)lane_bit(blk, P) << (31 - k);
    }
    keyed_block(seed, P, t, colour, TAG_ACC_TAIL, 0, blk);
    u |= blk[0] >> 8;
    return u;
}

/* Scheme 2 ("plane + 56-bit tail", 64-bit thresholds): the same top byte
 * and the same tail block as scheme 1, but 56 tail bits instead of 24:
 *   u64 = top byte << 56 | (tail word 0 >> 8) << 32 | tail word 1.
 * Its top 32 bits are scheme 1's u32.  Lifts the 2^-32 floor on acceptance probabilities that
 * PAPER.md:159 mentions to 2^-64. */
uint64_t oracle_u64(uint64_t seed, uint32_t t, int colour, uint64_t P)
{
    uint32_t blk[4];
    uint64_t u = 0;
    for (int k = 0; k < 8; ++k) {
        keyed_block(seed, P >> 7, t, colour, TAG_ACC_PLANE, k, blk);
        u |= (uint64_t)lane_bit(blk, P) << (63 - k);
    }
    keyed_block(seed, P, t, colour, TAG_ACC_TAIL, 0, blk);
    u |= (uint64_t)(blk[0] >> 8) << 32;
    u |= (uint64_t)blk[1];
    return u;
}

int oracle_proposal_bit(uint64_t seed, uint32_t t, int colour, uint64_t P)
{
    uint32_t blk[4];
    keyed_block(seed, P >> 7, t, colour, TAG_PROP_PLANE, 0, blk);
    return lane_bit(blk, P);
}

int oracle_initial_spin(uint64_t seed, int model, uint32_t L, uint64_t i, uint64_t j)
{
    int colour = (int)((i + j) & 1u);
    uint64_t P = i * (uint64_t)(L / 2) + (j >> 1);
    uint32_t blk[4];
    if (model == ORACLE_ISING) {
        /* PAPER.md:65 fully disordered: sigma = +1 iff the site's INIT-plane bit is 1 */
        keyed_block(seed, P >> 7, 0, colour, TAG_INIT_PLANE, 0, blk);
        return lane_bit(blk, P) ? +1 : -1;
    }
    /* Blume-Capel: uniform on {-1,0,+1}: code = floor(3*u/2^32), sigma = code-1 */
    keyed_block(seed, P >> 2, 0, colour, TAG_INIT_QUAD, 0, blk);
    uint32_t u = blk[P & 3u];
    int code = (int)(((uint64_t)u * 3u) >> 32);
    return code - 1;
}

/* ------------------------------------------------------------------------------------ */
/* Thresholds: Metropolis acceptance min(1, exp(-beta*dE)) as a 32-bit integer compare   */
/* (PAPER.md:32-34, 159).  thr = floor(2^32 * exp(-beta*dE)) clamped to [0, 2^32];        */
/* accept iff (uint64)u32 < thr; dE <= 0 is stored as 2^32 ("always").                   */
/* ------------------------------------------------------------------------------------ */
static uint64_t threshold(double beta, double dE)
{
    if (dE <= 0.0) return (uint64_t)1 << 32;
    double p = exp(-(beta * dE));
    double x = floor(ldexp(p, 32));
    if (!(x > 0.0)) return 0;
    if (x >= 4294967296.0) return (uint64_t)1 << 32;
    return (uint64_t)x;
}

void oracle_thresholds(int model, double delta, double beta, uint64_t *out)
{
    if (model == ORACLE_ISING) {
        /* dE = 2*sigma*h; positive values 4 and 8 (J = 1, Eq. 1 in the Delta -> -inf limit) */
        out[0] = threshold(beta, 4.0);
        out[1] = threshold(beta, 8.0);
        return;
    }
    for (int code = 0; code < 3; ++code)
        for (int b = 0; b < 2; ++b)
            for (int h = -4; h <= 4; ++h) {
                int s = code - 1;
                int code2 = (code + 1 + b) % 3;     /* one of the two other values */
                int s2 = code2 - 1;
                /* Eq. (1): dE = -(s2 - s)*h + Delta*(s2^2 - s^2) */
                double dE = (double)(s - s2) * (double)h + delta * (double)(s2 * s2 - s * s);
                out[(code * 2 + b) * 9 + (h + 4)] = threshold(beta, dE);
            }
}

/* 64-bit thresholds (scheme 2): thr = floor(2^64 * exp(-beta*dE)); *always = 1 when dE <= 0 or
 * the product rounds to 2^64 (then thr is meaningless).  exp() carries 53 significant bits and
 * the scaling is exact, so floor(thr / 2^32) equals the 32-bit threshold of the same dE. */
static uint64_t threshold64(double beta, double dE, unsigned char *always)
{
    *always = 0;
    if (dE <= 0.0) { *always = 1; return 0; }
    double p = exp(-(beta * dE));
    double x = floor(ldexp(p, 64));
    if (!(x > 0.0)) return 0;
    if (x >= 18446744073709551616.0) { *always = 1; return 0; }
    return (uint64_t)x;
}

void oracle_thresholds64(int model, double delta, double beta, uint64_t *thr, unsigned char *always)
{
    if (model == ORACLE_ISING) {
        thr[0] = threshold64(beta, 4.0, &always[0]);
        thr[1] = threshold64(beta, 8.0, &always[1]);
        return;
    }
    for (int code = 0; code < 3; ++code)
        for (int b = 0; b < 2; ++b)
            for (int h = -4; h <= 4; ++h) {
                int s = code - 1;
                int code2 = (code + 1 + b) % 3;
                int s2 = code2 - 1;
                double dE = (double)(s - s2) * (double)h + delta * (double)(s2 * s2 - s * s);
                int e = (code * 2 + b) * 9 + (h + 4);
                thr[e] = threshold64(beta, dE, &always[e]);
            }
}

/* ------------------------------------------------------------------------------------ */
/* Lattice                                                                                */
/* ------------------------------------------------------------------------------------ */
struct oracle_lattice {
    uint32_t Lg;          /* side of the global periodic lattice                          */
    uint32_t h, w;        /* window extent (== Lg, Lg for the whole lattice)              */
    uint64_t i0, j0;      /* global coordinates of window site (0,0)                      */
    int model;
    double delta;
    uint64_t seed;
    int scheme;
    uint64_t t;
    int outside;          /* value of frozen sites outside a window                       */
    int8_t *s;            /* [h][w]                                                       */
};

static int g_threads = 1;

void oracle_set_threads(int n)
{
    if (n < 1) n = 1;
    g_threads = n;
}

int oracle_get_threads(void)
{
#ifdef _OPENMP
    return g_threads;
#else
    return 1;
#endif
}

static int valid_model(int model) { return model == ORACLE_ISING || model == ORACLE_BLUME_CAPEL; }

int oracle_create(oracle_lattice_t **out, uint32_t L, int model, double delta, uint64_t seed)
{
    if (!out || L < 2 || (L & 1u) || !valid_model(model) || !isfinite(delta)) return ORACLE_EINVAL;
    oracle_lattice_t *lat = (oracle_lattice_t *)calloc(1, sizeof *lat);
    if (!lat) return ORACLE_ENOMEM;
    lat->Lg = L; lat->h = L; lat->w = L; lat->i0 = 0; lat->j0 = 0;
    lat->model = model; lat->delta = delta; lat->seed = seed; lat->scheme = 1; lat->t = 0;
    lat->outside = 0;
    lat->s = (int8_t *)malloc((size_t)L * L);
    if (!lat->s) { free(lat); return ORACLE_ENOMEM; }
    for (uint64_t i = 0; i < L; ++i)
        for (uint64_t j = 0; j < L; ++j)
            lat->s[i * L + j] = (int8_t)oracle_initial_spin(seed, model, L, i, j);
    *out = lat;
    return ORACLE_OK;
}

int oracle_window_create(oracle_lattice_t **out, uint32_t Lg, int model, double delta,
                         uint64_t seed, int scheme, uint64_t t0, uint64_t i0, uint64_t j0,
                         uint32_t h, uint32_t w, const int8_t *spins, int outside)
{
    if (!out || Lg < 2 || (Lg & 1u) || !valid_model(model) || !isfinite(delta)) return ORACLE_EINVAL;
    if (h < 1 || w < 1 || h > Lg || w > Lg || i0 >= Lg || j0 >= Lg || !spins) return ORACLE_EINVAL;
    if (scheme < 0 || scheme > 2) return ORACLE_EINVAL;
    if (outside < -1 || outside > 1 || (model == ORACLE_ISING && outside == 0)) return ORACLE_EINVAL;
    oracle_lattice_t *lat = (oracle_lattice_t *)calloc(1, sizeof *lat);
    if (!lat) return ORACLE_ENOMEM;
    lat->Lg = Lg; lat->h = h; lat->w = w; lat->i0 = i0; lat->j0 = j0;
    lat->model = model; lat->delta = delta; lat->seed = seed; lat->scheme = scheme; lat->t = t0;
    lat->outside = outside;
    lat->s = (int8_t *)malloc((size_t)h * w);
    if (!lat->s) { free(lat); return ORACLE_ENOMEM; }
    memcpy(lat->s, spins, (size_t)h * w);
    *out = lat;
    return ORACLE_OK;
}

int oracle_set_rng_scheme(oracle_lattice_t *lat, int scheme)
{
    if (!lat || scheme < 0 || scheme > 2) return ORACLE_EINVAL;
    if (lat->t != 0) return ORACLE_ESTATE;
    lat->scheme = scheme;
    return ORACLE_OK;
}

uint64_t oracle_time(const oracle_lattice_t *lat) { return lat ? lat->t : 0; }

int oracle_destroy(oracle_lattice_t *lat)
{
    if (!lat) return ORACLE_EINVAL;
    free(lat->s);
    free(lat);
    return ORACLE_OK;
}

/* spin at window coordinates (a, b), which may be one step outside [0,h) x [0,w) */
static int spin_at(const oracle_lattice_t *lat, int64_t a, int64_t b)
{
    if (a < 0 || a >= (int64_t)lat->h) {
        if (lat->h != lat->Lg) return lat->outside;         /* frozen outside the window */
        a = (a + lat->h) % lat->h;                          /* periodic    */
    }
    if (b < 0 || b >= (int64_t)lat->w) {
        if (lat->w != lat->Lg) return lat->outside;
        b = (b + lat->w) % lat->w;
    }
    return lat->s[(uint64_t)a * lat->w + (uint64_t)b];
}

int oracle_half_sweep(oracle_lattice_t *lat, int colour, double beta)
{
    if (!lat || (colour != 0 && colour != 1) || isnan(beta) || beta < 0.0) return ORACLE_EINVAL;
    if (lat->t >= 0xffffffffull) return ORACLE_EINVAL;
    uint64_t thr[54], thr64[54];
    unsigned char alw64[54];
    oracle_thresholds(lat->model, lat->delta, beta, thr);
    oracle_thresholds64(lat->model, lat->delta, beta, thr64, alw64);
    const uint32_t t = (uint32_t)lat->t;
    const uint64_t half = lat->Lg / 2;

    /* sites of one colour do not interact: any order (here: rows in parallel) */
#pragma omp parallel for schedule(static) num_threads(g_threads)
    for (int64_t a = 0; a < (int64_t)lat->h; ++a) {
        uint64_t gi = (lat->i0 + (uint64_t)a) % lat->Lg;
        for (int64_t b = 0; b < (int64_t)lat->w; ++b) {
            uint64_t gj = (lat->j0 + (uint64_t)b) % lat->Lg;
            if ((int)((gi + gj) & 1u) != colour) continue;
            uint64_t P = gi * half + (gj >> 1);
            int s = lat->s[(uint64_t)a * lat->w + (uint64_t)b];
            /* 1. neighbour sum from the current array (white sees the new black spins) */
            int hsum = spin_at(lat, a - 1, b) + spin_at(lat, a + 1, b) +
                       spin_at(lat, a, b - 1) + spin_at(lat, a, b + 1);
            uint64_t th;
            int s_new, entry = -1;           /* entry: index into the tables, -1: dE <= 0 (Ising) */
            if (lat->model == ORACLE_ISING) {
                /* 2. dE = 2*sigma*h in {-8,-4,0,4,8} */
                int dE = 2 * s * hsum;
                th = dE <= 0 ? ((uint64_t)1 << 32) : (dE == 4 ? thr[0] : thr[1]);
                if (dE > 0) entry = dE == 4 ? 0 : 1;
                s_new = -s;
            } else {
                int bit = oracle_proposal_bit(lat->seed, t, colour, P);
                int code = s + 1;
                int code2 = (code + 1 + bit) % 3;
                s_new = code2 - 1;
                entry = (code * 2 + bit) * 9 + (hsum + 4);
                th = thr[entry];
            }
            int accept;
            if (lat->scheme == 2) {
                /* 3'. 64-bit compare: accept iff dE <= 0 / "always", or u64 < thr64 */
                if (entry < 0 || alw64[entry]) accept = 1;
                else accept = oracle_u64(lat->seed, t, colour, P) < thr64[entry];
            } else {
                /* 3. accept iff dE <= 0 (th = 2^32) or u32 < th */
                uint32_t u = oracle_u32(lat->seed, lat->scheme, t, colour, P);
                accept = (uint64_t)u < th;
            }
            if (accept) lat->s[(uint64_t)a * lat->w + (uint64_t)b] = (int8_t)s_new;
        }
    }
    return ORACLE_OK;
}

int oracle_sweep(oracle_lattice_t *lat, uint64_t n, const double *beta)
{
    if (!lat || (n && !beta)) return ORACLE_EINVAL;
    if (lat->t + n >= 0x100000000ull) return ORACLE_EINVAL;
    for (uint64_t k = 0; k < n; ++k)
        if (isnan(beta[k]) || beta[k] < 0.0) return ORACLE_EINVAL;
    for (uint64_t k = 0; k < n; ++k) {
        int rc = oracle_half_sweep(lat, 0, beta[k]);      /* black = (i+j) even first */
        if (rc) return rc;
        rc = oracle_half_sweep(lat, 1, beta[k]);
        if (rc) return rc;
        lat->t += 1;
    }
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------ */
/* Measurements by the literal double loops (Eq. 2: sum over pairs at separation r).      */
/*   M = sum sigma, Q = sum sigma^2,                                                      */
/*   Sx(r) = sum_{i,j} sigma(i,j) sigma(i,j+r),  Sy(r) = sum_{i,j} sigma(i,j) sigma(i+r,j)  */
/* over base rows i in [i0, i0+n_rows), all j, r = 1..r_max, periodic.                    */
/* ------------------------------------------------------------------------------------ */
int oracle_measure_rows(oracle_lattice_t *lat, uint64_t i0, uint64_t n_rows, uint32_t r_max,
                        int64_t *M, int64_t *Q, int64_t *Sx, int64_t *Sy)
{
    if (!lat || lat->h != lat->Lg || lat->w != lat->Lg) return ORACLE_EINVAL;
    const uint64_t L = lat->Lg;
    if (r_max < 1 || r_max > L - 1 || i0 >= L || n_rows > L || i0 + n_rows > L) return ORACLE_EINVAL;
    if (!M || !Q || !Sx || !Sy) return ORACLE_EINVAL;
    int64_t m = 0, q = 0;
#pragma omp parallel for reduction(+ : m, q) schedule(static) num_threads(g_threads)
    for (int64_t i = (int64_t)i0; i < (int64_t)(i0 + n_rows); ++i)
        for (uint64_t j = 0; j < L; ++j) {
            int s = lat->s[(uint64_t)i * L + j];
            m += s;
            q += s * s;
        }
    for (uint32_t r = 1; r <= r_max; ++r) {
        int64_t sx = 0, sy = 0;
#pragma omp parallel for reduction(+ : sx, sy) schedule(static) num_threads(g_threads)
        for (int64_t i = (int64_t)i0; i < (int64_t)(i0 + n_rows); ++i)
            for (uint64_t j = 0; j < L; ++j) {
                int s = lat->s[(uint64_t)i * L + j];
                sx += s * lat->s[(uint64_t)i * L + (j + r) % L];
                sy += s * lat->s[(((uint64_t)i + r) % L) * L + j];
            }
        Sx[r - 1] = sx;
        Sy[r - 1] = sy;
    }
    *M = m;
    *Q = q;
    return ORACLE_OK;
}

int oracle_measure(oracle_lattice_t *lat, uint32_t r_max, int64_t *M, int64_t *Q, int64_t *Sx,
                   int64_t *Sy)
{
    if (!lat) return ORACLE_EINVAL;
    return oracle_measure_rows(lat, 0, lat->Lg, r_max, M, Q, Sx, Sy);
}

/* Run n sweeps at constant beta and record, after each one, M, the bond sum Sx(1)+Sy(1), Q,
 * and (for lattices of at most 16 sites) the configuration as a base-3 number with digit
 * sigma+1 for site i*L+j at position i*L+j.  For the stationary-law pins on tiny lattices. */
int oracle_run_series(oracle_lattice_t *lat, uint64_t n, double beta, int64_t *M, int64_t *B,
                      int64_t *Q, int64_t *state)
{
    if (!lat || lat->h != lat->Lg || lat->w != lat->Lg || !M || !B || !Q) return ORACLE_EINVAL;
    const uint64_t L = lat->Lg;
    if (state && L * L > 16) return ORACLE_EINVAL;
    for (uint64_t k = 0; k < n; ++k) {
        int rc = oracle_sweep(lat, 1, &beta);
        if (rc) return rc;
        int64_t sx, sy;
        if (L >= 2) {
            /* r = 1 is legal for every even L >= 2 (L = 2: the wrap doubles each bond) */
            rc = oracle_measure_rows(lat, 0, L, 1, &M[k], &Q[k], &sx, &sy);
            if (rc) return rc;
            B[k] = sx + sy;
        }
        if (state) {
            int64_t code = 0, pw = 1;
            for (uint64_t x = 0; x < L * L; ++x) { code += pw * (lat->s[x] + 1); pw *= 3; }
            state[k] = code;
        }
    }
    return ORACLE_OK;
}

/* sum_k a[k]*b[(k+shift) mod n]: one row pair of Eq. (2), for spot checks on lattices too
 * large to hold unpacked (y axis: rows i and i+r, shift 0; x axis: the same row, shift r) */
int64_t oracle_pair_sum(const int8_t *a, const int8_t *b, uint64_t n, uint64_t shift)
{
    int64_t acc = 0;
    for (uint64_t k = 0; k < n; ++k) acc += (int64_t)a[k] * (int64_t)b[(k + shift) % n];
    return acc;
}

/* windows of unpacked spins, global coordinates, periodic wrap (whole lattices only) */
int oracle_get_spins(oracle_lattice_t *lat, uint64_t i0, uint64_t j0, uint32_t h, uint32_t w,
                     int8_t *out)
{
    if (!lat || !out) return ORACLE_EINVAL;
    if (lat->h != lat->Lg || lat->w != lat->Lg) {
        /* a window lattice only hands back a sub-window given in its own local coordinates */
        if (i0 + h > lat->h || j0 + w > lat->w) return ORACLE_EINVAL;
        for (uint32_t a = 0; a < h; ++a)
            for (uint32_t b = 0; b < w; ++b)
                out[(uint64_t)a * w + b] = lat->s[(i0 + a) * lat->w + (j0 + b)];
        return ORACLE_OK;
    }
    const uint64_t L = lat->Lg;
    if (h > L || w > L || i0 >= L || j0 >= L) return ORACLE_EINVAL;
    for (uint32_t a = 0; a < h; ++a)
        for (uint32_t b = 0; b < w; ++b)
            out[(uint64_t)a * w + b] = lat->s[((i0 + a) % L) * L + (j0 + b) % L];
    return ORACLE_OK;
}

int oracle_set_spins(oracle_lattice_t *lat, uint64_t i0, uint64_t j0, uint32_t h, uint32_t w,
                     const int8_t *in)
{
    if (!lat || !in || lat->h != lat->Lg || lat->w != lat->Lg) return ORACLE_EINVAL;
    const uint64_t L = lat->Lg;
    if (h > L || w > L || i0 >= L || j0 >= L) return ORACLE_EINVAL;
    for (uint64_t k = 0; k < (uint64_t)h * w; ++k) {
        int v = in[k];
        if (v < -1 || v > 1 || (lat->model == ORACLE_ISING && v == 0)) return ORACLE_EINVAL;
    }
    for (uint32_t a = 0; a < h; ++a)
        for (uint32_t b = 0; b < w; ++b)
            lat->s[((i0 + a) % L) * L + (j0 + b) % L] = in[(uint64_t)a * w + b];
    return ORACLE_OK;
}

/* ------------------------------------------------------------------------------------ */
/* Derived quantities in fp64.                                                            */
/* Energy density: e = -[Sx(1)+Sy(1)]/L^2 + Delta*Q/L^2  (Eq. 1 per site; Eq. 3 with the   */
/* sign fixed by E_eq = -sqrt(2)).                                           */
/* xi = I2/I1 (Eq. C1) for a single run: C(r) = (Sx+Sy)/(2 L^2); r_cut = (first r with     */
/* Sx+Sy <= 0) - 1, or r_max; trapezoid in r with half weight at r_cut; ascending sums.    */
/* ------------------------------------------------------------------------------------ */
double oracle_energy(const int64_t *Sx, const int64_t *Sy, int64_t Q, double delta, uint32_t L)
{
    double n = (double)L * (double)L;
    return -((double)(Sx[0] + Sy[0])) / n + delta * (double)Q / n;
}

double oracle_xi(const int64_t *Sx, const int64_t *Sy, uint32_t r_max, int64_t Q, uint32_t L,
                 uint32_t *r_cut_out)
{
    (void)Q;   /* C(0) = Q/L^2 multiplies r^n = 0 for n >= 1 */
    uint32_t r_cut = r_max;
    for (uint32_t r = 1; r <= r_max; ++r)
        if (Sx[r - 1] + Sy[r - 1] <= 0) { r_cut = r - 1; break; }
    if (r_cut_out) *r_cut_out = r_cut;
    if (r_cut < 1) return 0.0;
    double norm = 2.0 * (double)L * (double)L;
    double I1 = 0.0, I2 = 0.0;
    for (uint32_t r = 1; r <= r_cut; ++r) {
        double C = (double)(Sx[r - 1] + Sy[r - 1]) / norm;
        double wgt = (r == r_cut) ? 0.5 : 1.0;
        I1 += wgt * (double)r * C;
        I2 += wgt * (double)r * (double)r * C;
    }
    return I2 / I1;
}
