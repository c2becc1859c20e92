/*
 * Seeded synthetic TPC event generator (SURVEY.md 8(d) "Generator").
 *
 * This module is the ONLY code shared by the oracle's tests and the CUDA path's tests/bench.
 * It holds none of the tracker's arithmetic: it draws helices, intersects them with pad rows
 * and smears the crossings.  fp64 maths, fp32 output, own portable RNG (splitmix64-seeded
 * xoshiro256**), so a (config, seed) pair gives the same event on every box with this libm.
 *
 * Workload shape follows BASELINE.json:configs[0..4] (stand-ins for the ALICE raw data of
 * PAPER.md Table 2, which are not available): 36 sectors x 159 pad rows,
 * primaries from the origin, secondaries from r<50 cm, uniform noise, optional pile-up of
 * several events with z offsets.
 *
 * Plain C, no dependencies; built by datagen/__init__.py into datagen/libtpcgen.so.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define PI 3.14159265358979323846

typedef struct {
    int32_t n_sectors;        /* 36 (sector s<18: side A z>0, s>=18: side C z<0) */
    int32_t n_rows;           /* 159 */
    int32_t n_events;         /* 1, or 20 for the time frame (config 4) */
    int32_t n_primaries;      /* per event */
    int32_t n_secondaries;    /* per event, vertices uniform in r<50 cm, |vz|<50 cm */
    int32_t pt_mode;          /* 0: log-uniform 0.1..10 GeV/c; 1: 0.1 + Exp(scale 0.4) */
    int32_t single_sector;    /* config 0: only sector 0, phi0 in its 20 deg, eta folded, no edge cut */
    int32_t z_shift;          /* config 4: event e shifted by d_e~U(0,250) towards the readout */
    double  noise_frac;       /* noise clusters = noise_frac * track clusters */
    double  sigma;            /* Gaussian smear of y and z [cm] */
    double  bz;               /* Tesla */
    double  eta_max;          /* 0.9 */
    uint64_t seed;
} gen_config;

/* ---------------------------------------------------------------- RNG */
typedef struct { uint64_t s[4]; } rng_t;
static uint64_t splitmix64(uint64_t *x) {
    uint64_t z = (*x += 0x9E3779B97F4A7C15ULL);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
static void rng_seed(rng_t *r, uint64_t seed, uint64_t stream) {
    uint64_t x = seed * 0xD1342543DE82EF95ULL + stream * 0x2545F4914F6CDD1DULL + 0x1234567ULL;
    for (int i = 0; i < 4; i++) r->s[i] = splitmix64(&x);
}
static inline uint64_t rotl(uint64_t x, int k) { return (x << k) | (x >> (64 - k)); }
static uint64_t rng_next(rng_t *r) {
    uint64_t *s = r->s;
    uint64_t result = rotl(s[1] * 5, 7) * 9, t = s[1] << 17;
    s[2] ^= s[0]; s[3] ^= s[1]; s[1] ^= s[2]; s[0] ^= s[3]; s[2] ^= t; s[3] = rotl(s[3], 45);
    return result;
}
static double rng_uniform(rng_t *r) { return (double)(rng_next(r) >> 11) * (1.0 / 9007199254740992.0); }
static double rng_normal(rng_t *r) {
    double u1 = rng_uniform(r), u2 = rng_uniform(r);
    if (u1 < 1e-300) u1 = 1e-300;
    return sqrt(-2.0 * log(u1)) * cos(2.0 * PI * u2);
}
static uint64_t rng_below(rng_t *r, uint64_t n) { /* unbiased enough for shuffles: 64-bit multiply-high */
    return (uint64_t)(((__uint128_t)rng_next(r) * n) >> 64);
}

/* ---------------------------------------------------------------- geometry */
void tpcgen_default_row_x(int32_t n_rows, float *row_x) {
    /* rows 0-62 pitch 0.75 from 85.2; 63-126 pitch 1.0 from 135.0; 127-158 pitch 1.5 from 199.5 */
    for (int r = 0; r < n_rows; r++) {
        double x;
        if (r < 63) x = 85.2 + 0.75 * r;
        else if (r < 127) x = 135.0 + 1.0 * (r - 63);
        else x = 199.5 + 1.5 * (r - 127);
        row_x[r] = (float)x;
    }
}

typedef struct { int32_t sr; float y, z; int32_t truth; } clus_t;
typedef struct { clus_t *v; int64_t n, cap; } vec_t;
static void vec_push(vec_t *a, clus_t c) {
    if (a->n == a->cap) { a->cap = a->cap ? a->cap * 2 : (1 << 16); a->v = (clus_t *)realloc(a->v, a->cap * sizeof(clus_t)); }
    a->v[a->n++] = c;
}

typedef struct {
    vec_t clusters;
    int64_t n_track_clusters;
    int32_t n_tracks;
    /* per-track truth (global frame): vx,vy,vz,pt,q,phi0,eta,event,zshift_unused */
    double *trk; int64_t trk_cap;
} gen_state;

static void add_track(gen_state *g, const gen_config *cfg, const double *row_x, rng_t *r,
                      double vx, double vy, double vz, double pt, double q, double phi0, double eta,
                      int32_t truth_id, double zshift) {
    const double tan10 = tan(PI / 18.0);
    const double dphi = 2.0 * PI / 18.0;
    const double kappa = -q * 0.299792458e-2 * cfg->bz / pt;
    const double sk = kappa > 0 ? 1.0 : -1.0;
    const double shl = sinh(eta);
    for (int s = 0; s < cfg->n_sectors; s++) {
        if (cfg->single_sector && s != 0) continue;
        const double alpha = ((s % 18) + 0.5) * dphi;
        const double side = (s < 18) ? 1.0 : -1.0;
        const double ca = cos(alpha), sa = sin(alpha);
        const double vxl = vx * ca + vy * sa, vyl = -vx * sa + vy * ca;
        const double phil = phi0 - alpha;
        const double sp0 = sin(phil), cp0 = cos(phil);
        for (int row = 0; row < cfg->n_rows; row++) {
            const double xr = row_x[row];
            const double sr = sp0 + kappa * (xr - vxl);
            if (sr > 1.0 || sr < -1.0) continue;
            const double cr = sqrt(1.0 - sr * sr);
            const double ymax = xr * tan10;
            const double ya = vyl - (cr - cp0) / kappa, yb = vyl - (-cr - cp0) / kappa;
            if (!cfg->single_sector && fabs(ya) > ymax && fabs(yb) > ymax) continue; /* cheap reject */
            /* first crossing: smaller turning angle in (0,pi) of the two directions */
            double best_d = 1e30, best_y = 0;
            for (int c = 0; c < 2; c++) {
                const double cphi = c == 0 ? cr : -cr;
                const double phi = atan2(sr, cphi);
                double d = fmod((phi - phil) * sk, 2.0 * PI);
                if (d < 0) d += 2.0 * PI;
                if (d > 0 && d < PI && d < best_d) { best_d = d; best_y = c == 0 ? ya : yb; }
            }
            if (best_d > 1e29) continue;
            const double S = best_d / fabs(kappa);
            const double z = vz + S * shl;
            if (!cfg->single_sector && fabs(best_y) > ymax) continue;
            if (!(fabs(z) < 250.0)) continue;
            if (z * side < 0 || (z == 0 && side < 0)) continue;
            double ys = best_y + cfg->sigma * rng_normal(r);
            double zs = z + cfg->sigma * rng_normal(r);
            zs -= side * zshift;
            clus_t c = { s * cfg->n_rows + row, (float)ys, (float)zs, truth_id };
            vec_push(&g->clusters, c);
            g->n_track_clusters++;
        }
    }
}

static double draw_pt(const gen_config *cfg, rng_t *r) {
    if (cfg->pt_mode == 0) return 0.1 * pow(100.0, rng_uniform(r));
    double u = rng_uniform(r);
    if (u < 1e-300) u = 1e-300;
    return 0.1 - 0.4 * log(u);
}

typedef struct {
    int64_t n_clusters;
    int32_t n_tracks;
    int32_t *row_counts;   /* [n_sectors*n_rows] */
    float *y, *z;          /* [n_clusters], (sector,row)-major, shuffled within a row */
    int32_t *truth;        /* [n_clusters], -1 = noise */
    double *tracks;        /* [n_tracks*8]: vx,vy,vz,pt,q,phi0,eta,zshift */
} gen_event;

gen_event *tpcgen_generate(const gen_config *cfg, const float *row_x_f) {
    gen_state g; memset(&g, 0, sizeof(g));
    double *row_x = (double *)malloc(sizeof(double) * cfg->n_rows);
    for (int i = 0; i < cfg->n_rows; i++) row_x[i] = (double)row_x_f[i];
    const int tracks_per_event = cfg->n_primaries + cfg->n_secondaries;
    const int64_t n_tracks = (int64_t)tracks_per_event * cfg->n_events;
    double *trk = (double *)calloc((size_t)n_tracks * 8 + 8, sizeof(double));
    const int nsr = cfg->n_sectors * cfg->n_rows;

    for (int e = 0; e < cfg->n_events; e++) {
        rng_t re; rng_seed(&re, cfg->seed, 1000003ULL * (uint64_t)(e + 1));
        const double zshift = cfg->z_shift ? 250.0 * rng_uniform(&re) : 0.0;
        const int64_t first_cluster = g.clusters.n;
        for (int t = 0; t < tracks_per_event; t++) {
            const int32_t id = e * tracks_per_event + t;
            rng_t r; rng_seed(&r, cfg->seed, ((uint64_t)id << 8) | 7ULL);
            double vx = 0, vy = 0, vz = 0;
            if (t >= cfg->n_primaries) {
                double rv = 50.0 * sqrt(rng_uniform(&r)), pv = 2.0 * PI * rng_uniform(&r);
                vx = rv * cos(pv); vy = rv * sin(pv); vz = -50.0 + 100.0 * rng_uniform(&r);
            }
            double pt = draw_pt(cfg, &r);
            double q = rng_uniform(&r) < 0.5 ? -1.0 : 1.0;
            double phi0, eta = -cfg->eta_max + 2.0 * cfg->eta_max * rng_uniform(&r);
            if (cfg->single_sector) { phi0 = (PI / 9.0) * rng_uniform(&r); eta = fabs(eta); }
            else phi0 = 2.0 * PI * rng_uniform(&r);
            double *tp = trk + (size_t)id * 8;
            tp[0] = vx; tp[1] = vy; tp[2] = vz; tp[3] = pt; tp[4] = q; tp[5] = phi0; tp[6] = eta; tp[7] = zshift;
            add_track(&g, cfg, row_x, &r, vx, vy, vz, pt, q, phi0, eta, id, zshift);
        }
        /* noise for this event: fraction of this event's track clusters */
        const int64_t n_trk_cl = g.clusters.n - first_cluster;
        const int64_t n_noise = (int64_t)floor(cfg->noise_frac * (double)n_trk_cl + 0.5);
        const double tan10 = tan(PI / 18.0);
        for (int64_t i = 0; i < n_noise; i++) {
            int s = cfg->single_sector ? 0 : (int)rng_below(&re, (uint64_t)cfg->n_sectors);
            int row = (int)rng_below(&re, (uint64_t)cfg->n_rows);
            double ymax = row_x[row] * tan10;
            double y = (2.0 * rng_uniform(&re) - 1.0) * ymax;
            double z;
            if (cfg->z_shift) z = -250.0 + 500.0 * rng_uniform(&re);
            else z = ((s < 18) ? 1.0 : -1.0) * 250.0 * rng_uniform(&re);
            clus_t c = { s * cfg->n_rows + row, (float)y, (float)z, -1 };
            vec_push(&g.clusters, c);
        }
    }

    /* bucket by (sector,row), then Fisher-Yates per bucket so the load index carries no information */
    gen_event *ev = (gen_event *)calloc(1, sizeof(gen_event));
    const int64_t N = g.clusters.n;
    ev->n_clusters = N; ev->n_tracks = (int32_t)n_tracks; ev->tracks = trk;
    ev->row_counts = (int32_t *)calloc((size_t)nsr, sizeof(int32_t));
    ev->y = (float *)malloc(sizeof(float) * (size_t)(N + 1));
    ev->z = (float *)malloc(sizeof(float) * (size_t)(N + 1));
    ev->truth = (int32_t *)malloc(sizeof(int32_t) * (size_t)(N + 1));
    int64_t *off = (int64_t *)calloc((size_t)nsr + 1, sizeof(int64_t));
    for (int64_t i = 0; i < N; i++) ev->row_counts[g.clusters.v[i].sr]++;
    for (int i = 0; i < nsr; i++) off[i + 1] = off[i] + ev->row_counts[i];
    int64_t *cur = (int64_t *)malloc(sizeof(int64_t) * (size_t)nsr);
    memcpy(cur, off, sizeof(int64_t) * (size_t)nsr);
    for (int64_t i = 0; i < N; i++) {
        clus_t c = g.clusters.v[i];
        int64_t p = cur[c.sr]++;
        ev->y[p] = c.y; ev->z[p] = c.z; ev->truth[p] = c.truth;
    }
    for (int i = 0; i < nsr; i++) {
        rng_t r; rng_seed(&r, cfg->seed ^ 0xABCDEF12345ULL, (uint64_t)i + 17ULL);
        int64_t b = off[i], n = ev->row_counts[i];
        for (int64_t k = n - 1; k > 0; k--) {
            int64_t j = (int64_t)rng_below(&r, (uint64_t)(k + 1));
            float ty = ev->y[b + k]; ev->y[b + k] = ev->y[b + j]; ev->y[b + j] = ty;
            float tz = ev->z[b + k]; ev->z[b + k] = ev->z[b + j]; ev->z[b + j] = tz;
            int32_t tt = ev->truth[b + k]; ev->truth[b + k] = ev->truth[b + j]; ev->truth[b + j] = tt;
        }
    }
    free(cur); free(off); free(g.clusters.v); free(row_x);
    return ev;
}

int64_t tpcgen_n_clusters(const gen_event *e) { return e->n_clusters; }
int32_t tpcgen_n_tracks(const gen_event *e) { return e->n_tracks; }
void tpcgen_copy(const gen_event *e, int32_t n_sr, int32_t *row_counts, float *y, float *z, int32_t *truth, double *tracks) {
    memcpy(row_counts, e->row_counts, sizeof(int32_t) * (size_t)n_sr);
    memcpy(y, e->y, sizeof(float) * (size_t)e->n_clusters);
    memcpy(z, e->z, sizeof(float) * (size_t)e->n_clusters);
    memcpy(truth, e->truth, sizeof(int32_t) * (size_t)e->n_clusters);
    memcpy(tracks, e->tracks, sizeof(double) * (size_t)e->n_tracks * 8);
}
void tpcgen_free(gen_event *e) {
    if (!e) return;
    free(e->row_counts); free(e->y); free(e->z); free(e->truth); free(e->tracks); free(e);
}
