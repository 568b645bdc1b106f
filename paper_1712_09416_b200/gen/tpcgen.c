/*
 * tpcgen.c -- seeded synthetic TPC events (stand-in for the ALICE Pb-Pb / p-Pb data of PAPER.md:17,
 * which is not available).  Recipe: BASELINE.json configs (lines 7-11) as read in SURVEY.md 8(d).1 and
 * restated in DESIGN.md "Input recipe".
 *
 * This module is the ONE piece both the CPU oracle and the CUDA path are fed from.  It contains none of
 * the tracker's arithmetic: it draws helices, intersects them with the pad rows of every sector, smears,
 * drops, adds noise, shuffles, and hands out float32 SoA arrays plus truth labels.  Everything is done in
 * double and rounded once to float32.
 *
 * Geometry conventions: 36 sectors, s = 0..17 on the A side (z >= 0), s+18 on the C side
 * (z < 0); sector s is the 20 degree wedge centred on alpha_s = (20*(s mod 18) + 10) degrees; local frame =
 * global frame rotated by -alpha_s; a cluster of pad row r sits at local x = row_x[r] exactly.
 *
 * plain C, no dependencies beyond libm.  gcc -O2 -shared -fPIC.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define TPCGEN_PI 3.14159265358979323846
#define TPCGEN_K 0.00299792458 /* cm^-1 GeV T^-1 : curvature = K*Bz/pT */

typedef struct {
    int32_t n_sectors;      /* 36, or 1 (config 1: only sector 0 exists and all tracks are aimed into it) */
    int32_t n_rows;         /* 159 */
    const double* row_x;    /* [n_rows] cm */
    double tan_half_angle;  /* tan(10 deg) */
    double z_max;           /* 250 cm */
    double r_max;           /* 247 cm : a track ends when it leaves this radius */
    double bz;              /* Tesla */
    int32_t n_primaries;
    double frac_secondaries; /* n_sec = round(frac*n_prim); vertex r<50, |z|<50 */
    int32_t pt_mode;        /* 0: uniform [pt_a, pt_b];  1: pt_a + Exp(mean pt_b) */
    double pt_a, pt_b;
    double eta_max;
    double sigma_y, sigma_z;
    double inefficiency;    /* probability a crossing gives no cluster */
    double noise_frac;      /* noise clusters per sector = round(noise_frac * signal clusters of that sector) */
    int32_t loopers;        /* 0: outgoing branch only (turning angle < pi); 1: true loopers curl up to max_turns */
    int32_t max_turns;
    int32_t shuffle;        /* 1: shuffle clusters inside each sector */
} tpcgen_config;

typedef struct {
    int32_t n_clusters, n_tracks, n_sectors;
    int32_t* sector_offset; /* [n_sectors+1] */
    float *x, *y, *z;
    int32_t *row, *label;   /* label = track id or -1 */
    double* trk;            /* [n_tracks][TPCGEN_TRK_COLS] */
} tpcgen_event;

/* columns of the truth track table */
enum { TRK_PT = 0, TRK_CHARGE, TRK_ETA, TRK_PHI, TRK_VX, TRK_VY, TRK_VZ, TRK_PRIMARY, TPCGEN_TRK_COLS };

/* ---- counter-based random numbers: splitmix64 of (key, counter) ---- */
static uint64_t mix64(uint64_t z) {
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
typedef struct { uint64_t key, ctr; } rng_t;
static rng_t rng_make(uint64_t seed, uint64_t a, uint64_t b) {
    rng_t r;
    r.key = mix64(mix64(mix64(seed) ^ (a * 0xD1B54A32D192ED03ull)) ^ (b * 0x8CB92BA72F3D8DD7ull));
    r.ctr = 0;
    return r;
}
static double rng_u(rng_t* r) { /* uniform in (0,1) */
    uint64_t v = mix64(r->key + (r->ctr++) * 0x9E3779B97F4A7C15ull);
    return ((double)(v >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}
static double rng_normal(rng_t* r) {
    double u1 = rng_u(r), u2 = rng_u(r);
    return sqrt(-2.0 * log(u1)) * cos(2.0 * TPCGEN_PI * u2);
}

/* ---- growable cluster store, one per sector ---- */
typedef struct { int32_t n, cap; float *y, *z; int32_t *row, *label; } bucket_t;
static int bucket_push(bucket_t* b, float y, float z, int32_t row, int32_t label) {
    if (b->n == b->cap) {
        int32_t nc = b->cap ? 2 * b->cap : 1024;
        float* ny = (float*)realloc(b->y, sizeof(float) * nc);
        float* nz = (float*)realloc(b->z, sizeof(float) * nc);
        int32_t* nr = (int32_t*)realloc(b->row, sizeof(int32_t) * nc);
        int32_t* nl = (int32_t*)realloc(b->label, sizeof(int32_t) * nc);
        if (!ny || !nz || !nr || !nl) return -1;
        b->y = ny; b->z = nz; b->row = nr; b->label = nl; b->cap = nc;
    }
    b->y[b->n] = y; b->z[b->n] = z; b->row[b->n] = row; b->label[b->n] = label; b->n++;
    return 0;
}

static double wrap_2pi(double a) { /* into [0, 2pi) */
    a = fmod(a, 2.0 * TPCGEN_PI);
    if (a < 0) a += 2.0 * TPCGEN_PI;
    return a;
}

void tpcgen_free(tpcgen_event* ev) {
    if (!ev) return;
    free(ev->sector_offset); free(ev->x); free(ev->y); free(ev->z); free(ev->row); free(ev->label); free(ev->trk);
    free(ev);
}

/*
 * Generate one event.  Returns NULL on allocation failure or bad config.
 * Helix: circle of radius R = pT/(K|Bz|) through the vertex with initial direction
 * (cos phi, sin phi); h = -charge*sign(Bz), h = +1 turns counter-clockwise; centre = (vx - h R sin phi,
 * vy + h R cos phi); position at turning angle theta >= 0: c + R (cos psi, sin psi), psi = psi0 + h theta;
 * z = vz + t * R * theta with t = sinh(eta).
 */
tpcgen_event* tpcgen_generate(const tpcgen_config* cfg, uint64_t seed) {
    if (!cfg || cfg->n_rows <= 0 || !cfg->row_x || (cfg->n_sectors != 36 && cfg->n_sectors != 1)) return NULL;
    const int ns = cfg->n_sectors, nr = cfg->n_rows;
    const int n_prim = cfg->n_primaries;
    const int n_sec = (int)floor(cfg->frac_secondaries * n_prim + 0.5);
    const int n_trk = n_prim + n_sec;
    bucket_t* bk = (bucket_t*)calloc(ns, sizeof(bucket_t));
    tpcgen_event* ev = (tpcgen_event*)calloc(1, sizeof(tpcgen_event));
    if (!bk || !ev) { free(bk); free(ev); return NULL; }
    ev->trk = (double*)calloc((size_t)(n_trk > 0 ? n_trk : 1) * TPCGEN_TRK_COLS, sizeof(double));
    int fail = (ev->trk == NULL);
    const double absbz = fabs(cfg->bz);
    const double sgnbz = cfg->bz >= 0 ? 1.0 : -1.0;
    const double deg = TPCGEN_PI / 180.0;

    for (int it = 0; it < n_trk && !fail; it++) {
        rng_t rt = rng_make(seed, 1, (uint64_t)it);
        const int primary = it < n_prim;
        double pt = cfg->pt_mode == 0 ? cfg->pt_a + (cfg->pt_b - cfg->pt_a) * rng_u(&rt)
                                      : cfg->pt_a - cfg->pt_b * log(rng_u(&rt));
        double eta = (2.0 * rng_u(&rt) - 1.0) * cfg->eta_max;
        double phi = 2.0 * TPCGEN_PI * rng_u(&rt);
        double charge = rng_u(&rt) < 0.5 ? -1.0 : 1.0;
        double vx = 0, vy = 0, vz = 0;
        if (!primary) {
            double rv = 50.0 * rng_u(&rt), pv = 2.0 * TPCGEN_PI * rng_u(&rt);
            vx = rv * cos(pv); vy = rv * sin(pv); vz = 50.0 * (2.0 * rng_u(&rt) - 1.0);
        }
        if (ns == 1) { /* config 1: aim every track into sector 0 on the A side */
            phi = (10.0 + 9.0 * (2.0 * rng_u(&rt) - 1.0)) * deg;
            eta = fabs(eta);
        }
        double* T = ev->trk + (size_t)it * TPCGEN_TRK_COLS;
        T[TRK_PT] = pt; T[TRK_CHARGE] = charge; T[TRK_ETA] = eta; T[TRK_PHI] = phi;
        T[TRK_VX] = vx; T[TRK_VY] = vy; T[TRK_VZ] = vz; T[TRK_PRIMARY] = primary;

        const double t = sinh(eta);
        const double R = pt / (TPCGEN_K * absbz);
        const double h = -charge * sgnbz;
        const double cx = vx - h * R * sin(phi), cy = vy + h * R * cos(phi);
        const double psi0 = atan2(vy - cy, vx - cx);
        const double cnorm = sqrt(cx * cx + cy * cy);

        /* where does the track end?  theta_end = min(exit through r_max, exit through |z| = z_max, turn limit) */
        double theta_end;
        const int is_looper = (cnorm + R < cfg->r_max);
        if (cfg->loopers && is_looper) theta_end = 2.0 * TPCGEN_PI * cfg->max_turns;
        else theta_end = TPCGEN_PI;
        if (!is_looper && cnorm > 0) { /* first theta with |pos| = r_max */
            double m = (cfg->r_max * cfg->r_max - cnorm * cnorm - R * R) / (2.0 * R * cnorm);
            if (m >= -1.0 && m <= 1.0) {
                double ac = acos(m), argc = atan2(cy, cx);
                double th1 = wrap_2pi(h * (argc + ac - psi0)), th2 = wrap_2pi(h * (argc - ac - psi0));
                double the = th1 < th2 ? th1 : th2;
                if (the < theta_end) theta_end = the;
            }
        }
        if (t != 0.0) {
            double zlim = t > 0 ? cfg->z_max : -cfg->z_max;
            double thz = (zlim - vz) / (t * R);
            if (thz < theta_end) theta_end = thz;
        }

        rng_t rs = rng_make(seed, 2, (uint64_t)it); /* smearing / inefficiency stream */
        for (int sa = 0; sa < (ns == 1 ? 1 : 18) && !fail; sa++) {
            const double alpha = (20.0 * sa + 10.0) * deg;
            const double ca = cos(alpha), sn = sin(alpha);
            const double lcx = cx * ca + cy * sn, lcy = -cx * sn + cy * ca; /* centre in the local frame */
            for (int r = 0; r < nr && !fail; r++) {
                const double xr = cfg->row_x[r];
                const double ddx = xr - lcx;
                const double disc = R * R - ddx * ddx;
                if (disc <= 0) continue;
                const double sq = sqrt(disc);
                for (int root = 0; root < 2; root++) {
                    const double yl = lcy + (root ? sq : -sq);
                    if (fabs(yl) > xr * cfg->tan_half_angle) continue;
                    const double psi = atan2(yl - lcy, ddx) + alpha;
                    const double th0 = wrap_2pi(h * (psi - psi0));
                    for (int turn = 0; turn < (cfg->loopers ? cfg->max_turns : 1); turn++) {
                        const double th = th0 + 2.0 * TPCGEN_PI * turn;
                        if (th >= theta_end) break;
                        const double zz = vz + t * R * th;
                        if (fabs(zz) > cfg->z_max) break;
                        const int cside = zz < 0;
                        if (ns == 1 && cside) continue;
                        const int s = sa + (cside ? 18 : 0);
                        /* draw in a fixed order so the stream does not depend on acceptance */
                        const double drop = rng_u(&rs), gy = rng_normal(&rs), gz = rng_normal(&rs);
                        if (drop < cfg->inefficiency) continue;
                        if (bucket_push(&bk[ns == 1 ? 0 : s], (float)(yl + cfg->sigma_y * gy),
                                        (float)(zz + cfg->sigma_z * gz), r, it))
                            fail = 1;
                    }
                }
            }
        }
    }

    /* noise */
    for (int s = 0; s < ns && !fail; s++) {
        rng_t rn = rng_make(seed, 3, (uint64_t)s);
        const int nn = (int)floor(cfg->noise_frac * bk[s].n + 0.5);
        const int cside = s >= 18;
        for (int i = 0; i < nn && !fail; i++) {
            int r = (int)(rng_u(&rn) * nr);
            if (r >= nr) r = nr - 1;
            double ymax = cfg->row_x[r] * cfg->tan_half_angle;
            double y = (2.0 * rng_u(&rn) - 1.0) * ymax;
            double z = rng_u(&rn) * cfg->z_max;
            if (cside) z = -z;
            if (bucket_push(&bk[s], (float)y, (float)z, r, -1)) fail = 1;
        }
    }

    /* flatten, shuffling inside each sector (Fisher-Yates) */
    if (!fail) {
        int64_t tot = 0;
        for (int s = 0; s < ns; s++) tot += bk[s].n;
        size_t na = (size_t)(tot > 0 ? tot : 1);
        ev->n_clusters = (int32_t)tot; ev->n_tracks = n_trk; ev->n_sectors = ns;
        ev->sector_offset = (int32_t*)calloc(ns + 1, sizeof(int32_t));
        ev->x = (float*)malloc(sizeof(float) * na); ev->y = (float*)malloc(sizeof(float) * na);
        ev->z = (float*)malloc(sizeof(float) * na);
        ev->row = (int32_t*)malloc(sizeof(int32_t) * na); ev->label = (int32_t*)malloc(sizeof(int32_t) * na);
        if (!ev->sector_offset || !ev->x || !ev->y || !ev->z || !ev->row || !ev->label) fail = 1;
    }
    if (!fail) {
        int32_t off = 0;
        for (int s = 0; s < ns; s++) {
            const int n = bk[s].n;
            ev->sector_offset[s] = off;
            int32_t* perm = (int32_t*)malloc(sizeof(int32_t) * (n > 0 ? n : 1));
            if (!perm) { fail = 1; break; }
            for (int i = 0; i < n; i++) perm[i] = i;
            if (cfg->shuffle) {
                rng_t rp = rng_make(seed, 4, (uint64_t)s);
                for (int i = n - 1; i > 0; i--) {
                    int j = (int)(rng_u(&rp) * (i + 1));
                    if (j > i) j = i;
                    int32_t tmp = perm[i]; perm[i] = perm[j]; perm[j] = tmp;
                }
            }
            for (int i = 0; i < n; i++) {
                const int k = perm[i];
                ev->y[off + i] = bk[s].y[k]; ev->z[off + i] = bk[s].z[k];
                ev->row[off + i] = bk[s].row[k]; ev->label[off + i] = bk[s].label[k];
                ev->x[off + i] = (float)cfg->row_x[bk[s].row[k]];
            }
            free(perm);
            off += n;
        }
        ev->sector_offset[ns] = off;
    }
    for (int s = 0; s < ns; s++) { free(bk[s].y); free(bk[s].z); free(bk[s].row); free(bk[s].label); }
    free(bk);
    if (fail) { tpcgen_free(ev); return NULL; }
    return ev;
}

int32_t tpcgen_n_clusters(const tpcgen_event* ev) { return ev->n_clusters; }
int32_t tpcgen_n_tracks(const tpcgen_event* ev) { return ev->n_tracks; }
int32_t tpcgen_trk_cols(void) { return TPCGEN_TRK_COLS; }

/* copy out into caller arrays (sizes from the two getters above) */
void tpcgen_copy(const tpcgen_event* ev, int32_t* sector_offset, float* x, float* y, float* z, int32_t* row,
                 int32_t* label, double* trk) {
    const size_t n = (size_t)ev->n_clusters;
    memcpy(sector_offset, ev->sector_offset, sizeof(int32_t) * (ev->n_sectors + 1));
    memcpy(x, ev->x, sizeof(float) * n); memcpy(y, ev->y, sizeof(float) * n); memcpy(z, ev->z, sizeof(float) * n);
    memcpy(row, ev->row, sizeof(int32_t) * n); memcpy(label, ev->label, sizeof(int32_t) * n);
    memcpy(trk, ev->trk, sizeof(double) * (size_t)ev->n_tracks * TPCGEN_TRK_COLS);
}
