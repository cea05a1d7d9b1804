/*
 * ffgen.c -- seeded synthetic dipole ensembles (input generators only).
 *
 * These inputs STAND IN for the paper's self-generated random ensembles
 * ("randomly distributing particles in a cubic container", and
 * the chain-forming regime of Fig. 2); the paper uses no public
 * data set.  Shapes follow BASELINE.json `configs` / SURVEY.md 8(d).
 *
 * This module serves BOTH the CUDA path and the oracle and therefore holds
 * none of the method's arithmetic: no dipole field, no force, no Morton key,
 * no tree.  It only draws positions and moment directions.
 *
 * RNG: counter based.  u64 = splitmix64_finalizer(seed, stream, counter);
 * a draw is identified by (seed, stream, counter) and never depends on how
 * many other draws were made, so every config is reproducible bit for bit.
 *
 * Length unit: sphere diameter d = 1 (BASELINE.json), so contact is at
 * distance 1.  Box side from Eq. 16 with R = d/2:
 *   phi = N (pi d^3 / 6) / L^3   =>   L = (N pi / (6 phi))^(1/3).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define FFGEN_PI 3.14159265358979323846

static uint64_t mix64(uint64_t z)
{
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

/* uniform double in [0,1) identified by (seed, stream, counter) */
static double u01(uint64_t seed, uint64_t stream, uint64_t counter)
{
    uint64_t z = mix64(seed * 0x9E3779B97F4A7C15ULL + 0x632BE59BD9B4E019ULL);
    z = mix64(z ^ (stream * 0xD1B54A32D192ED03ULL + 0x8CB92BA72F3D8DD7ULL));
    z = mix64(z + counter * 0x9E3779B97F4A7C15ULL);
    return (double)(z >> 11) * (1.0 / 9007199254740992.0);
}

double ffgen_box_side(int64_t N, double phi)
{
    return cbrt((double)N * FFGEN_PI / (6.0 * phi));
}

/* ---- cell list over fp32 sphere centres (cell side >= 1) ---------------- */
typedef struct {
    double org;      /* grid origin (same for the 3 axes) */
    double inv;      /* 1 / cell side */
    int    n;        /* cells per axis */
    int*   head;     /* n^3, -1 = empty */
    int*   next;     /* per particle */
} grid_t;

static int grid_init(grid_t* g, double lo, double hi, int64_t cap)
{
    double ext = hi - lo;
    int n = (int)floor(ext);            /* side = ext / n >= 1 */
    if (n < 1) n = 1;
    if (n > 400) n = 400;               /* side only grows: still >= 1 */
    g->org = lo;
    g->n = n;
    g->inv = (double)n / ext;
    size_t nc = (size_t)n * n * n;
    g->head = (int*)malloc(nc * sizeof(int));
    g->next = (int*)malloc((size_t)cap * sizeof(int));
    if (!g->head || !g->next) return -1;
    memset(g->head, 0xFF, nc * sizeof(int));
    return 0;
}

static void grid_free(grid_t* g) { free(g->head); free(g->next); }

static int grid_coord(const grid_t* g, double x)
{
    int c = (int)floor((x - g->org) * g->inv);
    if (c < 0) c = 0;
    if (c >= g->n) c = g->n - 1;
    return c;
}

/* 1 if a sphere centred at p overlaps (distance < 1) any stored sphere */
static int grid_overlaps(const grid_t* g, const float* pos, const float p[3])
{
    int c[3];
    for (int a = 0; a < 3; ++a) c[a] = grid_coord(g, p[a]);
    for (int ix = c[0] - 1; ix <= c[0] + 1; ++ix) {
        if (ix < 0 || ix >= g->n) continue;
        for (int iy = c[1] - 1; iy <= c[1] + 1; ++iy) {
            if (iy < 0 || iy >= g->n) continue;
            for (int iz = c[2] - 1; iz <= c[2] + 1; ++iz) {
                if (iz < 0 || iz >= g->n) continue;
                size_t cell = ((size_t)ix * g->n + iy) * g->n + iz;
                for (int j = g->head[cell]; j >= 0; j = g->next[j]) {
                    double dx = (double)p[0] - pos[3 * (size_t)j];
                    double dy = (double)p[1] - pos[3 * (size_t)j + 1];
                    double dz = (double)p[2] - pos[3 * (size_t)j + 2];
                    if (dx * dx + dy * dy + dz * dz < 1.0) return 1;
                }
            }
        }
    }
    return 0;
}

static void grid_insert(grid_t* g, const float p[3], int idx)
{
    size_t cell = ((size_t)grid_coord(g, p[0]) * g->n + grid_coord(g, p[1])) * g->n
                  + grid_coord(g, p[2]);
    g->next[idx] = g->head[cell];
    g->head[cell] = idx;
}

/*
 * Hard spheres of diameter 1, centres uniform in [0,L)^3, by random
 * sequential addition: candidate c = 0,1,2,... is drawn from counters
 * 3c..3c+2 of stream 1 and kept iff its fp32 centre is at distance >= 1 from
 * every centre kept before.  pos: [N][3] fp32.  Returns the number of
 * candidates drawn (> 0) or -1 on allocation failure / -2 if the box jams.
 */
int64_t ffgen_hard_spheres(int64_t N, double L, uint64_t seed, float* pos)
{
    grid_t g;
    if (grid_init(&g, 0.0, L, N) != 0) return -1;
    int64_t n = 0;
    uint64_t c = 0;
    uint64_t limit = (uint64_t)N * 400u + 100000u;
    while (n < N) {
        if (c >= limit) { grid_free(&g); return -2; }
        float p[3];
        for (int a = 0; a < 3; ++a) {
            p[a] = (float)(u01(seed, 1, 3 * c + a) * L);
            if (p[a] >= (float)L) p[a] = nextafterf((float)L, 0.0f);
        }
        ++c;
        if (grid_overlaps(&g, pos, p)) continue;
        pos[3 * n] = p[0]; pos[3 * n + 1] = p[1]; pos[3 * n + 2] = p[2];
        grid_insert(&g, p, (int)n);
        ++n;
    }
    grid_free(&g);
    return (int64_t)c;
}

/* Isotropic unit vectors: z = 2 xi1 - 1, azimuth = 2 pi xi2 (stream 2). */
void ffgen_moments_isotropic(int64_t N, uint64_t seed, float* mom)
{
    for (int64_t i = 0; i < N; ++i) {
        double z = 2.0 * u01(seed, 2, 2 * (uint64_t)i) - 1.0;
        double a = 2.0 * FFGEN_PI * u01(seed, 2, 2 * (uint64_t)i + 1);
        double s = sqrt(fmax(0.0, 1.0 - z * z));
        mom[3 * i] = (float)(s * cos(a));
        mom[3 * i + 1] = (float)(s * sin(a));
        mom[3 * i + 2] = (float)z;
    }
}

/*
 * von Mises-Fisher about +z with concentration kappa (an applied field along
 * z): cos(theta) = 1 + ln(xi + (1 - xi) e^{-2 kappa}) / kappa,
 * azimuth uniform (stream 3).  <u_z> = coth(kappa) - 1/kappa, the Langevin
 * function of Eq. 17 with alpha = kappa.
 */
void ffgen_moments_vmf(int64_t N, double kappa, uint64_t seed, float* mom)
{
    double e = exp(-2.0 * kappa);
    for (int64_t i = 0; i < N; ++i) {
        double xi = u01(seed, 3, 2 * (uint64_t)i);
        double a = 2.0 * FFGEN_PI * u01(seed, 3, 2 * (uint64_t)i + 1);
        double z = 1.0 + log(xi + (1.0 - xi) * e) / kappa;
        if (z < -1.0) z = -1.0;
        if (z > 1.0) z = 1.0;
        double s = sqrt(fmax(0.0, 1.0 - z * z));
        mom[3 * i] = (float)(s * cos(a));
        mom[3 * i + 1] = (float)(s * sin(a));
        mom[3 * i + 2] = (float)z;
    }
}

/*
 * Clustered ensemble: n_chains straight head-to-tail chains of `len`
 * touching spheres (spacing 1).  Chain centre uniform in [0,L)^3, axis
 * uniform in the cap of half-angle cap_deg about +z (cos uniform in
 * [cos cap, 1], azimuth uniform), sphere i at centre + (i - (len-1)/2) axis.
 * Candidate chain c uses counters 5c..5c+4 of stream 4; it is rejected if any
 * of its fp32 sphere centres is closer than 1 to a sphere of an earlier
 * chain.  Chains may stick out of the cube.  Moments lie along the axis.
 * pos, mom: [n_chains*len][3].  Returns candidates drawn, -1 alloc, -2 jam.
 */
int64_t ffgen_chains(int64_t n_chains, int len, double L, double cap_deg,
                     uint64_t seed, float* pos, float* mom)
{
    int64_t N = n_chains * (int64_t)len;
    double half = 0.5 * (len - 1);
    grid_t g;
    if (grid_init(&g, -half - 1.0, L + half + 1.0, N) != 0) return -1;
    float* tmp = (float*)malloc((size_t)len * 3 * sizeof(float));
    if (!tmp) { grid_free(&g); return -1; }
    double cmin = cos(cap_deg * FFGEN_PI / 180.0);
    int64_t nc = 0;
    uint64_t c = 0;
    uint64_t limit = (uint64_t)n_chains * 400u + 100000u;
    while (nc < n_chains) {
        if (c >= limit) { free(tmp); grid_free(&g); return -2; }
        double cx = u01(seed, 4, 5 * c) * L;
        double cy = u01(seed, 4, 5 * c + 1) * L;
        double cz = u01(seed, 4, 5 * c + 2) * L;
        double ct = cmin + (1.0 - cmin) * u01(seed, 4, 5 * c + 3);
        double az = 2.0 * FFGEN_PI * u01(seed, 4, 5 * c + 4);
        ++c;
        double st = sqrt(fmax(0.0, 1.0 - ct * ct));
        double ax = st * cos(az), ay = st * sin(az), azz = ct;
        int bad = 0;
        for (int i = 0; i < len; ++i) {
            double t = (double)i - half;
            tmp[3 * i] = (float)(cx + t * ax);
            tmp[3 * i + 1] = (float)(cy + t * ay);
            tmp[3 * i + 2] = (float)(cz + t * azz);
            if (grid_overlaps(&g, pos, tmp + 3 * i)) { bad = 1; break; }
        }
        if (bad) continue;
        for (int i = 0; i < len; ++i) {
            int64_t k = nc * len + i;
            pos[3 * k] = tmp[3 * i]; pos[3 * k + 1] = tmp[3 * i + 1]; pos[3 * k + 2] = tmp[3 * i + 2];
            mom[3 * k] = (float)ax; mom[3 * k + 1] = (float)ay; mom[3 * k + 2] = (float)azz;
            grid_insert(&g, tmp + 3 * i, (int)k);
        }
        ++nc;
    }
    free(tmp);
    grid_free(&g);
    return (int64_t)c;
}

/* Uniform points without the hard core (degenerate / edge-case inputs). */
void ffgen_uniform_points(int64_t N, double L, uint64_t seed, float* pos)
{
    for (int64_t i = 0; i < 3 * N; ++i) pos[i] = (float)(u01(seed, 5, (uint64_t)i) * L);
}
