/*
 * vrgen.c — seeded synthetic spectral-cube generator (INPUT GENERATOR ONLY).
 *
 * This module holds none of the method's arithmetic (no ray-casting, no
 * reductions).  It produces the bytes that BOTH the CPU oracle (oracle/) and the
 * CUDA library (paper_1111_6661_b200/csrc/) consume, so that parity is decided
 * on identical inputs.  It stands in for the paper's spectral cubes
 * (Table 1), which are not available; recipe = SURVEY.md
 * §8(d) D.1 / BASELINE.json configs: i.i.d. N(0, sigma(z)^2) noise + a linear
 * ramp along x + anisotropic Gaussian sources.
 *
 * Determinism: every transcendental (log, sin/cos, exp) is evaluated by the
 * fixed polynomial sequences below using only IEEE-754 double +,-,*,/,sqrt,fma,
 * so the voxel value is a pure function of (seed, recipe, ix, iy, iz) that any
 * other implementation (e.g. a CUDA twin) can reproduce bit for bit.
 * Build: gcc -O2 -fopenmp -mfma -ffp-contract=off -shared -fPIC.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define VRGEN_EXPORT __attribute__((visibility("default")))

/* ---------------- Philox-4x32-10 (counter-based RNG) ---------------- */
static inline void philox4x32_10(uint32_t c[4], uint32_t k0, uint32_t k1)
{
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c[0];
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c[2];
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c[1] ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c[3] ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c[0] = n0; c[1] = n1; c[2] = n2; c[3] = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
}

/* uniform in (0,1), exact in double */
static inline double u01(uint32_t x) { return ((double)x + 0.5) * (1.0 / 4294967296.0); }

/* ---------------- deterministic elementary functions ---------------- */
static inline double det_log(double x) /* x > 0, normal */
{
    uint64_t b; memcpy(&b, &x, 8);
    int e = (int)((b >> 52) & 0x7ff) - 1023;
    b = (b & 0x000fffffffffffffull) | 0x3ff0000000000000ull;
    double m; memcpy(&m, &b, 8);               /* m in [1,2) */
    if (m > 1.4142135623730951) { m = m * 0.5; e += 1; }
    double s = (m - 1.0) / (m + 1.0);
    double z = s * s;
    double p = 1.0 / 23.0;
    p = fma(p, z, 1.0 / 21.0); p = fma(p, z, 1.0 / 19.0); p = fma(p, z, 1.0 / 17.0);
    p = fma(p, z, 1.0 / 15.0); p = fma(p, z, 1.0 / 13.0); p = fma(p, z, 1.0 / 11.0);
    p = fma(p, z, 1.0 / 9.0);  p = fma(p, z, 1.0 / 7.0);  p = fma(p, z, 1.0 / 5.0);
    p = fma(p, z, 1.0 / 3.0);
    double lm = fma(2.0 * s, p * z, 2.0 * s);   /* log(m) = 2s(1 + z p) */
    return fma((double)e, 0.6931471805599453, lm);
}

/* sin and cos of 2*pi*u, u in [0,1) */
static inline void det_sincos2pi(double u, double *sn, double *cs)
{
    double x = u * 4.0;
    double qf = floor(x + 0.5);
    double r = (x - qf) * 1.5707963267948966;   /* [-pi/4, pi/4] */
    int q = ((int)qf) & 3;
    double z = r * r;
    double ps = 1.0 / 355687428096000.0;                       /* +1/17! */
    ps = fma(ps, z, -1.0 / 1307674368000.0);                   /* -1/15! */
    ps = fma(ps, z, 1.0 / 6227020800.0);                       /* +1/13! */
    ps = fma(ps, z, -1.0 / 39916800.0);                        /* -1/11! */
    ps = fma(ps, z, 1.0 / 362880.0);                           /* +1/9!  */
    ps = fma(ps, z, -1.0 / 5040.0);                            /* -1/7!  */
    ps = fma(ps, z, 1.0 / 120.0);                              /* +1/5!  */
    ps = fma(ps, z, -1.0 / 6.0);                               /* -1/3!  */
    double s0 = fma(r * z, ps, r);
    double pc = 1.0 / 20922789888000.0;                        /*  1/16! */
    pc = fma(pc, z, -1.0 / 87178291200.0);                     /* -1/14! */
    pc = fma(pc, z, 1.0 / 479001600.0);                        /*  1/12! */
    pc = fma(pc, z, -1.0 / 3628800.0);                         /* -1/10! */
    pc = fma(pc, z, 1.0 / 40320.0);
    pc = fma(pc, z, -1.0 / 720.0);
    pc = fma(pc, z, 1.0 / 24.0);
    pc = fma(pc, z, -0.5);
    double c0 = fma(z, pc, 1.0);
    switch (q) {
    case 0: *sn = s0;  *cs = c0;  break;
    case 1: *sn = c0;  *cs = -s0; break;
    case 2: *sn = -s0; *cs = -c0; break;
    default: *sn = -c0; *cs = s0; break;
    }
}

/* exp(-a), 0 <= a <= 700 */
static inline double det_exp_neg(double a)
{
    double y = -a;
    double kf = floor(fma(y, 1.4426950408889634, 0.5));
    double r = fma(kf, -0.6931471803691238, y);           /* ln2 hi */
    r = fma(kf, -1.9082149292705877e-10, r);              /* ln2 lo */
    double p = 1.0 / 6227020800.0;                        /* 1/13! */
    p = fma(p, r, 1.0 / 479001600.0);
    p = fma(p, r, 1.0 / 39916800.0);
    p = fma(p, r, 1.0 / 3628800.0);
    p = fma(p, r, 1.0 / 362880.0);
    p = fma(p, r, 1.0 / 40320.0);
    p = fma(p, r, 1.0 / 5040.0);
    p = fma(p, r, 1.0 / 720.0);
    p = fma(p, r, 1.0 / 120.0);
    p = fma(p, r, 1.0 / 24.0);
    p = fma(p, r, 1.0 / 6.0);
    p = fma(p, r, 0.5);
    p = fma(p, r, 1.0);
    p = fma(p, r, 1.0);
    int k = (int)kf;                                      /* >= -1011 */
    uint64_t b = (uint64_t)(k + 1023) << 52;
    double sc; memcpy(&sc, &b, 8);
    return p * sc;
}

/* ---------------- recipe ---------------- */
typedef struct {
    uint32_t struct_size;
    uint32_t nx, ny, nz;
    uint64_t seed;
    uint32_t n_sources;
    float ramp_max;      /* linear ramp 0..ramp_max along x (cfg3: 2) */
    float sigma_mod;     /* sigma(z) = 1 + sigma_mod*sin(2 pi z / nz) (cfg4/5: 0.5) */
    float noise_amp;     /* 1 = N(0,1); 0 = sources/ramp only (smooth cubes for tests) */
} vrgen_recipe;

typedef struct { double A, hxy, hz, cx, cy, cz, rxy, rz; } vrgen_source;

struct vrgen_ctx {
    vrgen_recipe r;
    vrgen_source *src;
    /* per-z list of sources (index order) whose z support covers that slice */
    uint32_t *zlist_off; uint32_t *zlist;
    double *sigma_z;
};
typedef struct vrgen_ctx vrgen_ctx;

static void make_sources(vrgen_ctx *g)
{
    const vrgen_recipe *r = &g->r;
    uint32_t k0 = (uint32_t)r->seed, k1 = (uint32_t)(r->seed >> 32);
    for (uint32_t s = 0; s < r->n_sources; ++s) {
        uint32_t a[4] = { s, 0u, 1u, 0u }, b[4] = { s, 1u, 1u, 0u };
        philox4x32_10(a, k0, k1); philox4x32_10(b, k0, k1);
        vrgen_source *q = &g->src[s];
        q->A = 5.0 + 15.0 * u01(a[0]);
        double sxy = 2.0 + 4.0 * u01(a[1]);
        double sz = 4.0 + 8.0 * u01(a[2]);
        q->cx = (double)r->nx * u01(a[3]);
        q->cy = (double)r->ny * u01(b[0]);
        q->cz = (double)r->nz * u01(b[1]);
        q->hxy = 1.0 / (2.0 * sxy * sxy);
        q->hz = 1.0 / (2.0 * sz * sz);
        q->rxy = 5.0 * sxy; q->rz = 5.0 * sz;
    }
}

VRGEN_EXPORT vrgen_ctx *vrgen_create(const vrgen_recipe *r)
{
    if (!r || r->struct_size != sizeof(vrgen_recipe) || !r->nx || !r->ny || !r->nz) return NULL;
    vrgen_ctx *g = (vrgen_ctx *)calloc(1, sizeof(*g));
    g->r = *r;
    g->src = (vrgen_source *)calloc(r->n_sources ? r->n_sources : 1, sizeof(vrgen_source));
    make_sources(g);
    g->sigma_z = (double *)malloc(sizeof(double) * r->nz);
    for (uint32_t z = 0; z < r->nz; ++z) {
        double sn, cs; det_sincos2pi((double)z / (double)r->nz, &sn, &cs);
        g->sigma_z[z] = (double)r->noise_amp * fma((double)r->sigma_mod, sn, 1.0);
    }
    g->zlist_off = (uint32_t *)calloc((size_t)r->nz + 1, sizeof(uint32_t));
    for (int pass = 0; pass < 2; ++pass) {
        if (pass == 1) {
            uint32_t acc = 0;
            for (uint32_t z = 0; z <= r->nz; ++z) { uint32_t c = g->zlist_off[z]; g->zlist_off[z] = acc; acc += c; }
            g->zlist = (uint32_t *)malloc(sizeof(uint32_t) * (acc ? acc : 1));
        }
        uint32_t *fill = pass ? (uint32_t *)calloc(r->nz, sizeof(uint32_t)) : NULL;
        for (uint32_t s = 0; s < r->n_sources; ++s) {   /* index order preserved per z */
            const vrgen_source *q = &g->src[s];
            for (uint32_t z = 0; z < r->nz; ++z) {
                if (fabs((double)z - q->cz) > q->rz) continue;
                if (!pass) g->zlist_off[z]++;
                else g->zlist[g->zlist_off[z] + fill[z]++] = s;
            }
        }
        free(fill);
    }
    return g;
}

VRGEN_EXPORT void vrgen_destroy(vrgen_ctx *g)
{
    if (!g) return;
    free(g->src); free(g->zlist_off); free(g->zlist); free(g->sigma_z); free(g);
}

/* four N(0,1) deviates for voxels 4c .. 4c+3 (c = linear voxel index / 4) */
static inline void noise4(const vrgen_ctx *g, uint64_t c, double z[4])
{
    uint32_t ctr[4] = { (uint32_t)c, (uint32_t)(c >> 32), 0u, 0u };
    philox4x32_10(ctr, (uint32_t)g->r.seed, (uint32_t)(g->r.seed >> 32));
    for (int p = 0; p < 2; ++p) {
        double rad = sqrt(-2.0 * det_log(u01(ctr[2 * p])));
        double sn, cs; det_sincos2pi(u01(ctr[2 * p + 1]), &sn, &cs);
        z[2 * p] = rad * cs; z[2 * p + 1] = rad * sn;
    }
}

static inline double base_value(const vrgen_ctx *g, double nz1, uint32_t ix, uint32_t iz)
{
    double ramp = g->r.nx > 1 ? (double)g->r.ramp_max * ((double)ix / (double)(g->r.nx - 1)) : 0.0;
    return fma(g->sigma_z[iz], nz1, ramp);
}

static inline double source_term(const vrgen_source *q, double dx, double dy, double dz)
{
    double arg = fma(dz * dz, q->hz, (dx * dx + dy * dy) * q->hxy);
    return q->A * det_exp_neg(arg);
}

/* one voxel, on demand; identical to the bulk path bit for bit */
VRGEN_EXPORT float vrgen_voxel(const vrgen_ctx *g, uint32_t ix, uint32_t iy, uint32_t iz)
{
    uint64_t lin = (uint64_t)ix + (uint64_t)g->r.nx * ((uint64_t)iy + (uint64_t)g->r.ny * iz);
    double z[4]; noise4(g, lin >> 2, z);
    double v = base_value(g, z[lin & 3], ix, iz);
    for (uint32_t i = g->zlist_off[iz]; i < g->zlist_off[iz + 1]; ++i) {
        const vrgen_source *q = &g->src[g->zlist[i]];
        double dy = (double)iy - q->cy, dx = (double)ix - q->cx;
        if (fabs(dy) > q->rxy || fabs(dx) > q->rxy) continue;
        v += source_term(q, dx, dy, (double)iz - q->cz);
    }
    return (float)v;
}

/* fill out[(z1-z0) * ny * nx] with slices z0 <= iz < z1, x fastest */
VRGEN_EXPORT int vrgen_fill(const vrgen_ctx *g, uint32_t z0, uint32_t z1, float *out)
{
    if (!g || !out || z1 > g->r.nz || z0 > z1) return -1;
    const uint32_t nx = g->r.nx, ny = g->r.ny;
    const int64_t nrows = (int64_t)(z1 - z0) * ny;
#pragma omp parallel
    {
        double *row = (double *)malloc(sizeof(double) * ((size_t)nx + 8));
#pragma omp for schedule(dynamic, 16)
        for (int64_t rr = 0; rr < nrows; ++rr) {
            uint32_t iz = z0 + (uint32_t)(rr / ny), iy = (uint32_t)(rr % ny);
            uint64_t lin0 = (uint64_t)nx * ((uint64_t)iy + (uint64_t)ny * iz);
            uint64_t lin = lin0, end = lin0 + nx;
            while (lin < end) {
                double z[4]; noise4(g, lin >> 2, z);
                uint32_t l = (uint32_t)(lin & 3);
                for (; l < 4 && lin < end; ++l, ++lin)
                    row[lin - lin0] = base_value(g, z[l], (uint32_t)(lin - lin0), iz);
            }
            for (uint32_t i = g->zlist_off[iz]; i < g->zlist_off[iz + 1]; ++i) {
                const vrgen_source *q = &g->src[g->zlist[i]];
                double dy = (double)iy - q->cy;
                if (fabs(dy) > q->rxy) continue;
                double dz = (double)iz - q->cz;
                double lo = ceil(q->cx - q->rxy), hi = floor(q->cx + q->rxy);
                if (lo < 0.0) lo = 0.0;
                if (hi > (double)nx - 1.0) hi = (double)nx - 1.0;
                for (int64_t ix = (int64_t)lo; ix <= (int64_t)hi; ++ix) {
                    double dx = (double)ix - q->cx;
                    if (fabs(dx) > q->rxy) continue;
                    row[ix] += source_term(q, dx, dy, dz);
                }
            }
            float *o = out + (size_t)rr * nx;
            for (uint32_t ix = 0; ix < nx; ++ix) o[ix] = (float)row[ix];
        }
        free(row);
    }
    return 0;
}

/* source parameters for tests / documentation: 8 doubles per source */
VRGEN_EXPORT int vrgen_sources(const vrgen_ctx *g, double *out8)
{
    if (!g || !out8) return -1;
    memcpy(out8, g->src, sizeof(vrgen_source) * g->r.n_sources);
    return 0;
}

/* 64-bit wrap-around sum of the float bit patterns: identity of a cube's bytes */
VRGEN_EXPORT uint64_t vrgen_checksum(const float *v, uint64_t n)
{
    uint64_t s = 0;
#pragma omp parallel for reduction(+ : s)
    for (int64_t i = 0; i < (int64_t)n; ++i) { uint32_t b; memcpy(&b, v + i, 4); s += b; }
    return s;
}

/* re-tile slices into brick-major layout with a +1 high-side halo (clamped at the
 * volume faces): out[brick][ (B+1)^3 ], brick id = bx + nbx*(by + nby*bz), x fastest.
 * Pure data movement (cfg5 host layout). */
VRGEN_EXPORT int vrgen_retile_halo(const float *lin, uint32_t nx, uint32_t ny, uint32_t nz,
                                   uint32_t B, float *out)
{
    if (!lin || !out || !B) return -1;
    uint32_t nbx = (nx + B - 1) / B, nby = (ny + B - 1) / B, nbz = (nz + B - 1) / B;
    uint32_t E = B + 1;
    int64_t nb = (int64_t)nbx * nby * nbz;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t b = 0; b < nb; ++b) {
        uint32_t bx = (uint32_t)(b % nbx), by = (uint32_t)((b / nbx) % nby), bz = (uint32_t)(b / ((int64_t)nbx * nby));
        float *o = out + (size_t)b * E * E * E;
        for (uint32_t z = 0; z < E; ++z) {
            uint32_t gz = bz * B + z; if (gz > nz - 1) gz = nz - 1;
            for (uint32_t y = 0; y < E; ++y) {
                uint32_t gy = by * B + y; if (gy > ny - 1) gy = ny - 1;
                const float *src = lin + (size_t)nx * (gy + (size_t)ny * gz);
                float *dst = o + (size_t)E * (y + (size_t)E * z);
                for (uint32_t x = 0; x < E; ++x) {
                    uint32_t gx = bx * B + x; if (gx > nx - 1) gx = nx - 1;
                    dst[x] = src[gx];
                }
            }
        }
    }
    return 0;
}

/* One brick LAYER (all bricks with the same bz) from a slab that holds the slices [bz*B, bz*B + nzs), nzs <= B + 1:
 * the slab is the layer's own z-range plus, unless it is the last layer, its one-slice halo.  Lets a cube
 * larger than spare host memory be generated straight into the brick-major layout, layer by layer. */
VRGEN_EXPORT int vrgen_retile_halo_layer(const float *slab, uint32_t nx, uint32_t ny, uint32_t nzs,
                                         uint32_t B, float *out)
{
    if (!slab || !out || !B || !nzs || nzs > B + 1) return -1;
    uint32_t nbx = (nx + B - 1) / B, nby = (ny + B - 1) / B;
    uint32_t E = B + 1;
    int64_t nb = (int64_t)nbx * nby;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t b = 0; b < nb; ++b) {
        uint32_t bx = (uint32_t)(b % nbx), by = (uint32_t)(b / nbx);
        float *o = out + (size_t)b * E * E * E;
        for (uint32_t z = 0; z < E; ++z) {
            uint32_t gz = z; if (gz > nzs - 1) gz = nzs - 1;
            for (uint32_t y = 0; y < E; ++y) {
                uint32_t gy = by * B + y; if (gy > ny - 1) gy = ny - 1;
                const float *src = slab + (size_t)nx * (gy + (size_t)ny * gz);
                float *dst = o + (size_t)E * (y + (size_t)E * z);
                for (uint32_t x = 0; x < E; ++x) {
                    uint32_t gx = bx * B + x; if (gx > nx - 1) gx = nx - 1;
                    dst[x] = src[gx];
                }
            }
        }
    }
    return 0;
}

/* test hooks: the deterministic elementary functions */
VRGEN_EXPORT double vrgen_det_log(double x) { return det_log(x); }
VRGEN_EXPORT double vrgen_det_exp_neg(double a) { return det_exp_neg(a); }
VRGEN_EXPORT void vrgen_det_sincos2pi(double u, double *s, double *c) { det_sincos2pi(u, s, c); }
