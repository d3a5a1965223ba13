/*
 * vr_oracle.c — CPU ORACLE for the bricked volume ray-caster and the data-summary
 * passes.  TEST INFRASTRUCTURE ONLY: plain, slow, obviously-correct loops.  Only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this.  It shares no code with paper_1111_6661_b200/csrc/ and
 * includes none of its headers.
 *
 * The paper names the operation — ray-cast volume rendering
 * of float spectral cubes, plus min/max and histogram, median
 * and standard deviation (L66), a viewer that only displays results (L48, L70) —
 * but gives no formulae; every step below follows the readings fixed in SURVEY.md
 * §8(c) C.0–C.8 and DESIGN.md §3 C.13 (statistics), C.14 (8-bit frame), S41
 * (histogram ranges that overflow the bin arithmetic), in that order and notation.
 *
 * Two precisions:
 *   f32-canonical (the parity gate): the exact binary32 operation sequence of
 *     C.1–C.7; fmaf = one correctly rounded fused multiply-add; nothing else is
 *     contracted (build with -ffp-contract=off -mfma, no fast-math).
 *   f64-truth (reported distance only): the same algorithm in plain double.
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"): P1 axis-aligned ortho MIP ==
 * per-column max (bit-exact); P2 constant cube => A = 1-(1-a)^K; P3 bricked ==
 * unbricked; P4 min/max/hist == brute force; P5 affine cube; P6 impulse tent;
 * P7 alpha 0 / alpha 1; P8 sample counts; P9/P10 mirror symmetry; P11 ERT bound;
 * P12 f32 vs f64 distance; P13 step-halving convergence; P14 halo layout; P15
 * non-finite voxels in a render (S24); P16 mean / standard deviation / median
 * (closed forms, numpy float64 moments, np.sort rank); P17 8-bit frame (every byte,
 * ties, clamps, against the float64 formula).  No function here is "parity
 * unpinned"; all pins are self-consistency pins (the paper prints no number).
 *
 * Build: gcc -O2 -fopenmp -mfma -ffp-contract=off -shared -fPIC vr_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORACLE_EXPORT __attribute__((visibility("default")))

enum { ORACLE_EA = 0, ORACLE_MIP = 1 };
enum { ORACLE_F32 = 0, ORACLE_F64 = 1 };
enum { ORACLE_LINEAR = 0, ORACLE_BRICKED_HALO1 = 1 };

typedef struct {
    uint32_t struct_size, width, height;
    float o0[3], ou[3], ov[3];      /* origin(i,j) = o0 + (i+.5)ou + (j+.5)ov            */
    float d0[3], du[3], dv[3];      /* dir(i,j)    = normalize(d0 + (i+.5)du + (j+.5)dv) */
    float step, ert_alpha;
} oracle_camera;

typedef struct {
    uint32_t struct_size;
    uint32_t nx, ny, nz;
    uint32_t layout, layout_brick;  /* ORACLE_LINEAR, or brick-major (B+1)^3 with high-side halo */
    const float *vol;
    const float *tf;                /* 256*4 rgba (EA) */
    float vmin, vmax;
    int32_t mode, precision;
    uint32_t brick;                 /* 0: one march per ray.  >0 (and ert_alpha == 0): per-brick
                                       partials folded in visibility-key order (C.7) */
    const uint8_t *mask;            /* optional W*H; 0 = skip pixel (outputs untouched) */
    float *image;                   /* W*H*4 (EA) or W*H (MIP) */
    double *image64;                /* optional, f64-truth results unrounded */
    int32_t *K;                     /* optional W*H: nominal sample count per pixel (C.2) */
    int32_t *K_ert;                 /* optional W*H: samples up to and including the ERT stop */
    uint8_t *fragile;               /* optional W*H: ERT-fragile flag (S14) */
    uint64_t n_nominal, n_ert;      /* out: sums over rendered pixels */
    uint64_t n_noncontig;           /* out (bricked): rays whose owner runs were not contiguous */
    uint64_t n_order_mismatch;      /* out (bricked): rays whose key order != order along the ray */
} oracle_render_args;

/* ------------------------------------------------------------------ */
/* voxel access (C.0: x fastest; value at the voxel centre)           */
/* ------------------------------------------------------------------ */
typedef struct { const float *v; int64_t nx, ny, nz; int layout; int64_t B, nbx, nby; } volume;

static inline float vox_linear(const volume *V, int64_t x, int64_t y, int64_t z)
{
    return V->v[x + V->nx * (y + V->ny * z)];
}
/* brick-major with +1 high-side halo: corner (dx,dy,dz) of base index (x,y,z) is read from the
 * brick that OWNS the base index, so the halo voxels themselves are exercised */
static inline float vox_corner(const volume *V, int64_t x, int64_t y, int64_t z, int dx, int dy, int dz)
{
    if (V->layout == ORACLE_LINEAR) return vox_linear(V, x + dx, y + dy, z + dz);
    int64_t B = V->B, E = B + 1;
    int64_t bx = x / B, by = y / B, bz = z / B;
    int64_t b = bx + V->nbx * (by + V->nby * bz);
    int64_t lx = x - bx * B + dx, ly = y - by * B + dy, lz = z - bz * B + dz;
    return V->v[b * E * E * E + lx + E * (ly + E * lz)];
}

/* exact-ends lerp (C.0): returns a at f=0 and b at f=1 exactly */
static inline float L32(float a, float b, float f) { return fmaf(f, b, fmaf(-f, a, a)); }
static inline double L64(double a, double b, double f) { return f * b + (a - f * a); }

/* ------------------------------------------------------------------ */
/* f32-canonical ray                                                   */
/* ------------------------------------------------------------------ */
typedef struct { float o[3], d[3], oc[3], t_enter, t_exit, t_first; int hit; } ray32;

static void make_ray32(const oracle_camera *c, const float n[3], int i, int j, ray32 *r)
{
    /* C.1 */
    float px = (float)i + 0.5f, py = (float)j + 0.5f, g[3];
    for (int a = 0; a < 3; ++a) {
        r->o[a] = fmaf(py, c->ov[a], fmaf(px, c->ou[a], c->o0[a]));
        g[a] = fmaf(py, c->dv[a], fmaf(px, c->du[a], c->d0[a]));
    }
    float len = sqrtf(fmaf(g[2], g[2], fmaf(g[1], g[1], g[0] * g[0])));
    for (int a = 0; a < 3; ++a) r->d[a] = g[a] / len;
    /* C.2 */
    float t_enter = 0.0f, t_exit = INFINITY;
    r->hit = 1;
    for (int a = 0; a < 3; ++a) {
        float lo, hi;
        if (r->d[a] != 0.0f) {
            float inv = 1.0f / r->d[a];
            float ta = (0.0f - r->o[a]) * inv, tb = (n[a] - r->o[a]) * inv;
            lo = fminf(ta, tb); hi = fmaxf(ta, tb);
        } else {
            if (r->o[a] < 0.0f || r->o[a] > n[a]) r->hit = 0;
            lo = -INFINITY; hi = INFINITY;
        }
        t_enter = fmaxf(t_enter, lo);
        t_exit = fminf(t_exit, hi);
    }
    if (!(t_exit > t_enter)) r->hit = 0;
    r->t_enter = t_enter; r->t_exit = t_exit;
    r->t_first = fmaf(0.5f, c->step, t_enter);
    /* C.3 */
    for (int a = 0; a < 3; ++a) r->oc[a] = r->o[a] - 0.5f;
}

/* C.3: reconstruction at t; returns s and the clamped base index i0[3] */
static inline float sample32(const volume *V, const ray32 *r, float t, int64_t i0[3])
{
    const int64_t nn[3] = { V->nx, V->ny, V->nz };
    float f[3];
    for (int a = 0; a < 3; ++a) {
        float q = fmaf(t, r->d[a], r->oc[a]);
        q = fminf(fmaxf(q, 0.0f), (float)(nn[a] - 1));
        int64_t i = (int64_t)floorf(q);
        if (i > nn[a] - 2) i = nn[a] - 2;
        f[a] = q - (float)i;
        i0[a] = i;
    }
    int64_t x = i0[0], y = i0[1], z = i0[2];
    float c00 = L32(vox_corner(V, x, y, z, 0, 0, 0), vox_corner(V, x, y, z, 1, 0, 0), f[0]);
    float c10 = L32(vox_corner(V, x, y, z, 0, 1, 0), vox_corner(V, x, y, z, 1, 1, 0), f[0]);
    float c01 = L32(vox_corner(V, x, y, z, 0, 0, 1), vox_corner(V, x, y, z, 1, 0, 1), f[0]);
    float c11 = L32(vox_corner(V, x, y, z, 0, 1, 1), vox_corner(V, x, y, z, 1, 1, 1), f[0]);
    float c0 = L32(c00, c10, f[1]);
    float c1 = L32(c01, c11, f[1]);
    return L32(c0, c1, f[2]);
}

/* C.4: post-interpolative classification, linear between table entries */
static inline void classify32(const float *tf, float scale, float bias, float s, float rgba[4])
{
    float u = fminf(fmaxf(fmaf(s, scale, bias), 0.0f), 1.0f);   /* NaN -> 0 */
    float x = u * 255.0f;
    int i = (int)x;
    if (i > 254) i = 254;
    float f = x - (float)i;
    for (int c = 0; c < 4; ++c) rgba[c] = L32(tf[4 * i + c], tf[4 * (i + 1) + c], f);
}

/* ------------------------------------------------------------------ */
/* f64-truth twins (same algorithm, plain double)                      */
/* ------------------------------------------------------------------ */
typedef struct { double o[3], d[3], oc[3], t_enter, t_exit, t_first; int hit; } ray64;

static void make_ray64(const oracle_camera *c, const double n[3], int i, int j, ray64 *r)
{
    double px = (double)i + 0.5, py = (double)j + 0.5, g[3];
    for (int a = 0; a < 3; ++a) {
        r->o[a] = (double)c->o0[a] + px * (double)c->ou[a] + py * (double)c->ov[a];
        g[a] = (double)c->d0[a] + px * (double)c->du[a] + py * (double)c->dv[a];
    }
    double len = sqrt(g[0] * g[0] + g[1] * g[1] + g[2] * g[2]);
    for (int a = 0; a < 3; ++a) r->d[a] = g[a] / len;
    double t_enter = 0.0, t_exit = INFINITY;
    r->hit = 1;
    for (int a = 0; a < 3; ++a) {
        double lo, hi;
        if (r->d[a] != 0.0) {
            double inv = 1.0 / r->d[a];
            double ta = (0.0 - r->o[a]) * inv, tb = (n[a] - r->o[a]) * inv;
            lo = fmin(ta, tb); hi = fmax(ta, tb);
        } else {
            if (r->o[a] < 0.0 || r->o[a] > n[a]) r->hit = 0;
            lo = -INFINITY; hi = INFINITY;
        }
        t_enter = fmax(t_enter, lo);
        t_exit = fmin(t_exit, hi);
    }
    if (!(t_exit > t_enter)) r->hit = 0;
    r->t_enter = t_enter; r->t_exit = t_exit;
    r->t_first = t_enter + 0.5 * (double)c->step;
    for (int a = 0; a < 3; ++a) r->oc[a] = r->o[a] - 0.5;
}

static inline double sample64(const volume *V, const ray64 *r, double t, int64_t i0[3])
{
    const int64_t nn[3] = { V->nx, V->ny, V->nz };
    double f[3];
    for (int a = 0; a < 3; ++a) {
        double q = r->oc[a] + t * r->d[a];
        q = fmin(fmax(q, 0.0), (double)(nn[a] - 1));
        int64_t i = (int64_t)floor(q);
        if (i > nn[a] - 2) i = nn[a] - 2;
        f[a] = q - (double)i;
        i0[a] = i;
    }
    int64_t x = i0[0], y = i0[1], z = i0[2];
    double c00 = L64(vox_corner(V, x, y, z, 0, 0, 0), vox_corner(V, x, y, z, 1, 0, 0), f[0]);
    double c10 = L64(vox_corner(V, x, y, z, 0, 1, 0), vox_corner(V, x, y, z, 1, 1, 0), f[0]);
    double c01 = L64(vox_corner(V, x, y, z, 0, 0, 1), vox_corner(V, x, y, z, 1, 0, 1), f[0]);
    double c11 = L64(vox_corner(V, x, y, z, 0, 1, 1), vox_corner(V, x, y, z, 1, 1, 1), f[0]);
    double c0 = L64(c00, c10, f[1]);
    double c1 = L64(c01, c11, f[1]);
    return L64(c0, c1, f[2]);
}

static inline void classify64(const float *tf, double scale, double bias, double s, double rgba[4])
{
    double u = fmin(fmax(s * scale + bias, 0.0), 1.0);
    double x = u * 255.0;
    int i = (int)x;
    if (i > 254) i = 254;
    double f = x - (double)i;
    for (int c = 0; c < 4; ++c) rgba[c] = L64((double)tf[4 * i + c], (double)tf[4 * (i + 1) + c], f);
}

/* ------------------------------------------------------------------ */
/* per-brick partials (C.7)                                            */
/* ------------------------------------------------------------------ */
typedef struct { int64_t id; double key; float C[3], T, m; double C64[3], T64, m64; } run_t;

static double brick_key(const oracle_camera *c, int perspective, int64_t B, const int64_t b[3])
{
    double key = 0.0;
    for (int a = 0; a < 3; ++a) {
        double centre = (double)B * ((double)b[a] + 0.5) + 0.5;     /* ownership-lattice centre */
        if (perspective) { double e = (double)c->o0[a] - centre; key += e * e; }
        else key += centre * (double)c->d0[a];
    }
    return key;
}

static int is_zero3(const float v[3]) { return v[0] == 0.0f && v[1] == 0.0f && v[2] == 0.0f; }

/* ------------------------------------------------------------------ */
/* the renderer                                                        */
/* ------------------------------------------------------------------ */
ORACLE_EXPORT int oracle_render(const oracle_camera *cam, oracle_render_args *A)
{
    if (!cam || !A || cam->struct_size != sizeof(oracle_camera) || A->struct_size != sizeof(oracle_render_args))
        return -1;
    if (!A->vol || !A->image || A->nx < 2 || A->ny < 2 || A->nz < 2) return -2;
    if (A->mode == ORACLE_EA && (!A->tf || !(A->vmax > A->vmin))) return -3;
    if (!(cam->step > 0.0f) || cam->ert_alpha < 0.0f || cam->ert_alpha >= 1.0f) return -4;

    volume V = { A->vol, A->nx, A->ny, A->nz, (int)A->layout, (int64_t)A->layout_brick, 0, 0 };
    if (V.layout == ORACLE_BRICKED_HALO1) {
        if (!V.B) return -5;
        V.nbx = (V.nx + V.B - 1) / V.B; V.nby = (V.ny + V.B - 1) / V.B;
    }
    const int W = (int)cam->width, H = (int)cam->height;
    const int ch = A->mode == ORACLE_EA ? 4 : 1;
    const int ert_on = cam->ert_alpha > 0.0f && A->mode == ORACLE_EA;
    const int bricked = A->brick > 0 && !ert_on;    /* C.7: ERT => single march */
    const int64_t B = (int64_t)A->brick;
    int perspective = is_zero3(cam->ou) && is_zero3(cam->ov);
    int ortho = is_zero3(cam->du) && is_zero3(cam->dv);
    if (bricked && !perspective && !ortho) return -6;
    const int64_t nbx = bricked ? (V.nx + B - 1) / B : 1, nby = bricked ? (V.ny + B - 1) / B : 1,
                  nbz = bricked ? (V.nz + B - 1) / B : 1;
    const int max_runs = (int)(nbx + nby + nbz + 8);

    /* C.4 set-up */
    const float scale32 = A->mode == ORACLE_EA ? 1.0f / (A->vmax - A->vmin) : 0.0f;
    const float bias32 = -A->vmin * scale32;
    const double scale64 = A->mode == ORACLE_EA ? 1.0 / ((double)A->vmax - (double)A->vmin) : 0.0;
    const double bias64 = -(double)A->vmin * scale64;
    const float Tmin32 = 1.0f - cam->ert_alpha;
    const double Tmin64 = 1.0 - (double)cam->ert_alpha;
    const float n32[3] = { (float)A->nx, (float)A->ny, (float)A->nz };
    const double n64[3] = { (double)A->nx, (double)A->ny, (double)A->nz };

    uint64_t n_nominal = 0, n_ert = 0, n_noncontig = 0, n_mismatch = 0;

#pragma omp parallel reduction(+ : n_nominal, n_ert, n_noncontig, n_mismatch)
    {
        run_t *runs = (run_t *)malloc(sizeof(run_t) * (size_t)max_runs);
#pragma omp for schedule(dynamic, 1)
        for (int j = 0; j < H; ++j)
            for (int i = 0; i < W; ++i) {
                const size_t p = (size_t)j * W + i;
                if (A->mask && !A->mask[p]) continue;
                int32_t K = 0, Kert = 0;
                int frag = 0, nruns = 0, overflow = 0;
                float out32[4] = { 0, 0, 0, 0 };
                double out64[4] = { 0, 0, 0, 0 };

                if (A->precision == ORACLE_F32) {
                    ray32 r; make_ray32(cam, n32, i, j, &r);
                    float C[3] = { 0, 0, 0 }, T = 1.0f, m = -INFINITY;
                    int stopped = 0;
                    if (r.hit)
                        for (int32_t k = 0;; ++k) {
                            float t = fmaf((float)k, cam->step, r.t_first);
                            if (!(t < r.t_exit)) break;          /* C.2: sample k exists iff t_k < t_exit */
                            ++K;
                            if (stopped) continue;               /* after ERT only K keeps counting */
                            int64_t i0[3];
                            float s = sample32(&V, &r, t, i0);
                            run_t *R = NULL;
                            if (bricked) {
                                int64_t b[3] = { i0[0] / B, i0[1] / B, i0[2] / B };
                                int64_t id = b[0] + nbx * (b[1] + nby * b[2]);
                                if (nruns == 0 || runs[nruns - 1].id != id) {
                                    if (nruns == max_runs) { overflow = 1; nruns = max_runs - 1; }
                                    R = &runs[nruns++];
                                    R->id = id; R->key = brick_key(cam, perspective, B, b);
                                    R->C[0] = R->C[1] = R->C[2] = 0.0f; R->T = 1.0f; R->m = -INFINITY;
                                } else R = &runs[nruns - 1];
                            }
                            if (A->mode == ORACLE_MIP) {
                                if (bricked) R->m = fmaxf(R->m, s); else m = fmaxf(m, s);      /* C.6 */
                            } else {
                                float rgba[4]; classify32(A->tf, scale32, bias32, s, rgba);
                                float *Cc = bricked ? R->C : C;
                                float *Tc = bricked ? &R->T : &T;
                                float w = *Tc * rgba[3];                                      /* C.5 */
                                for (int c = 0; c < 3; ++c) Cc[c] = fmaf(w, rgba[c], Cc[c]);
                                *Tc = *Tc - w;
                                ++Kert;
                                if (ert_on) {
                                    if (fabsf(*Tc - Tmin32) <= 1e-5f) frag = 1;               /* S14 */
                                    if (*Tc <= Tmin32) stopped = 1;
                                }
                            }
                        }
                    if (bricked) {      /* C.7: fold partials in visibility-key order */
                        for (int a = 0; a < nruns; ++a)
                            for (int b2 = a + 1; b2 < nruns; ++b2)
                                if (runs[a].id == runs[b2].id) { overflow = 1; }
                        int mism = 0;
                        for (int a = 1; a < nruns; ++a) {         /* stable insertion sort by key */
                            run_t tmp = runs[a]; int b2 = a - 1;
                            while (b2 >= 0 && runs[b2].key > tmp.key) { runs[b2 + 1] = runs[b2]; --b2; mism = 1; }
                            runs[b2 + 1] = tmp;
                        }
                        n_noncontig += (uint64_t)overflow; n_mismatch += (uint64_t)mism;
                        for (int a = 0; a < nruns; ++a) {
                            if (A->mode == ORACLE_MIP) m = fmaxf(m, runs[a].m);
                            else {
                                for (int c = 0; c < 3; ++c) C[c] = fmaf(T, runs[a].C[c], C[c]);
                                T = T * runs[a].T;
                            }
                        }
                    }
                    if (A->mode == ORACLE_MIP) { out32[0] = m; out64[0] = (double)m; }
                    else {
                        out32[0] = C[0]; out32[1] = C[1]; out32[2] = C[2]; out32[3] = 1.0f - T;
                        for (int c = 0; c < 4; ++c) out64[c] = (double)out32[c];
                    }
                } else {
                    ray64 r; make_ray64(cam, n64, i, j, &r);
                    double C[3] = { 0, 0, 0 }, T = 1.0, m = -INFINITY;
                    int stopped = 0;
                    if (r.hit)
                        for (int32_t k = 0;; ++k) {
                            double t = r.t_first + (double)k * (double)cam->step;
                            if (!(t < r.t_exit)) break;
                            ++K;
                            if (stopped) continue;
                            int64_t i0[3];
                            double s = sample64(&V, &r, t, i0);
                            run_t *R = NULL;
                            if (bricked) {
                                int64_t b[3] = { i0[0] / B, i0[1] / B, i0[2] / B };
                                int64_t id = b[0] + nbx * (b[1] + nby * b[2]);
                                if (nruns == 0 || runs[nruns - 1].id != id) {
                                    if (nruns == max_runs) { overflow = 1; nruns = max_runs - 1; }
                                    R = &runs[nruns++];
                                    R->id = id; R->key = brick_key(cam, perspective, B, b);
                                    R->C64[0] = R->C64[1] = R->C64[2] = 0.0; R->T64 = 1.0; R->m64 = -INFINITY;
                                } else R = &runs[nruns - 1];
                            }
                            if (A->mode == ORACLE_MIP) {
                                if (bricked) R->m64 = fmax(R->m64, s); else m = fmax(m, s);
                            } else {
                                double rgba[4]; classify64(A->tf, scale64, bias64, s, rgba);
                                double *Cc = bricked ? R->C64 : C;
                                double *Tc = bricked ? &R->T64 : &T;
                                double w = *Tc * rgba[3];
                                for (int c = 0; c < 3; ++c) Cc[c] = Cc[c] + w * rgba[c];
                                *Tc = *Tc - w;
                                ++Kert;
                                if (ert_on) {
                                    if (fabs(*Tc - Tmin64) <= 1e-5) frag = 1;
                                    if (*Tc <= Tmin64) stopped = 1;
                                }
                            }
                        }
                    if (bricked) {
                        for (int a = 0; a < nruns; ++a)
                            for (int b2 = a + 1; b2 < nruns; ++b2)
                                if (runs[a].id == runs[b2].id) { overflow = 1; }
                        int mism = 0;
                        for (int a = 1; a < nruns; ++a) {
                            run_t tmp = runs[a]; int b2 = a - 1;
                            while (b2 >= 0 && runs[b2].key > tmp.key) { runs[b2 + 1] = runs[b2]; --b2; mism = 1; }
                            runs[b2 + 1] = tmp;
                        }
                        n_noncontig += (uint64_t)overflow; n_mismatch += (uint64_t)mism;
                        for (int a = 0; a < nruns; ++a) {
                            if (A->mode == ORACLE_MIP) m = fmax(m, runs[a].m64);
                            else {
                                for (int c = 0; c < 3; ++c) C[c] = C[c] + T * runs[a].C64[c];
                                T = T * runs[a].T64;
                            }
                        }
                    }
                    if (A->mode == ORACLE_MIP) { out64[0] = m; out32[0] = (float)m; }
                    else {
                        out64[0] = C[0]; out64[1] = C[1]; out64[2] = C[2]; out64[3] = 1.0 - T;
                        for (int c = 0; c < 4; ++c) out32[c] = (float)out64[c];
                    }
                }
                if (A->mode == ORACLE_MIP) Kert = K;
                for (int c = 0; c < ch; ++c) A->image[p * ch + c] = out32[c];
                if (A->image64) for (int c = 0; c < ch; ++c) A->image64[p * ch + c] = out64[c];
                if (A->K) A->K[p] = K;
                if (A->K_ert) A->K_ert[p] = Kert;
                if (A->fragile) A->fragile[p] = (uint8_t)frag;
                n_nominal += (uint64_t)K; n_ert += (uint64_t)Kert;
            }
        free(runs);
    }
    A->n_nominal = n_nominal; A->n_ert = n_ert;
    A->n_noncontig = n_noncontig; A->n_order_mismatch = n_mismatch;
    return 0;
}

/* ------------------------------------------------------------------ */
/* C.8: min/max over finite voxels + histogram                         */
/* ------------------------------------------------------------------ */
typedef struct {
    float vmin, vmax;
    uint64_t n_nonfinite, n_below, n_above;
} oracle_summary_head;

/* counts[nbins] follows the head.  range = NULL => [vmin, vmax] of the finite voxels.
 * layout/brick as above: halo voxels of a bricked layout are NOT counted. */
ORACLE_EXPORT int oracle_minmax_hist(const float *vol, uint32_t nx, uint32_t ny, uint32_t nz, uint32_t layout,
                                     uint32_t layout_brick, uint32_t nbins, const float *range,
                                     oracle_summary_head *head, uint64_t *counts)
{
    if (!vol || !head || !counts || !nbins || !nx || !ny || !nz) return -1;
    volume V = { vol, nx, ny, nz, (int)layout, (int64_t)layout_brick, 0, 0 };
    if (V.layout == ORACLE_BRICKED_HALO1) {
        if (!V.B) return -5;
        V.nbx = (V.nx + V.B - 1) / V.B; V.nby = (V.ny + V.B - 1) / V.B;
    }
    float vmin = INFINITY, vmax = -INFINITY;
    uint64_t nonfinite = 0;
#pragma omp parallel for reduction(min : vmin) reduction(max : vmax) reduction(+ : nonfinite)
    for (int64_t z = 0; z < V.nz; ++z)
        for (int64_t y = 0; y < V.ny; ++y)
            for (int64_t x = 0; x < V.nx; ++x) {
                float v = vox_corner(&V, x, y, z, 0, 0, 0);
                if (!isfinite(v)) { ++nonfinite; continue; }
                if (v < vmin) vmin = v;
                if (v > vmax) vmax = v;
            }
    head->vmin = vmin; head->vmax = vmax; head->n_nonfinite = nonfinite;
    for (uint32_t b = 0; b < nbins; ++b) counts[b] = 0;
    float lo = range ? range[0] : vmin, hi = range ? range[1] : vmax;
    float scale_h = (hi == lo) ? 0.0f : (float)nbins / (hi - lo);
    uint64_t n_below = 0, n_above = 0;
#pragma omp parallel for reduction(+ : n_below, n_above, counts[:nbins])
    for (int64_t z = 0; z < V.nz; ++z)
        for (int64_t y = 0; y < V.ny; ++y)
            for (int64_t x = 0; x < V.nx; ++x) {
                float v = vox_corner(&V, x, y, z, 0, 0, 0);
                if (!isfinite(v)) continue;
                if (v < lo) { ++n_below; continue; }
                if (v > hi) { ++n_above; continue; }
                float t = (v - lo) * scale_h;
                /* S41: a range so narrow or so wide that the bin arithmetic overflows gives t = +inf or NaN
                 * (inf * 0); the conversion is then DEFINED as: NaN -> bin 0, t >= nbins -> last bin */
                int64_t b = t != t ? 0 : t >= (float)nbins ? (int64_t)nbins - 1 : (int64_t)t;
                counts[b]++;
            }
    head->n_below = n_below; head->n_above = n_above;
    return 0;
}

/* ------------------------------------------------------------------ */
/* C.13: mean, standard deviation, median over finite voxels           */
/* (the "global view" statistics of PAPER.md:L66; readings S35-S37)    */
/* ------------------------------------------------------------------ */
typedef struct {
    uint64_t n_finite, n_nonfinite;
    double mean;        /* S35: sum(v)/n over finite voxels, accumulated in double */
    double stddev;      /* S36: POPULATION standard deviation sqrt(sum((v-mean)^2)/n), second pass, double */
    float median;       /* S37: LOWER median = the element of rank floor((n-1)/2) (0-based) of the finite voxels
                           sorted by value, -0 before +0 (IEEE totalOrder); a data value, so bit-exact */
    float pad;
} oracle_stats;

/* order-preserving key of a float: a < b (totalOrder) <=> key(a) < key(b) */
static inline uint32_t total_order_key(float f)
{
    uint32_t b; memcpy(&b, &f, 4);
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
static int cmp_key(const void *a, const void *b)
{
    uint32_t x = *(const uint32_t *)a, y = *(const uint32_t *)b;
    return x < y ? -1 : x > y ? 1 : 0;
}

/* Plain definition: gather the finite voxels (halo voxels of a bricked layout excluded), Neumaier-compensated
 * double sums in voxel order for the two moments, qsort of the keys for the median. */
ORACLE_EXPORT int oracle_statistics(const float *vol, uint32_t nx, uint32_t ny, uint32_t nz, uint32_t layout,
                                    uint32_t layout_brick, oracle_stats *out)
{
    if (!vol || !out || !nx || !ny || !nz) return -1;
    volume V = { vol, nx, ny, nz, (int)layout, (int64_t)layout_brick, 0, 0 };
    if (V.layout == ORACLE_BRICKED_HALO1) {
        if (!V.B) return -5;
        V.nbx = (V.nx + V.B - 1) / V.B; V.nby = (V.ny + V.B - 1) / V.B;
    }
    const uint64_t N = (uint64_t)nx * ny * nz;
    uint32_t *keys = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)N);
    if (!keys) return -7;
    uint64_t n = 0, nonfinite = 0;
    double sum = 0.0, comp = 0.0;
    for (int64_t z = 0; z < V.nz; ++z)
        for (int64_t y = 0; y < V.ny; ++y)
            for (int64_t x = 0; x < V.nx; ++x) {
                float v = vox_corner(&V, x, y, z, 0, 0, 0);
                if (!isfinite(v)) { ++nonfinite; continue; }
                keys[n++] = total_order_key(v);
                double t = sum + (double)v;                       /* Neumaier */
                comp += fabs(sum) >= fabs((double)v) ? (sum - t) + (double)v : ((double)v - t) + sum;
                sum = t;
            }
    out->n_finite = n; out->n_nonfinite = nonfinite;
    out->mean = 0.0; out->stddev = 0.0; out->median = 0.0f; out->pad = 0.0f;
    if (n == 0) { free(keys); out->mean = NAN; out->stddev = NAN; out->median = NAN; return 0; }
    const double mean = (sum + comp) / (double)n;
    double ss = 0.0, sc = 0.0;
    for (int64_t z = 0; z < V.nz; ++z)
        for (int64_t y = 0; y < V.ny; ++y)
            for (int64_t x = 0; x < V.nx; ++x) {
                float v = vox_corner(&V, x, y, z, 0, 0, 0);
                if (!isfinite(v)) continue;
                double d = (double)v - mean, q = d * d;
                double t = ss + q;
                sc += ss >= q ? (ss - t) + q : (q - t) + ss;
                ss = t;
            }
    out->mean = mean;
    out->stddev = sqrt((ss + sc) / (double)n);
    qsort(keys, (size_t)n, sizeof(uint32_t), cmp_key);
    uint32_t k = keys[(n - 1) / 2];
    uint32_t bits = (k & 0x80000000u) ? (k & 0x7fffffffu) : ~k;
    memcpy(&out->median, &bits, 4);
    free(keys);
    return 0;
}

/* ------------------------------------------------------------------ */
/* C.14: 8-bit frame for delivery to a thin client                     */
/* (the headless "service" side of PAPER.md:L48, L70; reading S40)     */
/* ------------------------------------------------------------------ */
/* EA image (premultiplied C, opacity A): the frame is composited over an opaque constant background,
 * x_c = fmaf(1 - A, bg_c, C_c), clamped to [0,1] (NaN -> 0), byte = round-half-even(x_c * 255); alpha byte 255.
 * MIP image (scalar m, miss = -inf): grey ramp u = sat(fmaf(m, scale, bias)) with scale = 1/(vmax - vmin),
 * bias = -vmin * scale (as C.4), byte = round-half-even(u * 255) in r, g, b; alpha byte 255.
 * img: [H][W][4] or [H][W] floats with a row pitch in floats; out: [H][W][4] bytes, tightly packed. */
static inline uint8_t byte_of_unit(float x)
{
    x = x != x ? 0.0f : fminf(fmaxf(x, 0.0f), 1.0f);
    return (uint8_t)lrintf(x * 255.0f);              /* default rounding mode: to nearest, ties to even */
}

ORACLE_EXPORT int oracle_encode_rgba8(const float *img, uint32_t W, uint32_t H, uint64_t pitch_f, int mode,
                                      const float bg[3], float vmin, float vmax, uint8_t *out)
{
    if (!img || !out || !W || !H) return -1;
    const float scale = 1.0f / (vmax - vmin), bias = -vmin * scale;
    for (uint32_t j = 0; j < H; ++j)
        for (uint32_t i = 0; i < W; ++i) {
            uint8_t *o = out + 4 * ((size_t)j * W + i);
            if (mode == ORACLE_EA) {
                const float *p = img + (size_t)j * pitch_f + 4 * (size_t)i;
                const float w = 1.0f - p[3];
                for (int c = 0; c < 3; ++c) o[c] = byte_of_unit(fmaf(w, bg[c], p[c]));
            } else {
                const uint8_t g = byte_of_unit(fmaf(img[(size_t)j * pitch_f + i], scale, bias));
                o[0] = o[1] = o[2] = g;
            }
            o[3] = 255;
        }
    return 0;
}

ORACLE_EXPORT int oracle_num_threads(void)
{
    int n = 1;
#ifdef _OPENMP
    extern int omp_get_max_threads(void);
    n = omp_get_max_threads();
#endif
    return n;
}
