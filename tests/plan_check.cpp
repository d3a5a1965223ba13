// plan_check.cpp — brute-force check of the per-frame brick plan geometry (paper_1111_6661_b200/csrc/vr_plan.h) on
// the host: for random cameras, volumes and brick sizes, (1) every pixel whose ray owns a sample in a brick lies in
// that brick's screen rectangle (else the sort-last / chain kernels would never evaluate it), and (2) along every
// ray the owner bricks appear in ascending visibility key (C.7).  Built with g++ and run by tests/test_plan_geometry.py.
#include <cstdio>
#include <cstdlib>
#include <random>
#include <string>
#include <vector>

#include "../paper_1111_6661_b200/csrc/vr_plan.h"

using namespace vr;

static void cross(const double a[3], const double b[3], double c[3])
{
    c[0] = a[1] * b[2] - a[2] * b[1]; c[1] = a[2] * b[0] - a[0] * b[2]; c[2] = a[0] * b[1] - a[1] * b[0];
}
static void norm(double a[3]) { double l = std::sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]); for (int i = 0; i < 3; ++i) a[i] /= l; }

// ---------------------------------------------------------------- the configs' own geometry, float32 rays
// The kernels decide ownership from the float32 positions of C.1-C.3 (coordinates up to 4096, t up to 12000: a few
// 1e-3 voxel of rounding), the plan from exact geometry with 0.01 voxel and one pixel of slack.  This part repeats
// the check at the sizes, brick edges, image sizes and orbit cameras of cfg3, cfg4 and cfg5 with the float32
// operation sequence (restated here; the kernels' own code is exercised by the emulated parity tests at small size).
static bool ray32(const vr_camera &c, const int n[3], int i, int j, float d[3], float oc[3], float &t_first, float &t_exit)
{
    const float px = (float)i + 0.5f, py = (float)j + 0.5f;
    float o[3], g[3];
    for (int a = 0; a < 3; ++a) {
        o[a] = fmaf(py, c.ov[a], fmaf(px, c.ou[a], c.o0[a]));
        g[a] = fmaf(py, c.dv[a], fmaf(px, c.du[a], c.d0[a]));
    }
    const float len = sqrtf(fmaf(g[2], g[2], fmaf(g[1], g[1], g[0] * g[0])));
    float t_enter = 0.0f;
    t_exit = INFINITY;
    bool hit = true;
    for (int a = 0; a < 3; ++a) {
        d[a] = g[a] / len;
        float lo = -INFINITY, hi = INFINITY;
        if (d[a] != 0.0f) {
            const float inv = 1.0f / d[a], ta = (0.0f - o[a]) * inv, tb = ((float)n[a] - o[a]) * inv;
            lo = fminf(ta, tb); hi = fmaxf(ta, tb);
        } else if (o[a] < 0.0f || o[a] > (float)n[a]) hit = false;
        t_enter = fmaxf(t_enter, lo); t_exit = fminf(t_exit, hi);
        oc[a] = o[a] - 0.5f;
    }
    t_first = fmaf(0.5f, c.step, t_enter);
    return hit && t_exit > t_enter && t_exit < INFINITY;
}

static int check_configs()
{
    struct Cfg { const char *name; int n[3], B, W, H, views; float step; };
    const Cfg cfgs[] = { { "cfg3", { 1024, 1024, 2048 }, 128, 1920, 1080, 32, 0.5f },
                         { "cfg4", { 2048, 2048, 4096 }, 128, 3840, 2160, 64, 1.0f },
                         { "cfg5", { 4096, 4096, 3072 }, 256, 1920, 1080, 8, 0.5f } };
    std::mt19937_64 rng(4242);
    std::uniform_real_distribution<double> U(0.0, 1.0);
    long long samples = 0, rect_bad = 0, order_bad = 0;
    for (const Cfg &cf : cfgs) {
        const int *n = cf.n, B = cf.B;
        const int nb[3] = { (n[0] + B - 1) / B, (n[1] + B - 1) / B, (n[2] + B - 1) / B };
        for (int view = 0; view < cf.views; view += cf.views / 8) {
            // workload/cameras.py orbit_camera: elevation 20 deg, azimuth 2 pi (view + 1/4) / V, FOV 45 deg
            const double c[3] = { n[0] / 2.0, n[1] / 2.0, n[2] / 2.0 };
            const double rb = 0.5 * std::sqrt((double)n[0] * n[0] + (double)n[1] * n[1] + (double)n[2] * n[2]);
            const double R = rb / std::sin(M_PI / 8.0), th = 2.0 * M_PI * (view + 0.25) / cf.views, el = M_PI / 9.0;
            const double eye[3] = { c[0] + R * std::cos(el) * std::sin(th), c[1] + R * std::sin(el), c[2] + R * std::cos(el) * std::cos(th) };
            double f[3] = { c[0] - eye[0], c[1] - eye[1], c[2] - eye[2] }, up[3] = { 0, 1, 0 }, r[3], u[3];
            norm(f); cross(f, up, r); norm(r); cross(r, f, u);
            const double tf = std::tan(M_PI / 8.0), asp = (double)cf.W / cf.H;
            vr_camera cam;
            cam.struct_size = sizeof(cam); cam.width = cf.W; cam.height = cf.H; cam.step = cf.step; cam.ert_alpha = 0.0f; cam.flags = 0;
            for (int a = 0; a < 3; ++a) {
                cam.o0[a] = (float)eye[a]; cam.ou[a] = cam.ov[a] = 0.0f;
                cam.d0[a] = (float)(f[a] - tf * asp * r[a] - tf * u[a]);
                cam.du[a] = (float)(2.0 * tf * asp / cf.W * r[a]); cam.dv[a] = (float)(2.0 * tf / cf.H * u[a]);
            }
            struct Br { int x0, y0, x1, y1; double key; };
            std::vector<Br> br((size_t)nb[0] * nb[1] * nb[2]);
            for (int bz = 0; bz < nb[2]; ++bz) for (int by = 0; by < nb[1]; ++by) for (int bx = 0; bx < nb[0]; ++bx) {
                const int b[3] = { bx, by, bz };
                Br &k = br[bx + (size_t)nb[0] * (by + (size_t)nb[1] * bz)];
                double lo[3], hi[3];
                k.key = 0.0;
                for (int a = 0; a < 3; ++a) {
                    brick_cell(B * b[a], std::min(B * b[a] + B - 1, n[a] - 2), n[a], lo[a], hi[a]);
                    k.key += brick_key_term(true, (double)B, (unsigned)b[a], (double)cam.o0[a], (double)cam.d0[a]);
                }
                box_rect(&cam, true, lo, hi, k.x0, k.y0, k.x1, k.y1);
            }
            for (int s = 0; s < 1500; ++s) {
                const int i = (int)(U(rng) * cf.W), j = (int)(U(rng) * cf.H);
                float d[3], oc[3], t_first, t_exit;
                if (!ray32(cam, n, i, j, d, oc, t_first, t_exit)) continue;
                double last_key = -1e300;
                long long last_id = -1;
                for (int k = 0; k < (1 << 24); ++k) {
                    const float t = fmaf((float)k, cam.step, t_first);
                    if (!(t < t_exit)) break;
                    long long id = 0, mul = 1;
                    for (int a = 0; a < 3; ++a) {
                        float q = fmaf(t, d[a], oc[a]);
                        q = fminf(fmaxf(q, 0.0f), (float)(n[a] - 1));
                        const int i0 = std::min((int)floorf(q), n[a] - 2);
                        id += mul * (i0 / B); mul *= nb[a];
                    }
                    const Br &b = br[(size_t)id];
                    ++samples;
                    if (i < b.x0 || i >= b.x1 || j < b.y0 || j >= b.y1) ++rect_bad;
                    if (id != last_id) { if (b.key < last_key) ++order_bad; last_key = b.key; last_id = id; }
                }
            }
        }
    }
    printf("configs: samples %lld rect_bad %lld order_bad %lld\n", samples, rect_bad, order_bad);
    return (rect_bad || order_bad || samples < 10000000) ? 1 : 0;
}

int main(int argc, char **argv)
{
    if (argc > 2 && std::string(argv[2]) == "configs") return check_configs();
    const int n_cams = argc > 1 ? atoi(argv[1]) : 60;
    std::mt19937_64 rng(777);
    std::uniform_real_distribution<double> U(0.0, 1.0);
    long long samples = 0, rect_bad = 0, order_bad = 0, rays = 0;
    for (int ci = 0; ci < n_cams; ++ci) {
        const int n[3] = { 8 + (int)(U(rng) * 120), 8 + (int)(U(rng) * 120), 8 + (int)(U(rng) * 120) };
        const int B = 2 + (int)(U(rng) * 40);
        const int W = 40 + (int)(U(rng) * 160), H = 30 + (int)(U(rng) * 120);
        const bool ortho = ci % 4 == 3;
        double c[3] = { n[0] / 2.0, n[1] / 2.0, n[2] / 2.0 }, e[3] = { U(rng) - .5, U(rng) - .5, U(rng) - .5 };
        norm(e);
        const double R = (ortho ? 1.2 : 0.2 + 2.5 * U(rng)) * std::max(n[0], std::max(n[1], n[2]));   // perspective: also eyes inside
        double eye[3], f[3], up[3] = { 0, 1, 0 }, r[3], u[3];
        for (int a = 0; a < 3; ++a) { eye[a] = c[a] + R * e[a]; f[a] = -e[a]; }
        if (std::fabs(e[1]) > 0.9) { up[1] = 0; up[2] = 1; }
        cross(f, up, r); norm(r); cross(r, f, u);
        vr_camera cam;
        cam.struct_size = sizeof(cam); cam.width = W; cam.height = H; cam.step = 0.5f; cam.ert_alpha = 0.0f; cam.flags = 0;
        const double th = std::tan((15.0 + 60.0 * U(rng)) * M_PI / 360.0), asp = (double)W / H, ext = (0.6 + U(rng)) * n[1];
        for (int a = 0; a < 3; ++a) {
            if (!ortho) {
                cam.o0[a] = (float)eye[a]; cam.ou[a] = cam.ov[a] = 0.0f;
                cam.d0[a] = (float)(f[a] - th * asp * r[a] - th * u[a]);
                cam.du[a] = (float)(2.0 * th * asp / W * r[a]); cam.dv[a] = (float)(2.0 * th / H * u[a]);
            } else {
                cam.o0[a] = (float)(eye[a] - 0.5 * ext * asp * r[a] - 0.5 * ext * u[a]);
                cam.ou[a] = (float)(ext * asp / W * r[a]); cam.ov[a] = (float)(ext / H * u[a]);
                cam.d0[a] = (float)f[a]; cam.du[a] = cam.dv[a] = 0.0f;
            }
        }
        const bool persp = !ortho;
        const int nb[3] = { (n[0] + B - 1) / B, (n[1] + B - 1) / B, (n[2] + B - 1) / B };
        // the plan: rectangle and key per brick, as plan_bricks() forms them
        struct Br { int x0, y0, x1, y1; double key; bool empty; };
        std::vector<Br> br((size_t)nb[0] * nb[1] * nb[2]);
        for (int bz = 0; bz < nb[2]; ++bz) for (int by = 0; by < nb[1]; ++by) for (int bx = 0; bx < nb[0]; ++bx) {
            const int b[3] = { bx, by, bz };
            Br &k = br[bx + (size_t)nb[0] * (by + (size_t)nb[1] * bz)];
            double lo[3], hi[3];
            k.key = 0.0; k.empty = false;
            for (int a = 0; a < 3; ++a) {
                const int ilo = B * b[a], ihi = std::min(B * b[a] + B - 1, n[a] - 2);
                if (ilo > ihi) k.empty = true;
                brick_cell(ilo, ihi, n[a], lo[a], hi[a]);
                k.key += brick_key_term(persp, (double)B, (unsigned)b[a], (double)cam.o0[a], (double)cam.d0[a]);
            }
            if (!k.empty) box_rect(&cam, persp, lo, hi, k.x0, k.y0, k.x1, k.y1);
        }
        for (int s = 0; s < 3000; ++s) {
            const int i = (int)(U(rng) * W), j = (int)(U(rng) * H);
            double o[3], g[3];
            for (int a = 0; a < 3; ++a) {
                o[a] = (double)cam.o0[a] + (i + .5) * (double)cam.ou[a] + (j + .5) * (double)cam.ov[a];
                g[a] = (double)cam.d0[a] + (i + .5) * (double)cam.du[a] + (j + .5) * (double)cam.dv[a];
            }
            norm(g);
            double t0 = 0.0, t1 = 1e300;
            bool hit = true;
            for (int a = 0; a < 3; ++a) {
                if (g[a] != 0.0) {
                    const double ta = (0 - o[a]) / g[a], tb = (n[a] - o[a]) / g[a];
                    t0 = std::max(t0, std::min(ta, tb)); t1 = std::min(t1, std::max(ta, tb));
                } else if (o[a] < 0 || o[a] > n[a]) hit = false;
            }
            if (!hit || !(t1 > t0)) continue;
            ++rays;
            double last_key = -1e300;
            long long last_id = -1;
            for (double t = t0 + 0.25; t < t1; t += 0.5) {
                long long id = 0, mul = 1;
                for (int a = 0; a < 3; ++a) {
                    int i0 = (int)std::floor(o[a] + t * g[a] - 0.5);
                    i0 = std::min(std::max(i0, 0), n[a] - 2);
                    id += mul * (i0 / B); mul *= nb[a];
                }
                const Br &k = br[(size_t)id];
                ++samples;
                if (k.empty || i < k.x0 || i >= k.x1 || j < k.y0 || j >= k.y1) ++rect_bad;
                if (id != last_id) {
                    if (k.key < last_key) ++order_bad;
                    last_key = k.key; last_id = id;
                }
            }
        }
    }
    printf("rays %lld samples %lld rect_bad %lld order_bad %lld\n", rays, samples, rect_bad, order_bad);
    return (rect_bad || order_bad || samples < 1000000) ? 1 : 0;
}
