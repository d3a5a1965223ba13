// geom_check.cu — brute-force check of the beam geometry of vr_beamgeom.cuh on the HOST (no GPU): for random
// cameras, volumes and beams, every sample position a ray of the beam can take must read only voxels inside
// plane_rect() of the two data planes it touches (a voxel outside would be read from stale shared memory); and a
// host model of the kernel's step loop runs the kernel's own schedule functions over random beams.
// Built and run by tests/test_beam_geometry.py (nvcc compiles it as host code).  Test infrastructure.
#include <cstdio>
#include <cstdlib>
#include <cmath>
#include <random>
#include <vector>

#include "../paper_1111_6661_b200/csrc/vr_beamgeom.cuh"

using namespace vr;

static void cross(const double a[3], const double b[3], double c[3])
{
    c[0] = a[1] * b[2] - a[2] * b[1]; c[1] = a[2] * b[0] - a[0] * b[2]; c[2] = a[0] * b[1] - a[1] * b[0];
}
static void norm(double a[3]) { double l = std::sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]); for (int i = 0; i < 3; ++i) a[i] /= l; }

// Host model of the step loop of run_beam() in vr_shear.cu, executing the SAME plan_window() / ring_slot() /
// plane_of_ordinal(): loads of step s + 1 are in flight while step s marches, the planner writes the address
// table two steps ahead.  Checks: every base plane is marched exactly once, in travel order; both data planes of
// a marched base plane are resident in a ring slot that no in-flight copy may overwrite; the 64-entry address
// table still points at them.
static long long check_schedule(std::mt19937_64 &rng, long long &bad)
{
    std::uniform_real_distribution<double> U(0.0, 1.0);
    const int iw_min = (int)(U(rng) * 300), iw_max = iw_min + (int)(U(rng) * (U(rng) < 0.3 ? 3 : 400));
    const int sgn = U(rng) < 0.5 ? 1 : -1, G = 1 + (int)(U(rng) * 16), NS = 2 * G + 1 + (U(rng) < 0.3 ? (int)(U(rng) * 4) : 0);
    const int n_base = iw_max - iw_min + 1;
    int next_ord = 0, wstart = 0, ord0[3];
    StepPlan rec[3];
    std::vector<int> ring(NS, -1), covered(n_base, 0);
    int tab[64];
    for (int i = 0; i < 64; ++i) tab[i] = -1;
    auto ordinal = [&](int q) { return sgn > 0 ? q - iw_min : iw_max + 1 - q; };
    auto plan = [&](int r, bool first) {
        ord0[r] = next_ord;
        rec[r] = plan_window(first, G, sgn, iw_min, iw_max, next_ord, wstart);
        for (int k = 0; k < rec[r].nload; ++k) { const int q = plane_of_ordinal(sgn, iw_min, iw_max, ord0[r] + k); tab[q & 63] = q; }
    };
    auto land = [&](int r) {
        for (int k = 0; k < rec[r].nload; ++k) ring[ring_slot(ord0[r] + k, NS)] = plane_of_ordinal(sgn, iw_min, iw_max, ord0[r] + k);
    };
    plan(0, true); plan(1, false);
    land(0);
    long long n = 0;
    int last = sgn > 0 ? iw_min - 1 : iw_max + 1;
    for (int it = 0;; ++it) {
        const StepPlan S = rec[it % 3];
        if (S.wn == 0) break;
        std::vector<char> inflight(NS, 0);
        const int r1 = (it + 1) % 3;
        for (int k = 0; k < rec[r1].nload; ++k) inflight[ring_slot(ord0[r1] + k, NS)] = 1;
        plan((it + 2) % 3, false);
        for (int t = 0; t < S.wn; ++t) {
            const int ia = sgn > 0 ? S.wlo + t : S.wlo + S.wn - 1 - t;            // travel order inside the window
            if (ia < iw_min || ia > iw_max) { ++bad; continue; }
            if (ia != last + sgn) ++bad;
            last = ia;
            covered[ia - iw_min]++;
            for (int q = ia; q <= ia + 1; ++q) {
                const int slot = ring_slot(ordinal(q), NS);
                if (ring[slot] != q || inflight[slot] || tab[q & 63] != q) ++bad;
                ++n;
            }
        }
        land(r1);
    }
    for (int c : covered) if (c != 1) ++bad;
    return n;
}

int main(int argc, char **argv)
{
    const int n_cams = argc > 1 ? atoi(argv[1]) : 60;
    std::mt19937_64 rng(12345);
    std::uniform_real_distribution<double> U(0.0, 1.0);
    long long checked = 0, rect_bad = 0, beams = 0, skipped = 0, convex_bad = 0;
    for (int ci = 0; ci < n_cams; ++ci) {
        const int n[3] = { 24 + (int)(U(rng) * 200), 24 + (int)(U(rng) * 200), 24 + (int)(U(rng) * 200) };
        const int W = 64 + (int)(U(rng) * 200), H = 48 + (int)(U(rng) * 150);
        const bool ortho = ci % 5 == 4;
        double c[3] = { n[0] / 2.0, n[1] / 2.0, n[2] / 2.0 }, e[3] = { U(rng) - .5, U(rng) - .5, U(rng) - .5 };
        norm(e);
        const double R = (0.3 + 2.5 * U(rng)) * std::max(n[0], std::max(n[1], n[2]));      // also eyes inside the volume
        double eye[3], f[3], up[3] = { 0, 1, 0 }, r[3], u[3];
        for (int a = 0; a < 3; ++a) { eye[a] = c[a] + R * e[a]; f[a] = -e[a]; }
        if (std::fabs(e[1]) > 0.9) { up[1] = 0; up[2] = 1; }
        cross(f, up, r); norm(r); cross(r, f, u);
        CamK cam;
        const double th = std::tan((15.0 + 50.0 * U(rng)) * M_PI / 360.0), asp = (double)W / H, ext = (0.5 + U(rng)) * n[1];
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
        cam.step = 0.5f; cam.t_min = 1.0f; cam.width = W; cam.height = H;
        for (int ty = 0; ty * kBH < H; ++ty)
            for (int tx = 0; tx * kBW < W; ++tx) {
                if (U(rng) > 0.25) continue;
                const int x0 = tx * kBW, y0 = ty * kBH;
                const int x1 = std::min(x0 + kBW, W), y1 = std::min(y0 + kBH, H);
                float oc[3], gc[3];
                cam_ray_at(cam, (float)x0 + 0.5f * kBW, (float)y0 + 0.5f * kBH, oc, gc);
                const int a = principal_axis(gc), sgn = gc[a] > 0.0f ? 1 : -1;
                int au, av;
                beam_axes(a, au, av);
                BeamLine L[4];
                bool ok = true;
                for (int k = 0; k < 4 && ok; ++k)
                    ok = beam_line(cam, (float)((k & 1) ? x1 : x0), (float)((k & 2) ? y1 : y0), a, sgn, L[k]);
                if (!ok) { ++skipped; continue; }          // such beams march from global memory
                ++beams;
                {   // the kernel sizes a beam by beam_rect_bound() + 1: no plane of the range may need more
                    int Pa = (int)(U(rng) * (n[a] - 1)), Pb = Pa + (int)(U(rng) * (n[a] - Pa));
                    if (U(rng) < 0.3) Pa = 0;                                   // the outer planes serve a thicker range
                    if (U(rng) < 0.3) Pb = n[a] - 1;
                    int u0, v0, wb, hb;
                    beam_rect_bound(L, Pa, Pb, n[a], n[au], n[av], wb, hb);
                    for (int P = Pa; P <= Pb; ++P) {
                        int w, h;
                        plane_rect(L, P, n[a], n[au], n[av], true, u0, v0, w, h);
                        if (w > wb + 1 || h > hb + 1) ++convex_bad;
                    }
                }
                for (int s = 0; s < 200; ++s) {
                    // a ray through a pixel centre of the tile, a position on it inside the volume
                    const int i = x0 + (int)(U(rng) * (x1 - x0)), j = y0 + (int)(U(rng) * (y1 - y0));
                    float of[3], gf[3];
                    cam_ray_at(cam, (float)i + 0.5f, (float)j + 0.5f, of, gf);
                    const double cpos = U(rng) * n[a];
                    const double lam = (cpos - (double)of[a]) / (double)gf[a];
                    if (!(lam > 0.0) && !ortho) continue;
                    double p[3];
                    for (int d = 0; d < 3; ++d) p[d] = (double)of[d] + lam * (double)gf[d];
                    if (p[au] < 0.0 || p[au] > n[au] || p[av] < 0.0 || p[av] > n[av]) continue;
                    auto base = [](double q, int nn) { int b = (int)std::floor(q - 0.5); return b < 0 ? 0 : (b > nn - 2 ? nn - 2 : b); };
                    const int ia = base(p[a], n[a]), iu = base(p[au], n[au]), iv = base(p[av], n[av]);
                    for (int dq = 0; dq < 2; ++dq) {
                        const int q = ia + dq;
                        int u0, v0, w, h;
                        plane_rect(L, q, n[a], n[au], n[av], false, u0, v0, w, h);
                        ++checked;
                        if (iu < u0 || iu + 1 > u0 + w - 1 || iv < v0 || iv + 1 > v0 + h - 1) ++rect_bad;
                    }
                }
            }
    }
    long long sched_bad = 0, sched_checked = 0;
    for (int k = 0; k < 20000; ++k) sched_checked += check_schedule(rng, sched_bad);
    printf("beams %lld skipped %lld checked %lld rect_bad %lld convex_bad %lld schedule_checked %lld schedule_bad %lld\n", beams,
           skipped, checked, rect_bad, convex_bad, sched_checked, sched_bad);
    return (rect_bad || convex_bad || sched_bad || checked < 100000 || sched_checked < 100000) ? 1 : 0;
}
