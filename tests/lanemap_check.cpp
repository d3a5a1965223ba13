// Host brute force of the pixel-to-lane map of the lane-mapped ray-caster (csrc/vr_lanemap.h: make_lane_map and
// lane_pixel, the function k_rows itself calls): for random perspective, orthographic and mixed cameras and image
// sizes, every pixel of the image is produced by exactly one (CTA, warp, lane) of the launched grid, for
// both volume copies and every pixel class.  Also reports how well the shear follows the fast axis.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <random>
#include <vector>

#include "../paper_1111_6661_b200/csrc/vr_lanemap.h"

using namespace vr;

int main(int argc, char **argv)
{
    const int n_cams = argc > 1 ? atoi(argv[1]) : 200;
    std::mt19937_64 rng(0x1111666100000001ull);
    std::uniform_real_distribution<double> U(-1.0, 1.0);
    long long bad = 0, cams = 0;
    for (int it = 0; it < n_cams; ++it) {
        vr_camera c{};
        c.struct_size = sizeof(c);
        c.width = 1 + (unsigned)(rng() % 300);
        c.height = 1 + (unsigned)(rng() % 200);
        const int kind = it % 3;                         // 0 perspective, 1 orthographic, 2 mixed
        for (int a = 0; a < 3; ++a) {
            c.o0[a] = (float)(200.0 * U(rng));
            c.d0[a] = (float)U(rng);
            c.du[a] = kind != 1 ? (float)(0.01 * U(rng)) : 0.0f;
            c.dv[a] = kind != 1 ? (float)(0.01 * U(rng)) : 0.0f;
            c.ou[a] = kind != 0 ? (float)U(rng) : 0.0f;
            c.ov[a] = kind != 0 ? (float)U(rng) : 0.0f;
        }
        c.step = 1.0f;
        const int n[3] = { 64, 48, 80 };
        for (int fast = 0; fast <= 2; fast += 2)
            for (int cls = 0; cls <= 2; ++cls) {
                for (int per_tile = 0; per_tile <= 1; ++per_tile) {
                LaneMapK M;
                int rows;
                make_lane_map(&c, n, fast, cls, 1, per_tile, M, rows);
                const int W = (int)c.width, H = (int)c.height;
                const int P = M.lane_axis == 0 ? W : H;
                std::vector<int> cnt((size_t)W * H, 0);
                const int gx = (P + 31) / 32, gy = rows / kLaneRowsPerCta;
                if (!(M.sigma >= -1.0f && M.sigma <= 1.0f) || M.paxis == fast || M.paxis < 0 || M.paxis > 2 || rows % kLaneRowsPerCta) ++bad;
                for (int by = 0; by < gy; ++by)
                    for (int bx = 0; bx < gx; ++bx)
                        for (int t = 0; t < 32 * kLaneRowsPerCta; ++t) {
                            int i, j, rt;
                            lane_pixel(c, M, 1, 0, 0, bx, by, t >> 5, t & 31, i, j, rt);      // the kernel's own pixel formula
                            if (rt < kLaneTileH || rt > kLaneTileH + 32) ++bad;
                            if (i >= 0 && i < W && j >= 0 && j < H) cnt[(size_t)j * W + i]++;
                        }
                for (int v : cnt) if (v != 1) ++bad;
                ++cams;
                }
            }
    }
    // the configs' own images and orbit cameras (workload/cameras.py): 1024^2, 1920x1080, 3840x2160, 8 views each
    const int sizes[3][5] = { { 1024, 1024, 512, 512, 1024 }, { 1920, 1080, 1024, 1024, 2048 }, { 3840, 2160, 2048, 2048, 4096 } };
    for (int si = 0; si < 3; ++si)
        for (int view = 0; view < 8; ++view) {
            const int W = sizes[si][0], H = sizes[si][1], n[3] = { sizes[si][2], sizes[si][3], sizes[si][4] };
            const double c[3] = { n[0] / 2.0, n[1] / 2.0, n[2] / 2.0 };
            const double rb = 0.5 * std::sqrt((double)n[0] * n[0] + (double)n[1] * n[1] + (double)n[2] * n[2]);
            const double R = rb / std::sin(M_PI / 8.0), th = 2.0 * M_PI * (view + 0.25) / 8.0, el = M_PI / 9.0;
            const double eye[3] = { c[0] + R * std::cos(el) * std::sin(th), c[1] + R * std::sin(el), c[2] + R * std::cos(el) * std::cos(th) };
            double f[3] = { c[0] - eye[0], c[1] - eye[1], c[2] - eye[2] };
            const double fl = std::sqrt(f[0] * f[0] + f[1] * f[1] + f[2] * f[2]);
            for (double &x : f) x /= fl;
            double r[3] = { f[1] * 0 - f[2] * 1, f[2] * 0 - f[0] * 0, f[0] * 1 - f[1] * 0 };      // f x (0,1,0)
            const double rl = std::sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]);
            for (double &x : r) x /= rl;
            const double u[3] = { r[1] * f[2] - r[2] * f[1], r[2] * f[0] - r[0] * f[2], r[0] * f[1] - r[1] * f[0] };
            const double tf = std::tan(M_PI / 8.0), asp = (double)W / H;
            vr_camera cam{};
            cam.struct_size = sizeof(cam); cam.width = (unsigned)W; cam.height = (unsigned)H; cam.step = 1.0f;
            for (int a = 0; a < 3; ++a) {
                cam.o0[a] = (float)eye[a];
                cam.d0[a] = (float)(f[a] - tf * asp * r[a] - tf * u[a]);
                cam.du[a] = (float)(2.0 * tf * asp / W * r[a]); cam.dv[a] = (float)(2.0 * tf / H * u[a]);
            }
            for (int fast = 0; fast <= 2; fast += 2) {
                LaneMapK M;
                int rows;
                make_lane_map(&cam, n, fast, fast == 0 ? 1 : 2, 1, 1, M, rows);
                const int P = M.lane_axis == 0 ? W : H;
                std::vector<unsigned char> cnt((size_t)W * H, 0);
                const int gx = (P + 31) / 32, gy = rows / kLaneRowsPerCta;
                for (int by = 0; by < gy; ++by)
                    for (int bx = 0; bx < gx; ++bx)
                        for (int t = 0; t < 32 * kLaneRowsPerCta; ++t) {
                            int i, j, rt;
                            lane_pixel(cam, M, 1, 0, 0, bx, by, t >> 5, t & 31, i, j, rt);
                            if (i >= 0 && i < W && j >= 0 && j < H) cnt[(size_t)j * W + i]++;
                        }
                for (unsigned char v : cnt) if (v != 1) ++bad;
                ++cams;
            }
        }
    printf("maps %lld bad %lld\n", cams, bad);
    return bad ? 1 : 0;
}
