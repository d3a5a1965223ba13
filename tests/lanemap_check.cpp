// Host brute force of the pixel-to-lane map of the lane-mapped ray-caster (csrc/vr_lanemap.h + the pixel
// formula of k_rows in csrc/vr_lanes.cu): for random perspective, orthographic and mixed cameras and image
// sizes, every pixel of the image is produced by exactly one (CTA, warp, lane) of the launched grid, for
// both volume copies and every pixel class.  Also reports how well the shear follows the fast axis.
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
                LaneMapK M;
                int rows;
                make_lane_map(&c, n, fast, cls, 1, M, rows);
                const int W = (int)c.width, H = (int)c.height;
                const int P = M.lane_axis == 0 ? W : H;
                std::vector<int> cnt((size_t)W * H, 0);
                const int gx = (P + 31) / 32, gy = (rows + 7) / 8;
                if (!(M.sigma >= -1.0f && M.sigma <= 1.0f) || M.paxis == fast || M.paxis < 0 || M.paxis > 2) ++bad;
                for (int by = 0; by < gy; ++by)
                    for (int bx = 0; bx < gx; ++bx)
                        for (int t = 0; t < 256; ++t) {
                            const int lane = t & 31, warp = t >> 5;
                            const int p = bx * 32 + lane;
                            const int q = M.q_lo + by * 8 + warp + lane_row_offset(M.sigma, p);
                            const int i = M.lane_axis == 0 ? p : q, j = M.lane_axis == 0 ? q : p;
                            if (i >= 0 && i < W && j >= 0 && j < H) cnt[(size_t)j * W + i]++;
                        }
                for (int v : cnt) if (v != 1) ++bad;
                ++cams;
            }
    }
    printf("maps %lld bad %lld\n", cams, bad);
    return bad ? 1 : 0;
}
