// vr_lanemap.h — the pixel-to-lane map of the lane-mapped ray-caster (vr_lanes.cu; SURVEY.md row A4's
// single-GPU analogue of the paper's scheduler): which image axis the 32 lanes of a warp run
// along and by how much the image rows are sheared, so that the samples a warp takes on one plane of the
// view's principal axis lie along the memory-fast axis of the volume copy it reads.
//
// The image (or the pixel lattice of a progressive pass) is cut into TILES of 32 lanes x kLaneTileH rows.  Inside
// a tile the rows are sheared by an integer offset off(lane) = floor(sigma lane + 1/2) with the tile's OWN sigma,
// evaluated at the tile's centre: under perspective the ideal shear changes several-fold across the image (the
// image lines that map to voxel rows meet in a vanishing point), and a lane that drifts off its voxel row costs
// a cache line of its own per load.  Any sigma gives a bijection of the tile's pixels (proof at lane_pixel), so
// the map never changes results, only speed.  Host and device use the SAME functions of this header; it is plain
// C++ (no CUDA needed): tests/lanemap_check.cpp executes them on the host and checks that every pixel is rendered
// exactly once for any camera.
#pragma once
#include <cmath>

#include "../../include/vr.h"

#if defined(__CUDACC__)
#define VR_HD __host__ __device__
#else
#define VR_HD
#endif

namespace vr {

constexpr int kLaneTileH = 64;          // rows of a tile
constexpr int kLaneRowsPerCta = 8;      // warps (sheared rows) of a CTA

struct LaneMapK {
    int lane_axis;      // 0: lanes run along image i (rows are j); 1: lanes run along image j
    float sigma;        // shear at the image centre, |sigma| <= 1 (used for every tile when per_tile == 0)
    int per_tile;       // 1: every tile evaluates its own shear (VR_OPT_TILE_SHEAR)
    int bpt;            // CTAs per tile along the rows: ceil((kLaneTileH + 32) / kLaneRowsPerCta)
    int cls;            // pixels this launch renders: 0 all, 1 those with |d_x| <= |d_z|, 2 those with |d_x| > |d_z|
    int lag;            // 0 off; else a lane more than `lag` base planes ahead of the slowest active lane waits
    int paxis, psign;   // principal axis of the view and the sign of travel along it (progress measure of `lag`)
    int w[3];           // psign on paxis, 0 elsewhere: progress of a sample = w . (ix, iy, iz)
    int reuse;          // 1: keep a ray's 8 corner voxels in registers while its samples stay in one cell (step < 1 voxel)
    int fast;           // memory-fast axis of the volume copy this launch reads (0 or 2)
    float plane_c;      // the plane coord[paxis] = plane_c on which the shear is evaluated (mid-volume)
};

VR_HD inline int lane_row_offset(float sigma, int lane) { return (int)floorf(fmaf(sigma, (float)lane, 0.5f)); }

// Shear that keeps a step along the lane axis, taken on the plane coord[paxis] = plane_c, free of any movement
// along the in-plane axis that is not the fast one, for the ray through the continuous image point (x, y).
// With P(x, y) = o + s g, s = (plane_c - o_pa) / g_pa:  dP/dx = ou + s_x g + s du,  s_x = -(ou_pa + s du_pa) / g_pa.
VR_HD inline float lane_pick(const float *a, int k) { return k == 0 ? a[0] : k == 1 ? a[1] : a[2]; }   // no dynamic indexing

template <typename Cam>
VR_HD inline float lane_shear_at(const Cam &c, int lane_axis, int paxis, int fast, float plane_c, float x, float y)
{
    const int other = 3 - paxis - fast;
    // the paxis and `other` components of origin, direction and their image derivatives
    const float ou_p = lane_pick(c.ou, paxis), ov_p = lane_pick(c.ov, paxis), du_p = lane_pick(c.du, paxis), dv_p = lane_pick(c.dv, paxis);
    const float ou_o = lane_pick(c.ou, other), ov_o = lane_pick(c.ov, other), du_o = lane_pick(c.du, other), dv_o = lane_pick(c.dv, other);
    const float o_p = lane_pick(c.o0, paxis) + x * ou_p + y * ov_p, g_p = lane_pick(c.d0, paxis) + x * du_p + y * dv_p;
    const float g_o = lane_pick(c.d0, other) + x * du_o + y * dv_o;
    if (g_p == 0.0f) return 0.0f;
    const float s = (plane_c - o_p) / g_p;
    const float si = -(ou_p + s * du_p) / g_p, sj = -(ov_p + s * dv_p) / g_p;
    const float Pi = ou_o + si * g_o + s * du_o, Pj = ov_o + sj * g_o + s * dv_o;
    const float L = lane_axis == 0 ? Pi : Pj, R = lane_axis == 0 ? Pj : Pi;
    float sg = R != 0.0f ? -L / R : 0.0f;
    if (!(sg >= -1.0f)) sg = sg < 0.0f ? -1.0f : 0.0f;        // NaN -> 0
    if (sg > 1.0f) sg = 1.0f;
    return sg;
}

// Lattice pixel (li, lj) of lane `lane` of warp `warp` of CTA (bx, by); (-1, -1) if that thread has none.
// Tile (bx, ty = by / bpt) holds lattice pixels p in [32 bx, 32 bx + 32) x q in [q0, q0 + kLaneTileH), q0 =
// kLaneTileH ty.  Sheared row r = (by % bpt) kLaneRowsPerCta + warp of the tile holds, for every lane, the pixel
// q = q0 + r - omax + off(lane) if that lies in the tile, with omin <= off(lane) <= omax (off is monotone in the
// lane and off(0) = 0).  For a fixed lane, r -> q is a shift, and r ranges over [0, kLaneTileH + omax - omin), which
// contains [omax - off, omax - off + kLaneTileH): every q of the tile is produced exactly once.
// sub, sx, sy: the lattice of a progressive pass (image pixel = sub * lattice pixel + (sx, sy)); 1, 0, 0 otherwise.
// rows_of_tile: how many sheared rows of this tile hold pixels (the same for every thread of the tile's CTAs).
template <typename Cam>
VR_HD inline void lane_pixel(const Cam &c, const LaneMapK &M, int sub, int sx, int sy, int bx, int by, int warp, int lane,
                             int &li, int &lj, int &rows_of_tile)
{
    const int ty = by / M.bpt, r = (by % M.bpt) * kLaneRowsPerCta + warp, q0 = ty * kLaneTileH;
    float sigma = M.sigma;
    if (M.per_tile) {
        const float pc = (float)(bx * 32 + 16), qc = (float)(q0 + kLaneTileH / 2);      // tile centre, lattice coordinates
        const float lx = M.lane_axis == 0 ? pc : qc, ly = M.lane_axis == 0 ? qc : pc;
        sigma = lane_shear_at(c, M.lane_axis, M.paxis, M.fast, M.plane_c, lx * (float)sub + (float)sx, ly * (float)sub + (float)sy);
    }
    const int o31 = lane_row_offset(sigma, 31), omax = o31 > 0 ? o31 : 0, omin = o31 < 0 ? o31 : 0;
    rows_of_tile = kLaneTileH + omax - omin;
    li = lj = -1;
    if (r >= rows_of_tile) return;
    const int p = bx * 32 + lane, q = q0 + r - omax + lane_row_offset(sigma, lane);
    if (q < q0 || q >= q0 + kLaneTileH) return;
    li = M.lane_axis == 0 ? p : q;
    lj = M.lane_axis == 0 ? q : p;
}

// point where the ray of pixel centre (x, y) (continuous pixel coordinates, C.1 in double) meets the plane
// `coord[paxis] = c`; false if the ray is parallel to it
inline bool lane_plane_point(const vr_camera *cam, double x, double y, int paxis, double c, double P[3])
{
    double o[3], g[3];
    for (int a = 0; a < 3; ++a) {
        o[a] = (double)cam->o0[a] + x * (double)cam->ou[a] + y * (double)cam->ov[a];
        g[a] = (double)cam->d0[a] + x * (double)cam->du[a] + y * (double)cam->dv[a];
    }
    if (g[paxis] == 0.0) return false;
    const double s = (c - o[paxis]) / g[paxis];
    for (int a = 0; a < 3; ++a) P[a] = o[a] + s * g[a];
    return std::isfinite(P[0]) && std::isfinite(P[1]) && std::isfinite(P[2]);
}

// fast: 0 = x-fastest array, 2 = z-fastest copy.  cls as in LaneMapK.  `cam` is the camera of the pixels this launch
// renders (the lattice camera of a progressive pass).  rows = sheared rows to launch (grid.y * kLaneRowsPerCta).
inline void make_lane_map(const vr_camera *cam, const int n[3], int fast, int cls, int lag, int per_tile, LaneMapK &M, int &rows)
{
    const int W = (int)cam->width, H = (int)cam->height;
    const double xc = 0.5 * W, yc = 0.5 * H;
    double g[3];
    for (int a = 0; a < 3; ++a) g[a] = (double)cam->d0[a] + xc * (double)cam->du[a] + yc * (double)cam->dv[a];
    // principal axis of the centre ray among the axes this launch's pixels can have as principal
    // (a pixel with |d_x| <= |d_z| is never x-principal, one with |d_x| > |d_z| never z-principal)
    int pa = -1;
    for (int a = 0; a < 3; ++a) {
        if ((cls == 1 && a == 0) || (cls == 2 && a == 2)) continue;
        if (pa < 0 || std::fabs(g[a]) > std::fabs(g[pa])) pa = a;
    }
    if (pa == fast) pa = fast == 0 ? 2 : 0;                           // cls 0 on a copy whose fast axis is principal
    M.paxis = pa;
    M.psign = g[pa] >= 0.0 ? 1 : -1;
    for (int a = 0; a < 3; ++a) M.w[a] = a == pa ? M.psign : 0;
    M.cls = cls;
    M.lag = lag;
    M.fast = fast;
    M.per_tile = per_tile;
    M.reuse = cam->step < 0.75f ? 1 : 0;
    M.plane_c = 0.5f * (float)n[pa];
    M.bpt = (kLaneTileH + 32 + kLaneRowsPerCta - 1) / kLaneRowsPerCta;
    M.lane_axis = 0;
    M.sigma = 0.0f;
    double P0[3], Pi[3], Pj[3];
    const double c = 0.5 * n[pa];
    if (lane_plane_point(cam, xc, yc, pa, c, P0) && lane_plane_point(cam, xc + 1.0, yc, pa, c, Pi) &&
        lane_plane_point(cam, xc, yc + 1.0, pa, c, Pj)) {
        for (int a = 0; a < 3; ++a) { Pi[a] -= P0[a]; Pj[a] -= P0[a]; }
        M.lane_axis = std::fabs(Pi[fast]) >= std::fabs(Pj[fast]) ? 0 : 1;
        M.sigma = lane_shear_at(*cam, M.lane_axis, pa, fast, M.plane_c, (float)xc, (float)yc);
    }
    const int Qn = M.lane_axis == 0 ? H : W;
    rows = (Qn + kLaneTileH - 1) / kLaneTileH * M.bpt * kLaneRowsPerCta;
}

}  // namespace vr
