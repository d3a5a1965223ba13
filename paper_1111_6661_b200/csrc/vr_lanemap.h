// vr_lanemap.h — host-only choice of the pixel-to-lane map of the lane-mapped ray-caster (vr_lanes.cu;
// SURVEY.md row A4's single-GPU analogue of the paper's scheduler): which image axis the 32
// lanes of a warp run along and by how much the image rows are sheared, so that the samples a warp takes at
// equal k lie along the memory-fast axis of the volume copy it reads.  O(1) per frame, plain C++ (no CUDA):
// tests/lanemap_check.cpp executes it and the kernel's pixel formula on the host and checks that every
// pixel is rendered exactly once for any camera.  The map never changes results, only speed.
#pragma once
#include <cmath>

#include "../../include/vr.h"

namespace vr {

// Pixel (lane coordinate p, sheared row qs) is image pixel (p, qs + off(p)) along the lane axis, with
// off(p) = floor(sigma p + 1/2) evaluated in float32 exactly as below (the kernel uses the same formula).
struct LaneMapK {
    int lane_axis;      // 0: lanes run along image i (rows are j); 1: lanes run along image j
    float sigma;        // shear of the rows, |sigma| <= 1
    int q_lo;           // first sheared row (may be negative)
    int cls;            // pixels this launch renders: 0 all, 1 those with |d_x| <= |d_z|, 2 those with |d_x| > |d_z|
    int lag;            // 0 off; else a lane more than `lag` base planes ahead of the slowest active lane waits
    int paxis, psign;   // principal axis of the view and the sign of travel along it (progress measure of `lag`)
    int w[3];           // psign on paxis, 0 elsewhere: progress of a sample = w . (ix, iy, iz)
};

inline int lane_row_offset(float sigma, int p) { return (int)floorf(fmaf(sigma, (float)p, 0.5f)); }

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

// fast: 0 = x-fastest array, 2 = z-fastest copy.  cls as in LaneMapK.  rows = sheared rows to launch.
inline void make_lane_map(const vr_camera *cam, const int n[3], int fast, int cls, int lag, LaneMapK &M, int &rows)
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
    const int other = 3 - pa - fast;                                  // the in-plane axis that is not the fast one
    M.lane_axis = 0;
    M.sigma = 0.0f;
    double P0[3], Pi[3], Pj[3];
    const double c = 0.5 * n[pa];
    if (lane_plane_point(cam, xc, yc, pa, c, P0) && lane_plane_point(cam, xc + 1.0, yc, pa, c, Pi) &&
        lane_plane_point(cam, xc, yc + 1.0, pa, c, Pj)) {
        for (int a = 0; a < 3; ++a) { Pi[a] -= P0[a]; Pj[a] -= P0[a]; }
        M.lane_axis = std::fabs(Pi[fast]) >= std::fabs(Pj[fast]) ? 0 : 1;
        const double *L = M.lane_axis == 0 ? Pi : Pj, *R = M.lane_axis == 0 ? Pj : Pi;
        // one lane step plus sigma row steps must not move along `other`
        double s = R[other] != 0.0 ? -L[other] / R[other] : 0.0;
        if (!std::isfinite(s)) s = 0.0;
        s = s > 1.0 ? 1.0 : s < -1.0 ? -1.0 : s;
        M.sigma = (float)s;
    }
    const int Pn = M.lane_axis == 0 ? W : H, Qn = M.lane_axis == 0 ? H : W;
    const int o0 = lane_row_offset(M.sigma, 0), o1 = lane_row_offset(M.sigma, Pn > 0 ? Pn - 1 : 0);
    const int omin = (o0 < o1 ? o0 : o1) - 1, omax = (o0 < o1 ? o1 : o0) + 1;   // one row of slack each side
    M.q_lo = -omax;                                                   // q = qs + off in [0, Qn)  =>  qs in [-omax, Qn - 1 - omin]
    rows = Qn - omin + omax;
}

}  // namespace vr
